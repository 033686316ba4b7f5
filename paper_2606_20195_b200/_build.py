"""In-tree build of the CUDA library (nvcc, sm_100a only).  No JIT cache: the .so sits next to the
sources so it travels to the GPU box with the repository snapshot."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libsparse_sketch.so"
SOURCES = [CSRC / "sparse_sketch.cu"]
DEPS = SOURCES + [CSRC / "kernels.cuh", CSRC / "kernel_smem.cuh", CSRC / "device_util.cuh", HERE.parent / "include" / "sparse_sketch.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
]


def is_stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in DEPS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not is_stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB.with_suffix(".so.tmp%d" % os.getpid())
    cmd = [nvcc] + NVCC_FLAGS + ["-o", str(tmp)] + [str(s) for s in SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    (HERE / "build_ptxas.log").write_text(res.stderr)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libsparse_sketch.so")
    if verbose:
        sys.stderr.write(res.stderr)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
