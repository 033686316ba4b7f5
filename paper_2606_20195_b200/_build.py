"""In-tree build of the CUDA library (nvcc, sm_100a only).  No JIT cache: the .so sits next to the
sources so it travels to the GPU box with the repository snapshot.  One translation unit per kernel
family, compiled concurrently, then linked into libsparse_sketch.so."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
OBJ = HERE / "_obj"
LIB = HERE / "libsparse_sketch.so"
SOURCES = [CSRC / n for n in ("sparse_sketch.cu", "tmem_host.cu", "launch_flat_f16.cu", "launch_flat_bf16.cu", "launch_flat_f32.cu", "launch_smem.cu",
                              "launch_tmem.cu")]
HEADERS = [CSRC / n for n in ("args.h", "launch.h", "device_util.cuh", "kernel_flat.cuh", "kernel_misc.cuh", "kernel_smem.cuh", "kernel_small.cuh", "kernel_tmem.cuh")]
# (source, object stem, extra flags): launch_tmem.cu is compiled once per (zeta, accumulation mode) family; the largest
# units (FP16-RN with its deferral kernels) go first so the pool finishes together
UNITS = [(CSRC / "launch_tmem.cu", "launch_tmem_z%d_m%d" % (z, mo), ["-DSK_TMEM_ZETA=%d" % z, "-DSK_TMEM_MODE=%d" % mo])
         for mo in (0, 1, 4, 2, 3) for z in (8, 4, 2, 1)]
UNITS += [(src, src.stem, []) for src in SOURCES if src.name != "launch_tmem.cu"]
HEADERS.append(HERE.parent / "include" / "sparse_sketch.h")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC",
    "-Xptxas", "-v",
]


def _nvcc() -> str:
    return os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def _stale(target: Path, deps) -> bool:
    if not target.exists():
        return True
    t = target.stat().st_mtime
    return any(p.stat().st_mtime > t for p in deps)


def _compile(unit, force: bool) -> Path:
    src, stem, extra = unit
    obj = OBJ / (stem + ".o")
    if force or _stale(obj, [src] + HEADERS):
        res = subprocess.run([_nvcc()] + NVCC_FLAGS + extra + ["-c", str(src), "-o", str(obj)], capture_output=True, text=True)
        (OBJ / (stem + ".ptxas.log")).write_text(res.stderr)
        if res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
            raise RuntimeError("nvcc failed on %s" % src.name)
    return obj


def build(force: bool = False, verbose: bool = False) -> Path:
    OBJ.mkdir(exist_ok=True)
    if not force and not _stale(LIB, SOURCES + HEADERS):
        return LIB
    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 4)) as ex:
        objs = list(ex.map(lambda u: _compile(u, force), UNITS))
    tmp = LIB.with_suffix(".so.tmp%d" % os.getpid())
    res = subprocess.run([_nvcc(), "-shared", "-o", str(tmp)] + [str(o) for o in objs], capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("link of libsparse_sketch.so failed")
    os.replace(tmp, LIB)
    if verbose:
        for _, stem, _ in UNITS:
            sys.stderr.write((OBJ / (stem + ".ptxas.log")).read_text())
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
