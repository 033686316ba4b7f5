"""CPU oracle for the sparse-sketch hot path -- TEST INFRASTRUCTURE, not product code.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports
``paper_2606_20195_b200`` and shares no code with its CUDA sources.

The arithmetic lives in ``sketch_oracle.cpp`` (plain C++17, FP64 unless the paper
fixes the precision); this file only compiles it with g++ and marshals numpy
arrays through ctypes.  Function-by-function citations are in the C++ source.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = [_HERE / "sketch_oracle.cpp", _HERE / "f16c_crosscheck.cpp", _HERE / "bf16_crosscheck.cpp"]
_LIB = _HERE / "_build" / "liboracle.so"
_lock = threading.Lock()
_lib = None

IDEAL, BQ, BC = 0, 1, 2  # modes of f64_sketch (Eq. 7)
RN, SR, DITHER = 0, 1, 2   # conversion rules of PAPER.md:193-207 (Sec. III-D)


def _host_has_f16c() -> bool:
    try:
        return " f16c" in Path("/proc/cpuinfo").read_text()
    except OSError:
        return False


def build(force: bool = False) -> Path:
    """Compile the oracle shared library with g++ (no CUDA involved)."""
    with _lock:
        newest = max(p.stat().st_mtime for p in _SRC)
        if not force and _LIB.exists() and _LIB.stat().st_mtime >= newest:
            return _LIB
        _LIB.parent.mkdir(exist_ok=True)
        common = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fPIC", "-pthread", "-Wall"]
        objs = []
        o0 = _LIB.parent / "sketch_oracle.o"
        subprocess.check_call(common + ["-c", str(_SRC[0]), "-o", str(o0)])
        objs.append(str(o0))
        o2 = _LIB.parent / "bf16_crosscheck.o"
        subprocess.check_call(common + ["-c", str(_SRC[2]), "-o", str(o2)])
        objs.append(str(o2))
        if _host_has_f16c():
            o1 = _LIB.parent / "f16c_crosscheck.o"
            subprocess.check_call(common + ["-mf16c", "-c", str(_SRC[1]), "-o", str(o1)])
            objs.append(str(o1))
        tmp = _LIB.with_suffix(".so.tmp%d" % os.getpid())
        subprocess.check_call(["g++", "-shared", "-pthread", "-o", str(tmp)] + objs)
        os.replace(tmp, _LIB)
        return _LIB


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(str(build()))
        u64, i64, i32, u32, u16 = C.c_uint64, C.c_int64, C.c_int32, C.c_uint32, C.c_uint16
        vp = C.c_void_p
        L.orc_splitmix64.restype = u64
        L.orc_splitmix64.argtypes = [u64]
        L.orc_rn16.restype = u16
        L.orc_rn16.argtypes = [C.c_float]
        L.orc_rn16_from_double.restype = u16
        L.orc_rn16_from_double.argtypes = [C.c_double]
        L.orc_half_to_double.restype = C.c_double
        L.orc_half_to_double.argtypes = [u16]
        L.orc_add16.restype = u16
        L.orc_add16.argtypes = [u16, u16]
        L.orc_sr16.restype = u16
        L.orc_sr16.argtypes = [C.c_float, u32]
        L.orc_scale_f32.restype = C.c_float
        L.orc_scale_f32.argtypes = [i32]
        L.orc_rn16_array.restype = None
        L.orc_rn16_array.argtypes = [vp, i64, vp]
        L.orc_add16_array.restype = None
        L.orc_add16_array.argtypes = [vp, vp, i64, vp]
        L.orc_sr16_array.restype = None
        L.orc_sr16_array.argtypes = [vp, vp, i64, vp]
        L.orc_hash.restype = C.c_int
        L.orc_hash.argtypes = [u64, i32, i32, i64, i64, vp, vp]
        L.orc_dense_S.restype = C.c_int
        L.orc_dense_S.argtypes = [u64, i64, i32, i32, vp]
        L.orc_f64_accumulate.restype = C.c_int
        L.orc_f64_accumulate.argtypes = [u64, i32, i32, C.c_int, vp, i64, i64, i32, i64, vp, i32]
        L.orc_f64_finalize.restype = None
        L.orc_f64_finalize.argtypes = [i32, i64, vp]
        L.orc_seq16_accumulate.restype = C.c_int
        L.orc_seq16_accumulate.argtypes = [u64, i32, i32, vp, i64, i64, i32, i64, C.c_int, u64, vp]
        L.orc_seq32_accumulate.restype = C.c_int
        L.orc_seq32_accumulate.argtypes = [u64, i32, i32, vp, i64, i64, i32, i64, vp]
        L.orc_range_counts.restype = C.c_int
        L.orc_range_counts.argtypes = [i32, vp, i64, i32, i64, vp]
        L.orc_bf16_rn.restype = u16
        L.orc_bf16_rn.argtypes = [C.c_float]
        L.orc_bf16_to_double.restype = C.c_double
        L.orc_bf16_to_double.argtypes = [u16]
        L.orc_bf16_add.restype = u16
        L.orc_bf16_add.argtypes = [u16, u16]
        L.orc_xorshift64.restype = u64
        L.orc_xorshift64.argtypes = [u64]
        L.orc_dither_c.restype = C.c_float
        L.orc_dither_c.argtypes = []
        L.orc_bf16_rn_array.restype = None
        L.orc_bf16_rn_array.argtypes = [vp, i64, vp]
        L.orc_bf16_add_array.restype = None
        L.orc_bf16_add_array.argtypes = [vp, vp, i64, vp]
        L.orc_bf16_to_double_array.restype = None
        L.orc_bf16_to_double_array.argtypes = [vp, i64, vp]
        L.orc_dither16_array.restype = None
        L.orc_dither16_array.argtypes = [vp, vp, C.c_float, i64, vp]
        L.orc_seqbf16_accumulate.restype = C.c_int
        L.orc_seqbf16_accumulate.argtypes = [u64, i32, i32, vp, i64, i64, i32, i64, vp]
        L.orc_x_bf16_vs_bits.restype = i64
        L.orc_x_bf16_vs_bits.argtypes = [u32, u64, u32, i32, vp]
        L.orc_x_bf16_add_vs_float.restype = i64
        L.orc_x_bf16_add_vs_float.argtypes = [u32, u32, i32, vp]
        if hasattr(L, "orc_x_rn16_vs_f16c"):
            L.orc_x_rn16_vs_f16c.restype = i64
            L.orc_x_rn16_vs_f16c.argtypes = [u32, u64, u32, i32, vp]
            L.orc_x_add16_vs_f16c.restype = i64
            L.orc_x_add16_vs_f16c.argtypes = [u32, u32, i32, vp]
        _lib = L
    return _lib


def _ptr(a: np.ndarray) -> int:
    return a.ctypes.data


def _check_A(A: np.ndarray) -> np.ndarray:
    if A.dtype != np.float32 or A.ndim != 2 or A.strides[1] != 4 or A.strides[0] % 4:
        raise ValueError("A must be a 2-D float32 array with unit column stride")
    return A


def _ok(rc: int) -> None:
    if rc != 0:
        raise ValueError("oracle rejected the arguments (d %% zeta, n, lda)")


# ---------------------------------------------------------------- scalars
def splitmix64(x: int) -> int:
    return int(lib().orc_splitmix64(x & (2**64 - 1)))


def scale_f32(zeta: int) -> np.float32:
    return np.float32(lib().orc_scale_f32(zeta))


def rn16(p) -> np.ndarray:
    """RN16 of float32 values -> uint16 bit patterns."""
    p = np.ascontiguousarray(p, dtype=np.float32)
    out = np.empty(p.shape, dtype=np.uint16)
    lib().orc_rn16_array(_ptr(p), p.size, _ptr(out))
    return out


def add16(z, v) -> np.ndarray:
    """RN16(z + v) on uint16 bit patterns."""
    z = np.ascontiguousarray(z, dtype=np.uint16)
    v = np.ascontiguousarray(v, dtype=np.uint16)
    assert z.shape == v.shape
    out = np.empty(z.shape, dtype=np.uint16)
    lib().orc_add16_array(_ptr(z), _ptr(v), z.size, _ptr(out))
    return out


def sr16(p, r24) -> np.ndarray:
    p = np.ascontiguousarray(p, dtype=np.float32)
    r24 = np.ascontiguousarray(r24, dtype=np.uint32)
    assert p.shape == r24.shape
    out = np.empty(p.shape, dtype=np.uint16)
    lib().orc_sr16_array(_ptr(p), _ptr(r24), p.size, _ptr(out))
    return out


def bf16_rn(p) -> np.ndarray:
    """RN to bfloat16 of float32 values -> uint16 bit patterns."""
    p = np.ascontiguousarray(p, dtype=np.float32)
    out = np.empty(p.shape, dtype=np.uint16)
    lib().orc_bf16_rn_array(_ptr(p), p.size, _ptr(out))
    return out


def bf16_add(z, v) -> np.ndarray:
    """RN_bf16(z + v) on uint16 bit patterns."""
    z = np.ascontiguousarray(z, dtype=np.uint16)
    v = np.ascontiguousarray(v, dtype=np.uint16)
    assert z.shape == v.shape
    out = np.empty(z.shape, dtype=np.uint16)
    lib().orc_bf16_add_array(_ptr(z), _ptr(v), z.size, _ptr(out))
    return out


def bf16_bits_to_f64(b) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint16)
    out = np.empty(b.shape, dtype=np.float64)
    lib().orc_bf16_to_double_array(_ptr(b), b.size, _ptr(out))
    return out


def xorshift64(x: int) -> int:
    return int(lib().orc_xorshift64(x & (2**64 - 1)))


def dither_c() -> np.float32:
    """The FP32 coefficient c of Eq. (6)."""
    return np.float32(lib().orc_dither_c())


def dither16(p, r24, c=None) -> np.ndarray:
    """Q_dith(p) = RN16(p + (u0 - 1/2) c p), u0 = r24 * 2^-24 (Eq. 6) -> uint16 bit patterns."""
    p = np.ascontiguousarray(p, dtype=np.float32)
    r24 = np.ascontiguousarray(r24, dtype=np.uint32)
    assert p.shape == r24.shape
    out = np.empty(p.shape, dtype=np.uint16)
    lib().orc_dither16_array(_ptr(p), _ptr(r24), float(dither_c() if c is None else c), p.size, _ptr(out))
    return out


def half_bits_to_f64(h) -> np.ndarray:
    """Exact widening of binary16 bit patterns (numpy's float16 view is exact)."""
    return np.ascontiguousarray(h, dtype=np.uint16).view(np.float16).astype(np.float64)


# ---------------------------------------------------------------- hash
def hashes(seed: int, d: int, zeta: int, rows: int, row_begin: int = 0):
    """(bucket:int32[rows,zeta], signbit:uint8[rows,zeta]) for rows [row_begin, row_begin+rows)."""
    bucket = np.empty((rows, zeta), dtype=np.int32)
    sign = np.empty((rows, zeta), dtype=np.uint8)
    _ok(lib().orc_hash(seed, d, zeta, row_begin, rows, _ptr(bucket), _ptr(sign)))
    return bucket, sign


def dense_S(seed: int, m: int, d: int, zeta: int) -> np.ndarray:
    S = np.empty((d, m), dtype=np.float64)
    _ok(lib().orc_dense_S(seed, m, d, zeta, _ptr(S)))
    return S


# ---------------------------------------------------------------- sketches
def f64_accumulate(B: np.ndarray, seed: int, d: int, zeta: int, A: np.ndarray, row_begin: int = 0,
                   mode: int = IDEAL, threads: int = 1) -> None:
    A = _check_A(A)
    assert B.dtype == np.float64 and B.shape == (d, A.shape[1]) and B.flags.c_contiguous
    _ok(lib().orc_f64_accumulate(seed, d, zeta, mode, _ptr(A), row_begin, A.shape[0], A.shape[1],
                                 A.strides[0] // 4, _ptr(B), threads))


def f64_sketch(seed: int, d: int, zeta: int, A: np.ndarray, mode: int = IDEAL, threads: int = 1,
               row_begin: int = 0) -> np.ndarray:
    """B = S A in FP64 (mode IDEAL), or the analytical references B_q / B_c of Eq. (7)."""
    B = np.zeros((d, A.shape[1]), dtype=np.float64)
    f64_accumulate(B, seed, d, zeta, A, row_begin, mode, threads)
    if mode == IDEAL:
        lib().orc_f64_finalize(zeta, B.size, _ptr(B))
    return B


def f64_finalize(B: np.ndarray, zeta: int) -> None:
    lib().orc_f64_finalize(zeta, B.size, _ptr(B))


def seq16_accumulate(D: np.ndarray, seed: int, d: int, zeta: int, A: np.ndarray, row_begin: int = 0,
                     rounding: int = RN, sr_seed: int = 0) -> None:
    A = _check_A(A)
    assert D.dtype == np.uint16 and D.shape == (d, A.shape[1]) and D.flags.c_contiguous
    _ok(lib().orc_seq16_accumulate(seed, d, zeta, _ptr(A), row_begin, A.shape[0], A.shape[1],
                                   A.strides[0] // 4, rounding, sr_seed, _ptr(D)))


def seq16_sketch(seed: int, d: int, zeta: int, A: np.ndarray, rounding: int = RN, sr_seed: int = 0,
                 row_begin: int = 0) -> np.ndarray:
    """Sequential FP16 accumulation in ascending (i, j) order -> uint16 bit patterns [d, n]."""
    D = np.zeros((d, A.shape[1]), dtype=np.uint16)
    seq16_accumulate(D, seed, d, zeta, A, row_begin, rounding, sr_seed)
    return D


def seqbf16_sketch(seed: int, d: int, zeta: int, A: np.ndarray, row_begin: int = 0) -> np.ndarray:
    """Sequential bfloat16 accumulation in ascending (i, j) order -> uint16 bit patterns [d, n]."""
    A = _check_A(A)
    D = np.zeros((d, A.shape[1]), dtype=np.uint16)
    _ok(lib().orc_seqbf16_accumulate(seed, d, zeta, _ptr(A), row_begin, A.shape[0], A.shape[1],
                                     A.strides[0] // 4, _ptr(D)))
    return D


def seq32_sketch(seed: int, d: int, zeta: int, A: np.ndarray, row_begin: int = 0) -> np.ndarray:
    A = _check_A(A)
    B = np.zeros((d, A.shape[1]), dtype=np.float32)
    _ok(lib().orc_seq32_accumulate(seed, d, zeta, _ptr(A), row_begin, A.shape[0], A.shape[1],
                                   A.strides[0] // 4, _ptr(B)))
    return B


def range_counts(zeta: int, A: np.ndarray) -> dict:
    A = _check_A(A)
    c = np.zeros(4, dtype=np.int64)
    _ok(lib().orc_range_counts(zeta, _ptr(A), A.shape[0], A.shape[1], A.strides[0] // 4, _ptr(c)))
    return {"n_sub": int(c[0]), "n_zero": int(c[1]), "n_convinf": int(c[2]), "n_contrib": int(c[3])}


# ---------------------------------------------------------------- F16C cross-check (pin only)
def has_f16c_crosscheck() -> bool:
    return hasattr(lib(), "orc_x_rn16_vs_f16c")


def rn16_vs_f16c(first: int, count: int, stride: int, threads: int):
    bad = C.c_uint32(0)
    n = lib().orc_x_rn16_vs_f16c(first, count, stride, threads, C.addressof(bad))
    return int(n), int(bad.value)


def add16_vs_f16c(v0: int, v_stride: int, threads: int):
    bad = C.c_uint32(0)
    n = lib().orc_x_add16_vs_f16c(v0, v_stride, threads, C.addressof(bad))
    return int(n), int(bad.value)


def bf16_vs_bits(first: int, count: int, stride: int, threads: int):
    bad = C.c_uint32(0)
    n = lib().orc_x_bf16_vs_bits(first, count, stride, threads, C.addressof(bad))
    return int(n), int(bad.value)


def bf16_add_vs_float(v0: int, v_stride: int, threads: int):
    bad = C.c_uint32(0)
    n = lib().orc_x_bf16_add_vs_float(v0, v_stride, threads, C.addressof(bad))
    return int(n), int(bad.value)
