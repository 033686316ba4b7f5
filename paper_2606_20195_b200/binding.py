"""ctypes binding of include/sparse_sketch.h -- argument marshalling only.

The method names mirror the C entry points (sketch_create -> Sketch(...), sketch_apply_f16acc ->
Sketch.apply_f16acc, ...).  Tensors are torch CUDA tensors (device memory + streams are PyTorch's
job here); only their data pointers, sizes and the current stream handle cross the boundary.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

from . import _build

RN, SR, DITHER = 0, 1, 2
VARIANT_AUTO, VARIANT_FLAT_PAIR, VARIANT_FLAT_VEC, VARIANT_SMEM, VARIANT_GENERIC, VARIANT_TMEM, VARIANT_SMALL = 0, 1, 2, 3, 4, 5, 6
VARIANT_NAMES = {0: "auto", 1: "flat_pair", 2: "flat_vec", 3: "smem", 4: "generic", 5: "tmem", 6: "small"}


class SketchOpts(C.Structure):
    _fields_ = [
        ("variant", C.c_int32),
        ("replicas", C.c_int32),
        ("hash_mode", C.c_int32),
        ("accumulate", C.c_int32),
        ("row_begin", C.c_int64),
        ("rows", C.c_int64),
        ("grid_ctas", C.c_int32),
        ("tmem_group_mode", C.c_int32),
    ]


class SketchError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        detail = lib().sketch_last_error().decode() if code in (-7, -9, -10) else ""
        super().__init__("%s failed: %s (%d) %s" % (where, lib().sketch_strerror(code).decode(), code, detail))


_lib = None

# every symbol include/sparse_sketch.h declares: name -> (restype, argtypes)
_vp, _i32, _i64, _u64, _int = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_int
_OP = C.POINTER(SketchOpts)
SYMBOLS = {
    "sketch_create": (_int, [_i64, _i32, _i32, _u64, C.POINTER(_vp)]),
    "sketch_destroy": (_int, [_vp]),
    "sketch_hashes_dump": (_int, [_vp, _vp, _vp, _vp]),
    "sketch_precompute_hashes": (_int, [_vp, _vp]),
    "sketch_apply_f32acc": (_int, [_vp, _vp, _i32, _i64, _vp, _vp]),
    "sketch_apply_f16acc": (_int, [_vp, _vp, _i32, _i64, _vp, _int, _u64, _vp]),
    "sketch_apply_bf16acc": (_int, [_vp, _vp, _i32, _i64, _vp, _vp]),
    "sketch_apply_f16acc_noalloc": (_int, [_vp, _vp, _i32, _i64, _vp, _int, _u64, _vp]),
    "sketch_apply_bf16acc_ex": (_int, [_vp, _vp, _i32, _i64, _vp, _OP, _vp]),
    "sketch_apply_f16acc_with_rhs": (_int, [_vp, _vp, _i32, _i64, _vp, _vp, _vp, _OP, _vp]),
    "sketch_apply_f32acc_with_rhs": (_int, [_vp, _vp, _i32, _i64, _vp, _vp, _vp, _OP, _vp]),
    "sketch_widen": (_int, [_vp, _i64, _int, _vp, _vp]),
    "sketch_apply_f32acc_ex": (_int, [_vp, _vp, _i32, _i64, _vp, _OP, _vp]),
    "sketch_apply_f16acc_ex": (_int, [_vp, _vp, _i32, _i64, _vp, _int, _u64, _OP, _vp]),
    "sketch_apply_f32acc_host": (_int, [_vp, _vp, _i32, _i64, _vp, _OP]),
    "sketch_apply_f16acc_host": (_int, [_vp, _vp, _i32, _i64, _vp, _int, _u64, _OP]),
    "sketch_red_probe": (_int, [_vp, _i32, _i32, _i32, _i32, _i32, _i32, C.POINTER(_u64), _vp]),
    "sketch_convert_probe": (_int, [_vp, _vp, _i64, _i32, _vp, _vp]),
    "sketch_stream_probe": (_int, [_vp, _i64, _i32, _i32, _vp, _vp]),
    "sketch_plan": (_int, [_vp, _i32, _i64, _int, _int, _OP, C.POINTER(_i32), C.POINTER(_i32), C.POINTER(_i32), C.POINTER(_i32)]),
    "sketch_launch_count": (_u64, []),
    "sketch_strerror": (C.c_char_p, [_int]),
    "sketch_last_error": (C.c_char_p, []),
    "sketch_version": (C.c_char_p, []),
}


def library_path() -> Path:
    return _build.LIB


def lib() -> C.CDLL:
    """Load (building in-tree if stale) libsparse_sketch.so; raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(str(path))
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)  # AttributeError if the library does not export it
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def sketch_strerror(code: int) -> str:
    return lib().sketch_strerror(code).decode()


def sketch_version() -> str:
    return lib().sketch_version().decode()


def sketch_launch_count() -> int:
    return int(lib().sketch_launch_count())


def _stream_ptr(stream=None) -> int:
    import torch

    st = stream if stream is not None else torch.cuda.current_stream()
    return int(st.cuda_stream)


def _opts(variant=0, replicas=0, hash_mode=0, accumulate=False, row_begin=0, rows=0, grid_ctas=0, tmem_group_mode=0):
    return SketchOpts(int(variant), int(replicas), int(hash_mode), int(bool(accumulate)), int(row_begin), int(rows),
                      int(grid_ctas), int(tmem_group_mode))


def _check_cuda(t, dtype, what):
    if not t.is_cuda or t.dtype != dtype:
        raise TypeError("%s must be a CUDA tensor of dtype %s" % (what, dtype))


def sketch_red_probe(scratch, d: int, n: int, kind: int, replicas: int, grid_ctas: int, iters: int, stream=None) -> int:
    """Launch the L2 atomic-throughput probe; returns the number of lane-level RED ops issued."""
    ops = _u64(0)
    rc = lib().sketch_red_probe(scratch.data_ptr(), d, n, kind, replicas, grid_ctas, iters, C.byref(ops), _stream_ptr(stream))
    if rc:
        raise SketchError(rc, "sketch_red_probe")
    return int(ops.value)


def sketch_stream_probe(src, kind: int = 1, grid_ctas: int = 0, stream=None) -> int:
    """Read the CUDA tensor `src` once and discard it (sketch_stream_probe); returns the bytes read.  Time it with events."""
    import torch

    if not src.is_cuda or not src.is_contiguous():
        raise TypeError("src must be a contiguous CUDA tensor")
    nbytes = src.numel() * src.element_size()
    if grid_ctas <= 0:
        sms = torch.cuda.get_device_properties(src.device).multi_processor_count
        grid_ctas = sms if kind == 1 else sms * 8
    rc = lib().sketch_stream_probe(src.data_ptr(), nbytes, kind, grid_ctas, None, _stream_ptr(stream))
    if rc:
        raise SketchError(rc, "sketch_stream_probe")
    return nbytes // 32768 * 32768 if kind == 1 else nbytes // 32 * 32


def sketch_widen(B16, out=None, stream=None):
    """Exact FP32 copy of a binary16 / bfloat16 sketch (sketch_widen)."""
    import torch

    if not B16.is_cuda or B16.dtype not in (torch.float16, torch.bfloat16) or not B16.is_contiguous():
        raise TypeError("B16 must be a contiguous CUDA tensor of dtype float16 or bfloat16")
    if out is None:
        out = torch.empty(B16.shape, dtype=torch.float32, device=B16.device)
    _check_cuda(out, torch.float32, "out")
    assert out.is_contiguous() and out.numel() == B16.numel()
    rc = lib().sketch_widen(B16.data_ptr(), B16.numel(), int(B16.dtype == torch.bfloat16), out.data_ptr(), _stream_ptr(stream))
    if rc:
        raise SketchError(rc, "sketch_widen")
    return out


def sketch_convert_probe(p, rbits, kind: int, out=None, stream=None):
    """The conversion step alone (sketch_convert_probe): p FP32 CUDA tensor, rbits int32 CUDA tensor of the same size or
    None; returns the 16-bit patterns as an int16 tensor."""
    import torch

    _check_cuda(p, torch.float32, "p")
    if rbits is not None:
        _check_cuda(rbits, torch.int32, "rbits")
        assert rbits.is_contiguous() and rbits.numel() == p.numel()
    assert p.is_contiguous()
    if out is None:
        out = torch.empty(p.shape, dtype=torch.int16, device=p.device)
    rc = lib().sketch_convert_probe(p.data_ptr(), rbits.data_ptr() if rbits is not None else None, p.numel(), kind, out.data_ptr(),
                                    _stream_ptr(stream))
    if rc:
        raise SketchError(rc, "sketch_convert_probe")
    return out


class Sketch:
    """Owns one sketch_t handle (sketch_create / sketch_destroy)."""

    def __init__(self, m: int, d: int, zeta: int, seed: int):
        h = _vp()
        rc = lib().sketch_create(m, d, zeta, seed & (2**64 - 1), C.byref(h))
        if rc:
            raise SketchError(rc, "sketch_create")
        self._h = h
        self.m, self.d, self.zeta, self.seed = m, d, zeta, seed

    def close(self):
        if getattr(self, "_h", None):
            lib().sketch_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- hash stage
    def hashes_dump(self, stream=None):
        import torch

        bucket = torch.empty((self.m, self.zeta), dtype=torch.int32, device="cuda")
        sign = torch.empty((self.m, self.zeta), dtype=torch.uint8, device="cuda")
        rc = lib().sketch_hashes_dump(self._h, bucket.data_ptr(), sign.data_ptr(), _stream_ptr(stream))
        if rc:
            raise SketchError(rc, "sketch_hashes_dump")
        return bucket, sign

    def precompute_hashes(self, stream=None):
        rc = lib().sketch_precompute_hashes(self._h, _stream_ptr(stream))
        if rc:
            raise SketchError(rc, "sketch_precompute_hashes")

    # ---- device-buffer applies
    def _A_args(self, A):
        import torch

        _check_cuda(A, torch.float32, "A")
        if A.dim() != 2 or A.stride(1) != 1:
            raise ValueError("A must be 2-D row-major (unit column stride)")
        return A.data_ptr(), int(A.shape[1]), int(A.stride(0)) if A.shape[0] > 1 else max(int(A.stride(0)), int(A.shape[1]))

    def _range_opts(self, A, opts):
        """rows defaults to the rows of A.  The ABI reads rows = 0 as "through row m - 1", so an EMPTY A is passed as the
        empty range that starts at m (nothing is read; B is zeroed unless accumulate is set)."""
        opts = dict(opts)
        opts.setdefault("rows", int(A.shape[0]))
        if int(opts["rows"]) == 0:
            if int(A.shape[0]) != 0:
                raise ValueError("rows=0 is ambiguous: pass the number of rows of A")
            opts["row_begin"] = self.m
        return opts

    def apply_f32acc(self, A, out=None, stream=None, **opts):
        import torch

        ap, n, lda = self._A_args(A)
        if out is None:
            out = torch.empty((self.d, n), dtype=torch.float32, device=A.device)
        _check_cuda(out, torch.float32, "out")
        assert out.is_contiguous() and tuple(out.shape) == (self.d, n)
        if opts:
            o = _opts(**self._range_opts(A, opts))
            rc = lib().sketch_apply_f32acc_ex(self._h, ap, n, lda, out.data_ptr(), C.byref(o), _stream_ptr(stream))
        else:
            if A.shape[0] != self.m:
                raise ValueError("A has %d rows, sketch was created for m=%d (pass row_begin=/rows= for a slice)" % (A.shape[0], self.m))
            rc = lib().sketch_apply_f32acc(self._h, ap, n, lda, out.data_ptr(), _stream_ptr(stream))
        if rc:
            raise SketchError(rc, "sketch_apply_f32acc")
        return out

    def apply_f16acc(self, A, out=None, rounding: int = RN, sr_seed: int = 0, stream=None, **opts):
        import torch

        ap, n, lda = self._A_args(A)
        if out is None:
            out = torch.empty((self.d, n), dtype=torch.float16, device=A.device)
        _check_cuda(out, torch.float16, "out")
        assert out.is_contiguous() and tuple(out.shape) == (self.d, n)
        if opts:
            o = _opts(**self._range_opts(A, opts))
            rc = lib().sketch_apply_f16acc_ex(self._h, ap, n, lda, out.data_ptr(), rounding, sr_seed & (2**64 - 1), C.byref(o),
                                              _stream_ptr(stream))
        else:
            if A.shape[0] != self.m:
                raise ValueError("A has %d rows, sketch was created for m=%d (pass row_begin=/rows= for a slice)" % (A.shape[0], self.m))
            rc = lib().sketch_apply_f16acc(self._h, ap, n, lda, out.data_ptr(), rounding, sr_seed & (2**64 - 1), _stream_ptr(stream))
        if rc:
            raise SketchError(rc, "sketch_apply_f16acc")
        return out

    def apply_f16acc_noalloc(self, A, out, rounding: int = RN, sr_seed: int = 0, stream=None):
        """sketch_apply_f16acc_noalloc: the complete FP16 sketch of A (all m rows) for callers that may not allocate device
        memory while running -- the partial sketches live in an 8 MiB array built into the library instead of a
        cudaMalloc'ed buffer.  `out` is required (this wrapper allocates nothing either).  Raises SketchError -9 when two
        partial sketches of d x n do not fit that array.  All calls on a device share the array: do not let two overlap."""
        import torch

        ap, n, lda = self._A_args(A)
        _check_cuda(out, torch.float16, "out")
        assert out.is_contiguous() and tuple(out.shape) == (self.d, n)
        if A.shape[0] != self.m:
            raise ValueError("A has %d rows, sketch was created for m=%d" % (A.shape[0], self.m))
        rc = lib().sketch_apply_f16acc_noalloc(self._h, ap, n, lda, out.data_ptr(), rounding, sr_seed & (2**64 - 1), _stream_ptr(stream))
        if rc:
            raise SketchError(rc, "sketch_apply_f16acc_noalloc")
        return out

    def apply_bf16acc(self, A, out=None, stream=None, **opts):
        import torch

        ap, n, lda = self._A_args(A)
        if out is None:
            out = torch.empty((self.d, n), dtype=torch.bfloat16, device=A.device)
        _check_cuda(out, torch.bfloat16, "out")
        assert out.is_contiguous() and tuple(out.shape) == (self.d, n)
        if opts:
            o = _opts(**self._range_opts(A, opts))
            rc = lib().sketch_apply_bf16acc_ex(self._h, ap, n, lda, out.data_ptr(), C.byref(o), _stream_ptr(stream))
        else:
            if A.shape[0] != self.m:
                raise ValueError("A has %d rows, sketch was created for m=%d (pass row_begin=/rows= for a slice)" % (A.shape[0], self.m))
            rc = lib().sketch_apply_bf16acc(self._h, ap, n, lda, out.data_ptr(), _stream_ptr(stream))
        if rc:
            raise SketchError(rc, "sketch_apply_bf16acc")
        return out

    # ---- least-squares front end: [A | b] in one pass, exact widening
    def _with_rhs(self, name, dtype, A, b, out, Sb, stream, opts):
        import torch

        ap, n, lda = self._A_args(A)
        _check_cuda(b, torch.float32, "b")
        if b.dim() != 1 or not b.is_contiguous() or b.shape[0] != A.shape[0]:
            raise ValueError("b must be a contiguous vector with one entry per row of A")
        if out is None:
            out = torch.empty((self.d, n), dtype=dtype, device=A.device)
        if Sb is None:
            Sb = torch.empty((self.d,), dtype=torch.float32, device=A.device)
        _check_cuda(out, dtype, "out")
        _check_cuda(Sb, torch.float32, "Sb")
        assert out.is_contiguous() and tuple(out.shape) == (self.d, n) and Sb.is_contiguous() and tuple(Sb.shape) == (self.d,)
        o = _opts(**self._range_opts(A, opts))
        rc = getattr(lib(), name)(self._h, ap, n, lda, b.data_ptr(), out.data_ptr(), Sb.data_ptr(), C.byref(o), _stream_ptr(stream))
        if rc:
            raise SketchError(rc, name)
        return out, Sb

    def apply_f16acc_with_rhs(self, A, b, out=None, Sb=None, stream=None, **opts):
        import torch

        return self._with_rhs("sketch_apply_f16acc_with_rhs", torch.float16, A, b, out, Sb, stream, opts)

    def apply_f32acc_with_rhs(self, A, b, out=None, Sb=None, stream=None, **opts):
        import torch

        return self._with_rhs("sketch_apply_f32acc_with_rhs", torch.float32, A, b, out, Sb, stream, opts)

    # ---- host-buffer applies (end-to-end: H2D streaming + kernels + D2H inside the call)
    def apply_f16acc_host(self, A_host, out_host=None, rounding: int = RN, sr_seed: int = 0, **opts):
        import torch

        assert not A_host.is_cuda and A_host.dtype == torch.float32 and A_host.dim() == 2 and A_host.stride(1) == 1
        n = int(A_host.shape[1])
        if out_host is None:
            out_host = torch.empty((self.d, n), dtype=torch.float16, pin_memory=True)
        assert not out_host.is_cuda and out_host.dtype == torch.float16 and out_host.is_contiguous()
        o = _opts(**self._range_opts(A_host, opts))
        rc = lib().sketch_apply_f16acc_host(self._h, A_host.data_ptr(), n, int(A_host.stride(0)), out_host.data_ptr(), rounding,
                                            sr_seed & (2**64 - 1), C.byref(o))
        if rc:
            raise SketchError(rc, "sketch_apply_f16acc_host")
        return out_host

    def apply_f32acc_host(self, A_host, out_host=None, **opts):
        import torch

        assert not A_host.is_cuda and A_host.dtype == torch.float32 and A_host.dim() == 2 and A_host.stride(1) == 1
        n = int(A_host.shape[1])
        if out_host is None:
            out_host = torch.empty((self.d, n), dtype=torch.float32, pin_memory=True)
        assert not out_host.is_cuda and out_host.dtype == torch.float32 and out_host.is_contiguous()
        o = _opts(**self._range_opts(A_host, opts))
        rc = lib().sketch_apply_f32acc_host(self._h, A_host.data_ptr(), n, int(A_host.stride(0)), out_host.data_ptr(), C.byref(o))
        if rc:
            raise SketchError(rc, "sketch_apply_f32acc_host")
        return out_host

    # ---- planning (host only)
    def plan(self, n: int, lda: int | None = None, f16=True, rounding: int = RN, **opts):
        """f16: False / 0 = f32acc, True / 1 = f16acc, 2 = bf16acc."""
        v, p, h, g = _i32(0), _i32(0), _i32(0), _i32(0)
        o = _opts(**opts)
        rc = lib().sketch_plan(self._h, n, lda or n, int(f16), rounding, C.byref(o), C.byref(v), C.byref(p), C.byref(h), C.byref(g))
        if rc:
            raise SketchError(rc, "sketch_plan")
        return {"variant": VARIANT_NAMES[v.value], "replicas": p.value, "hash_mode": h.value, "grid": g.value}
