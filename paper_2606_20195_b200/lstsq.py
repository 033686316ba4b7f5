"""Sketch-and-solve least squares on the GPU (Sec. V-D).

    "We sketch A in the chosen precision and b in FP32 with the same map, widen FP16 SA exactly, then use FP32 thin QR
     and a triangular solve."
    wall time = "shared-map SA, Sb, layout/promotion, FP32 QR, projection, and solve"

Stages and who runs them:
    SA, Sb ........... this library, ONE pass over the rows (sketch_apply_f{16,32}acc_with_rhs / sketch_apply_bf16acc)
    promotion ........ this library (sketch_widen; exact)
    FP32 thin QR ..... cuSOLVER geqrf through torch.geqrf (a library factorisation, as in the paper)
    projection ....... cuSOLVER ormqr through torch.ormqr: Q^T Sb from the Householder vectors -- Q is never formed
    solve ............ cuBLAS trsm through torch.linalg.solve_triangular
The sketch is the product; the factorisation and the solve are library calls composed here, not re-implemented.
"""
from __future__ import annotations

from .binding import Sketch, sketch_widen

PRECISIONS = ("f16", "f32", "bf16")


def sketch_system(sk: Sketch, A, b, precision: str = "f16", SA=None, Sb=None, stream=None, **opts):
    """(SA in the chosen precision, Sb in FP32) with the same map.  f16 / f32: one fused pass; bf16 (the control of
    PAPER.md:396): the bfloat16 apply, then b through the FP32 path."""
    if precision == "f16":
        return sk.apply_f16acc_with_rhs(A, b, out=SA, Sb=Sb, stream=stream, **opts)
    if precision == "f32":
        return sk.apply_f32acc_with_rhs(A, b, out=SA, Sb=Sb, stream=stream, **opts)
    if precision == "bf16":
        SA = sk.apply_bf16acc(A, out=SA, stream=stream, **opts) if opts else sk.apply_bf16acc(A, out=SA, stream=stream)
        col = b.unsqueeze(1)
        Sb2 = Sb.unsqueeze(1) if Sb is not None else None
        Sb = (sk.apply_f32acc(col, out=Sb2, stream=stream, **opts) if opts else sk.apply_f32acc(col, out=Sb2, stream=stream))[:, 0]
        return SA, Sb
    raise ValueError("precision must be one of %s" % (PRECISIONS,))


def solve_sketched(SA, Sb, W=None, stream=None):
    """x = argmin ||SA x - Sb||_2 in FP32: exact promotion, Householder QR, Q^T Sb, back substitution.  W: optional
    FP32 d x n workspace for the promoted copy.  stream: the torch stream SA and Sb were produced on (None = the current
    one); the promotion and the library calls are issued on that same stream, so they are ordered behind the sketch, and the
    returned vector is ready on it."""
    import torch

    st = stream if stream is not None else torch.cuda.current_stream()
    with torch.cuda.stream(st):
        M = SA if SA.dtype == torch.float32 else sketch_widen(SA, out=W, stream=st)
        n = M.shape[1]
        a, tau = torch.geqrf(M)
        y = torch.ormqr(a, tau, Sb.reshape(-1, 1), left=True, transpose=True)[:n]
        return torch.linalg.solve_triangular(a[:n].triu(), y, upper=True)[:, 0]


def sketch_and_solve(sk: Sketch, A, b, precision: str = "f16", SA=None, Sb=None, W=None, stream=None, **opts):
    """The complete pipeline of PAPER.md:356 on device buffers; returns the FP32 solution vector (length n).  Every stage
    runs on `stream` (None = torch's current stream); with a side stream the caller orders its own reads of the result
    behind that stream, as for any torch op issued there."""
    import torch

    st = stream if stream is not None else torch.cuda.current_stream()
    with torch.cuda.stream(st):       # the buffers sketch_system allocates belong to the stream that fills them
        SA, Sb = sketch_system(sk, A, b, precision, SA=SA, Sb=Sb, stream=st, **opts)
    return solve_sketched(SA, Sb, W=W, stream=st)
