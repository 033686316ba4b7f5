"""Host-side FP64 evaluation of a returned sketch (not part of the hot path, no method arithmetic).

These are the downstream quantities BASELINE.json:north_star asks to be "computed on the host
from the GPU sketch": subspace distortion (Eq. 4) and the sketch-and-solve
least-squares residual ratio.  numpy/LAPACK in FP64 only; used identically on
GPU sketches and oracle sketches by tests/ and bench.py.
"""
from __future__ import annotations

import numpy as np


def rel_fro(X, ref) -> float:
    """||X - ref||_F / ||ref||_F over entries finite in both (reading R18)."""
    X = np.asarray(X, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    ok = np.isfinite(X) & np.isfinite(ref)
    den = np.linalg.norm(ref[ok])
    return float(np.linalg.norm((X - ref)[ok]) / den) if den > 0 else float(np.linalg.norm((X - ref)[ok]))


def gram_R(A_chunks, n: int) -> np.ndarray:
    """Upper-triangular R with A = Q R, from streamed FP64 QR of row chunks (TSQR, reading R17)."""
    R = np.zeros((0, n))
    for Ak in A_chunks:
        R = np.linalg.qr(np.vstack([R, np.asarray(Ak, dtype=np.float64)]), mode="r")
    return R


def distortion(D, R) -> float:
    """eta = max|sigma_i(D R^-1) - 1| (Eq. 4 applied to the returned matrix):
    for U = A R^-1 orthonormal, S U = (S A) R^-1 in exact arithmetic (reading R17)."""
    D = np.asarray(D, dtype=np.float64)
    X = np.linalg.solve(R.T, D.T).T  # D R^-1
    s = np.linalg.svd(X, compute_uv=False)
    return float(max(abs(s.max() - 1.0), abs(1.0 - s.min())))


def distortion_operator(D, R) -> np.ndarray:
    D = np.asarray(D, dtype=np.float64)
    return np.linalg.solve(R.T, D.T).T


def eta_of(X) -> float:
    """eta(X) = sup_{|v|=1} | ||Xv|| - 1 | (Prop. 2's extension of Eq. 4)."""
    s = np.linalg.svd(np.asarray(X, dtype=np.float64), compute_uv=False)
    return float(max(abs(s.max() - 1.0), abs(1.0 - s.min())))


def sketch_and_solve(SA, Sb) -> np.ndarray:
    """argmin ||SA x - Sb|| in FP64 (QR-based lstsq); the paper solves in FP32,
    BASELINE.json config 4 asks for the FP64 host solve."""
    x, *_ = np.linalg.lstsq(np.asarray(SA, dtype=np.float64), np.asarray(Sb, dtype=np.float64), rcond=None)
    return x


def residual_norm(A_chunks, b_chunks, x) -> float:
    acc = 0.0
    for Ak, bk in zip(A_chunks, b_chunks):
        r = np.asarray(Ak, dtype=np.float64) @ x - np.asarray(bk, dtype=np.float64)
        acc += float(r @ r)
    return float(np.sqrt(acc))
