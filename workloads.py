"""Seeded synthetic inputs shared by the tests, the bench and the smoke check.

This module holds NONE of the method's arithmetic (no hash, no rounding, no
sketching): it only produces input matrices, right-hand sides and seed
constants.  Both the CUDA path and the CPU oracle are fed the *same bytes*
made here; parity never depends on the generator being reproducible across
library versions, only on both sides seeing one buffer.

The paper's own workloads are synthetic as well (PAPER.md:318, :346, :362-366,
:380); the recipes below are the BASELINE.json `configs[0..4]` stand-ins, as
listed in DESIGN.md "Input recipe".
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass

import numpy as np


def sketch_seed(t: int) -> int:
    """Full-width 64-bit sketch seed number t (reading R15: never small consecutive seeds,
    because `seed ^ counter` aliases seeds that differ only in low bits)."""
    return int.from_bytes(hashlib.sha256(b"sparse-sketch-seed-%d" % t).digest()[:8], "little")


@dataclass(frozen=True)
class Config:
    name: str
    m: int
    n: int
    d: int
    zeta: int
    matrix_seed: int


# BASELINE.json configs[0..4]; config 3 and 4 sweep zeta / d around these defaults.
CONFIGS = {
    "c1": Config("c1", 4096, 16, 32, 4, 0),
    "c2": Config("c2", 1 << 20, 64, 128, 4, 1),
    "c3": Config("c3", 1 << 22, 128, 256, 4, 2),
    "c4": Config("c4", 1 << 23, 256, 512, 4, 3),
    "c5": Config("c5", 1 << 25, 128, 256, 4, 4),
}


# ----------------------------------------------------------------------------- numpy (host)
def gaussian(m: int, n: int, seed: int, pow2: int = 0) -> np.ndarray:
    """A ~ i.i.d. N(0,1) FP32 row-major, times 2**pow2 (exact in FP32)."""
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((m, n), dtype=np.float32)
    if pow2:
        A = np.ldexp(A, pow2).astype(np.float32)
    return A


def integer_valued(m: int, n: int, seed: int, lo: int = -3, hi: int = 3) -> np.ndarray:
    """Entries uniform in {lo..hi}: with zeta in {1,4} every FP16 partial sum is exact in any order."""
    rng = np.random.default_rng(seed)
    return rng.integers(lo, hi + 1, size=(m, n)).astype(np.float32)


def heavy_rows(m: int, n: int, alpha: float, seed: int) -> np.ndarray:
    """Config 3 (reading R16): G ~ N(0,1); permutation pi from the matrix seed;
    A[pi(i), :] = (1+i)^(-alpha) * G[pi(i), :]  -- heavy-leverage rows at random positions."""
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((m, n), dtype=np.float32)
    pi = rng.permutation(m)
    w = np.empty(m, dtype=np.float64)
    w[pi] = (1.0 + np.arange(m, dtype=np.float64)) ** (-alpha)
    A *= w.astype(np.float32)[:, None]
    return A


def ls_system(m: int, n: int, seed: int, sigma_min: float = 1e-4, noise: float = 1e-3):
    """Config 4: A = G diag(sigma), sigma geometric 1 -> sigma_min; b = A x* + noise*N(0,1)."""
    rng = np.random.default_rng(seed)
    sigma = np.geomspace(1.0, sigma_min, n).astype(np.float32)
    A = rng.standard_normal((m, n), dtype=np.float32) * sigma[None, :]
    xstar = rng.standard_normal(n)
    b = (A.astype(np.float64) @ xstar + noise * rng.standard_normal(m)).astype(np.float32)
    return A, b, xstar


def ls_paper_low_coherence(m: int, n: int, seed: int):
    """The paper's low-coherence least-squares family: singular values decreasing linearly from 100 to 1,
    b = A 1 + nu, nu_i ~ N(0, 0.1^2).  Built as A = (G / sqrt(m)) diag(sigma): for m >> n the Gaussian factor has
    nearly orthonormal columns, so the singular values are sigma up to O(sqrt(n/m))."""
    rng = np.random.default_rng(seed)
    sigma = np.linspace(100.0, 1.0, n)
    A = (rng.standard_normal((m, n), dtype=np.float32) * (sigma / np.sqrt(m)).astype(np.float32)[None, :]).astype(np.float32)
    b = (A.astype(np.float64) @ np.ones(n) + 0.1 * rng.standard_normal(m)).astype(np.float32)
    return A, b


def ls_paper_coherent(m: int, n: int, seed: int):
    """The paper's coherent family: A = [I_n; T], T = 1e-3 G / sqrt(m - n), b = [x0 + nu; T x0] with
    Gaussian G, x0, head noise nu_i ~ N(0, 0.5^2), and a common row permutation."""
    rng = np.random.default_rng(seed)
    A = np.empty((m, n), dtype=np.float32)
    A[:n] = np.eye(n, dtype=np.float32)
    A[n:] = rng.standard_normal((m - n, n), dtype=np.float32) * np.float32(1e-3 / np.sqrt(m - n))
    x0 = rng.standard_normal(n)
    b = np.empty(m, dtype=np.float64)
    b[:n] = x0 + 0.5 * rng.standard_normal(n)
    b[n:] = A[n:].astype(np.float64) @ x0
    pi = rng.permutation(m)
    return np.ascontiguousarray(A[pi]), b[pi].astype(np.float32)


# ----------------------------------------------------------------------------- torch (device)
def gaussian_device(m: int, n: int, seed: int, device, pow2: int = 0, chunk_rows: int = 1 << 22):
    """N(0,1) FP32 [m, n] generated on `device` in row chunks (no 2x peak memory)."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    A = torch.empty((m, n), dtype=torch.float32, device=device)
    for r0 in range(0, m, chunk_rows):
        r1 = min(m, r0 + chunk_rows)
        A[r0:r1].normal_(generator=g)
    if pow2:
        A.mul_(float(2.0 ** pow2))
    return A


def integer_valued_device(m: int, n: int, seed: int, device, lo: int = -3, hi: int = 3):
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return torch.randint(lo, hi + 1, (m, n), generator=g, device=device).to(torch.float32)


def sparse_signs_device(m: int, n: int, seed: int, device, density: float = 1.0 / 64, chunk_rows: int = 1 << 22):
    """Entries +-1 with probability `density`, else 0, FP32 [m, n] on `device`: integer-valued AND sparse, so that the
    sums of even 2^19-deep buckets stay far below 1024 and every FP16 partial sum is exact in any order."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    A = torch.empty((m, n), dtype=torch.float32, device=device)
    for r0 in range(0, m, chunk_rows):
        r1 = min(m, r0 + chunk_rows)
        u = torch.rand((r1 - r0, n), generator=g, device=device)
        A[r0:r1] = (u < density / 2).to(torch.float32) - (u > 1.0 - density / 2).to(torch.float32)
        del u
    return A


def heavy_rows_device(m: int, n: int, alpha: float, seed: int, device):
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    A = gaussian_device(m, n, seed + 1000003, device)
    pi = torch.randperm(m, generator=g, device=device)
    w = torch.empty(m, dtype=torch.float64, device=device)
    w[pi] = (1.0 + torch.arange(m, dtype=torch.float64, device=device)) ** (-alpha)
    A.mul_(w.to(torch.float32)[:, None])
    return A


def ls_system_device(m: int, n: int, seed: int, device, sigma_min: float = 1e-4, noise: float = 1e-3):
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    sigma = torch.from_numpy(np.geomspace(1.0, sigma_min, n).astype(np.float32)).to(device)
    A = gaussian_device(m, n, seed + 2000003, device)
    A.mul_(sigma[None, :])
    xstar = torch.randn(n, generator=g, device=device, dtype=torch.float64)
    b = torch.empty(m, dtype=torch.float32, device=device)
    step = 1 << 20
    for r0 in range(0, m, step):
        r1 = min(m, r0 + step)
        e = torch.randn(r1 - r0, generator=g, device=device, dtype=torch.float64)
        b[r0:r1] = (A[r0:r1].to(torch.float64) @ xstar + noise * e).to(torch.float32)
    return A, b, xstar


def ls_paper_low_coherence_device(m: int, n: int, seed: int, device):
    """Device form of `ls_paper_low_coherence`: A = (G / sqrt(m)) diag(sigma), sigma linear 100 -> 1,
    b = A 1 + 0.1 N(0,1).  Returns (A [m, n] FP32, b [m, 1] FP32)."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    sigma = torch.linspace(100.0, 1.0, n, dtype=torch.float64, device=device) / float(np.sqrt(m))
    A = gaussian_device(m, n, seed + 3000003, device)
    A.mul_(sigma.to(torch.float32)[None, :])
    b = torch.empty((m, 1), dtype=torch.float32, device=device)
    step = 1 << 18
    for r0 in range(0, m, step):
        r1 = min(m, r0 + step)
        e = torch.randn(r1 - r0, generator=g, device=device, dtype=torch.float64)
        b[r0:r1, 0] = (A[r0:r1].double().sum(dim=1) + 0.1 * e).to(torch.float32)
    return A, b


def ls_paper_coherent_device(m: int, n: int, seed: int, device):
    """Device form of `ls_paper_coherent`: A = [I_n; T] with T = 1e-3 G / sqrt(m - n), b = [x0 + nu; T x0],
    nu_i ~ N(0, 0.5^2), under one row permutation: the n unit rows land at seeded random positions.  Returns (A [m, n] FP32,
    b [m, 1] FP32)."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(seed)
    A = gaussian_device(m, n, seed + 4000003, device)
    A.mul_(float(1e-3 / np.sqrt(m - n)))
    x0 = torch.randn(n, generator=g, device=device, dtype=torch.float64)
    b = torch.empty((m, 1), dtype=torch.float32, device=device)
    step = 1 << 18
    for r0 in range(0, m, step):
        r1 = min(m, r0 + step)
        b[r0:r1, 0] = (A[r0:r1].double() @ x0).to(torch.float32)
    pos = torch.randperm(m, generator=g, device=device)[:n]          # where the identity rows sit
    A[pos] = torch.eye(n, dtype=torch.float32, device=device)
    b[pos, 0] = (x0 + 0.5 * torch.randn(n, generator=g, device=device, dtype=torch.float64)).to(torch.float32)
    return A, b


def coherence_basis_device(m: int, n: int, thetas, seed: int, device):
    """The paper's coherence sweep (Sec. V-C): U(theta) = orth((1 - theta) Q_rand + theta [I_n 0]^T) with
    Q_rand an orthogonalised m x n Gaussian matrix.  Yields (theta, U FP32 [m, n] on `device`, coherence of Eq. (2) =
    (m / n) max_i ||U_i||^2: between 1 and m / n, the coordinate subspace attains m / n).  The orthogonalisations run in FP64 (library QR), so U's columns are orthonormal to FP32 rounding;
    theta = 1 is the coordinate subspace [I_n 0]^T exactly."""
    import torch

    Q = gaussian_device(m, n, seed + 5000011, device).double()
    Q = torch.linalg.qr(Q, mode="reduced")[0]
    for theta in thetas:
        theta = float(theta)
        if theta >= 1.0:
            U = torch.zeros((m, n), dtype=torch.float64, device=device)
            U[:n] = torch.eye(n, dtype=torch.float64, device=device)
        else:
            M = Q * (1.0 - theta)
            M[:n] += theta * torch.eye(n, dtype=torch.float64, device=device)
            U = torch.linalg.qr(M, mode="reduced")[0] if theta > 0.0 else Q
            del M
        mu = float((U * U).sum(dim=1).max()) * m / n
        yield theta, U.to(torch.float32).contiguous(), mu    # library QR returns column-major factors
        del U
