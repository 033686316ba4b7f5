"""Pins for the oracle's hash stage: none of these compares the oracle with itself."""
import math
import os

import numpy as np
import pytest

import oracle
from workloads import sketch_seed

GOLD = os.path.join(os.path.dirname(__file__), "golden")
M64 = (1 << 64) - 1


def _lines(name):
    with open(os.path.join(GOLD, name)) as f:
        for ln in f:
            ln = ln.strip()
            if ln and not ln.startswith("#"):
                yield ln.split()


def test_splitmix64_published_vector():
    for x, want in _lines("splitmix64_vector.txt"):
        assert oracle.splitmix64(int(x, 16)) == int(want, 16)


def test_hash_golden_pins():
    # values fixed before any code existed; a wrong shift, precedence, sign bit or
    # counter (i*zeta+j vs j*m+i) fails here
    for tok in _lines("hash_pins.txt"):
        seed, d, zeta, i = int(tok[0], 0), int(tok[1]), int(tok[2]), int(tok[3])
        vals = list(map(int, tok[4:]))
        b, s = oracle.hashes(seed, d, zeta, 1, row_begin=i)
        assert b[0].tolist() == vals[0::2], (seed, d, zeta, i)
        assert s[0].tolist() == vals[1::2], (seed, d, zeta, i)


def test_hash_golden_aggregates():
    for tok in _lines("hash_aggregates.txt"):
        zeta, cmin, cmax, ssum = map(int, tok[:4])
        first8 = list(map(int, tok[4:]))
        b, s = oracle.hashes(0, 32, zeta, 4096)
        cnt = np.bincount(b.ravel(), minlength=32)
        assert (cnt.min(), cnt.max(), int(s.sum())) == (cmin, cmax, ssum)
        assert cnt[:8].tolist() == first8


def _py_splitmix64(x):
    z = (x + 0x9E3779B97F4A7C15) & M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
    return z ^ (z >> 31)


def test_hash_against_python_bigints_wraparound():
    # unbounded Python integers with explicit masking vs the C++ uint64 arithmetic, on counters
    # large enough that seed ^ ctr and the multiplies wrap (row 2^40, full-width seeds)
    rng = np.random.default_rng(7)
    for _ in range(200):
        seed = int(rng.integers(0, 1 << 63)) * 2 + int(rng.integers(0, 2))
        zeta = int(rng.choice([1, 2, 3, 4, 8, 16]))
        db = int(rng.integers(1, 5000))
        d = db * zeta
        i = int(rng.integers(0, 1 << 40))
        b, s = oracle.hashes(seed, d, zeta, 2, row_begin=i)
        for r in range(2):
            for j in range(zeta):
                h = _py_splitmix64(seed ^ ((i + r) * zeta + j))
                assert b[r, j] == j * db + (((h >> 32) * db) >> 32)
                assert s[r, j] == (h & 1)


@pytest.mark.parametrize("zeta,d", [(1, 32), (2, 64), (4, 32), (8, 256), (3, 30)])
def test_one_bucket_per_block(zeta, d):
    # block t draws its target inside its own d/zeta rows -> exactly zeta nonzeros
    # per column of S, one per block
    b, s = oracle.hashes(sketch_seed(3), d, zeta, 5000)
    db = d // zeta
    j = np.arange(zeta)[None, :]
    assert np.all(b >= j * db) and np.all(b < (j + 1) * db)
    assert set(np.unique(s)) <= {0, 1}


def test_rejects_d_not_divisible():
    with pytest.raises(ValueError):
        oracle.hashes(1, 30, 4, 8)  # PAPER.md:59 "Let d be divisible by zeta"


@pytest.mark.parametrize("n,d,want", [(8, 64, 0.63403), (16, 256, 0.61971)])
def test_birthday_full_rank_probability_eq3(n, d, want):
    # Eq. (3): for zeta=1 and U=[I_n 0]^T, Pr{rank(SU)=n} = prod_{j<n}(1-j/d):
    # the fraction of seeds whose first n rows land in n distinct buckets.
    closed = math.prod(1 - j / d for j in range(n))
    assert abs(closed - want) < 5e-6
    N = 12000
    hits = 0
    for t in range(N):
        b, _ = oracle.hashes(sketch_seed(1000 + t), d, 1, n)
        hits += len(set(b[:, 0].tolist())) == n
    p = hits / N
    sigma = math.sqrt(closed * (1 - closed) / N)
    assert abs(p - closed) < 4.5 * sigma, (p, closed, sigma)


def test_uniformity_and_depth():
    # mean bucket depth m*zeta/d and a chi-square uniformity test per block
    m, d, zeta = 1 << 16, 256, 4
    b, s = oracle.hashes(sketch_seed(5), d, zeta, m)
    cnt = np.bincount(b.ravel(), minlength=d)
    assert cnt.sum() == m * zeta and abs(cnt.mean() - m * zeta / d) < 1e-9
    exp = m * zeta / d
    chi2 = ((cnt - exp) ** 2 / exp).sum()
    dof = d - zeta
    assert abs(chi2 - dof) < 5 * math.sqrt(2 * dof), chi2
    # equiprobable signs, and sign independent of bucket parity
    frac = s.mean()
    assert abs(frac - 0.5) < 5 * 0.5 / math.sqrt(m * zeta)
    par = ((b & 1) ^ s).mean()
    assert abs(par - 0.5) < 5 * 0.5 / math.sqrt(m * zeta)


def test_row_begin_is_a_pure_offset():
    b0, s0 = oracle.hashes(sketch_seed(9), 128, 4, 300)
    b1, s1 = oracle.hashes(sketch_seed(9), 128, 4, 100, row_begin=150)
    assert np.array_equal(b0[150:250], b1) and np.array_equal(s0[150:250], s1)


def test_low_bit_seed_aliasing_documented():
    # reading R15: seeds that differ only below bit log2(zeta) permute the blocks' counters --
    # seed^1 swaps (i,0)<->(i,1) and (i,2)<->(i,3); this is why sketch seeds are full-width.
    b0, s0 = oracle.hashes(8, 32, 4, 64)
    b1, s1 = oracle.hashes(9, 32, 4, 64)
    db = 8
    assert np.array_equal(b0[:, 0] % db, b1[:, 1] % db) and np.array_equal(s0[:, 0], s1[:, 1])
