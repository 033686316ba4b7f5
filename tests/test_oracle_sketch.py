"""Pins for the oracle's sketch modes (F64 / BQ / BC / SEQ16 / SEQ32 / SR / range counts)."""
import math

import numpy as np
import pytest

import evaluation as ev
import oracle
import workloads as wl
from workloads import sketch_seed

U = 2.0 ** -11
H = 2.0 ** -24


@pytest.mark.parametrize("zeta,d,m,n", [(1, 8, 40, 5), (2, 12, 50, 3), (3, 12, 37, 4), (4, 32, 64, 6), (8, 32, 33, 2)])
def test_f64_mode_equals_dense_S_times_A(zeta, d, m, n):
    # brute force: materialise S of Eq. (1) and multiply with numpy's matmul
    seed = sketch_seed(zeta)
    A = wl.gaussian(m, n, 11)
    S = oracle.dense_S(seed, m, d, zeta)
    # structure of S: zeta nonzeros per column, one per block, magnitude 1/sqrt(zeta)
    nz = S != 0
    assert np.all(nz.sum(axis=0) == zeta)
    db = d // zeta
    for j in range(zeta):
        assert np.all(nz[j * db:(j + 1) * db].sum(axis=0) == 1)
    assert np.allclose(np.abs(S[nz]), 1 / math.sqrt(zeta), rtol=1e-15)
    B = oracle.f64_sketch(seed, d, zeta, A)
    assert np.allclose(B, S @ A.astype(np.float64), rtol=1e-13, atol=1e-13)
    # and S is what the hash says (a transposed operand or swapped index fails here)
    b, s = oracle.hashes(seed, d, zeta, m)
    for i in (0, m // 2, m - 1):
        for j in range(zeta):
            assert S[b[i, j], i] == (-1 if s[i, j] else 1) / math.sqrt(zeta)


def test_expected_squared_norm_is_preserved():
    # PAPER.md:63 "E||Sv||^2 = ||v||^2": mean over 1000 full-width seeds within 1% (BASELINE north_star);
    # 16 Gaussian columns so the mean's std is ~0.002
    A = wl.gaussian(4096, 16, 0)
    na = np.linalg.norm(A.astype(np.float64)) ** 2
    for zeta in (4, 1):
        r = [np.linalg.norm(oracle.f64_sketch(sketch_seed(t), 32, zeta, A)) ** 2 / na for t in range(1000)]
        assert abs(np.mean(r) - 1.0) < 0.01, np.mean(r)
        assert 0.01 < np.std(r) < 0.2  # it is random, not trivially 1


def test_f64_scaling_by_power_of_two_is_exact():
    # config 5 needs one FP64 pass for all k: S(2^k A) = 2^k S A exactly
    A = wl.gaussian(500, 8, 5)
    B0 = oracle.f64_sketch(sketch_seed(1), 64, 4, A)
    for k in (-24, 12):
        Bk = oracle.f64_sketch(sketch_seed(1), 64, 4, np.ldexp(A, k).astype(np.float32))
        assert np.array_equal(Bk, np.ldexp(B0, k))


def test_chunked_rows_and_threads_and_lda():
    seed, d, zeta = sketch_seed(2), 48, 4
    A = wl.gaussian(1000, 12, 6)
    B = oracle.f64_sketch(seed, d, zeta, A)
    Bc = np.zeros_like(B)
    for r0, r1 in ((0, 10), (10, 611), (611, 1000)):
        oracle.f64_accumulate(Bc, seed, d, zeta, A[r0:r1], row_begin=r0)
    oracle.f64_finalize(Bc, zeta)
    assert np.allclose(B, Bc, rtol=1e-14, atol=1e-14)
    assert np.allclose(B, oracle.f64_sketch(seed, d, zeta, A, threads=4), rtol=1e-13, atol=1e-13)
    # SEQ16 state carries across chunks bit-exactly (same ascending order)
    D = oracle.seq16_sketch(seed, d, zeta, A)
    Dc = np.zeros_like(D)
    for r0, r1 in ((0, 10), (10, 611), (611, 1000)):
        oracle.seq16_accumulate(Dc, seed, d, zeta, A[r0:r1], row_begin=r0)
    assert np.array_equal(D, Dc)
    # padded rows (lda > n) read only the first n columns
    Ap = np.full((1000, 20), np.nan, dtype=np.float32)
    Ap[:, :12] = A
    assert np.array_equal(oracle.seq16_sketch(seed, d, zeta, Ap[:, :12]), D)


@pytest.mark.parametrize("zeta", [4, 1])
def test_integer_valued_input_is_exact_in_every_mode(zeta):
    # SURVEY 8c / PAPER.md:225: scale 1/2 (zeta=4) or 1 (zeta=1) is exact; entries in {-3..3};
    # every partial sum is a multiple of 1/2 bounded well below 2048*(1/2), hence exact in FP16
    # in any order: SEQ16 == RN16(F64) == SEQ32 bit for bit.
    A = wl.integer_valued(4096, 16, 0)
    seed = sketch_seed(0)
    B = oracle.f64_sketch(seed, 32, zeta, A)
    assert np.abs(B).max() < 1024
    D = oracle.seq16_sketch(seed, 32, zeta, A)
    assert np.array_equal(oracle.half_bits_to_f64(D), B)
    assert np.array_equal(oracle.seq32_sketch(seed, 32, zeta, A).astype(np.float64), B)
    assert np.array_equal(oracle.f64_sketch(seed, 32, zeta, A, mode=oracle.BC), B)


@pytest.mark.parametrize("zeta", [1, 2, 4])
def test_seq16_against_numpy_float16_loop(zeta):
    # Listing 2 retyped with numpy scalar types on a tiny case:
    # float32 product -> float16 (RN) -> float16 += (numpy rounds each half add once)
    m, n, d = 96, 4, 8
    seed = sketch_seed(20 + zeta)
    A = wl.gaussian(m, n, 21)
    b, s = oracle.hashes(seed, d, zeta, m)
    sc = np.float32(1.0 / math.sqrt(zeta))
    D = np.zeros((d, n), dtype=np.float16)
    B32 = np.zeros((d, n), dtype=np.float32)
    for i in range(m):
        for j in range(zeta):
            es = np.float32(-sc if s[i, j] else sc)
            for c in range(n):
                p = np.float32(es * A[i, c])
                D[b[i, j], c] = np.float16(D[b[i, j], c] + np.float16(p))
                B32[b[i, j], c] = np.float32(B32[b[i, j], c] + p)
    assert np.array_equal(oracle.seq16_sketch(seed, d, zeta, A), D.view(np.uint16))
    assert np.array_equal(oracle.seq32_sketch(seed, d, zeta, A), B32)


def test_scale_bits():
    # reading R5: s = fp32(1/sqrt(zeta)) correctly rounded; SURVEY 8c row 5 bit patterns
    want = {1: 0x3F800000, 2: 0x3F3504F3, 4: 0x3F000000, 8: 0x3EB504F3, 16: 0x3E800000}
    for z, bits in want.items():
        assert int(oracle.scale_f32(z).view(np.uint32)) == bits


def test_error_decomposition_and_proposition1():
    # Eq. (7): E = P + Delta_c + Delta_a, and Prop. 1:
    #   E Delta_c = 0,  E||Delta_c||_F^2 = sum e^2 (seed independent since RN is odd),  <= V of Eq. (9)
    m, n, d, zeta = 2048, 8, 32, 4
    A = wl.gaussian(m, n, 31)
    sc = np.float32(0.5)
    q = (sc * np.abs(A)).astype(np.float32)
    with np.errstate(under="ignore"):
        e = q.astype(np.float16).astype(np.float64) - q.astype(np.float64)   # numpy's RN16, not the oracle's
    sum_e2 = zeta * float((e ** 2).sum())
    qd = q.astype(np.float64)
    V = U * U * zeta * float((qd[qd >= 2.0 ** -14] ** 2).sum()) + H * H / 4 * zeta * int(((qd > 0) & (qd < 2.0 ** -14)).sum())
    assert sum_e2 <= V
    norms, means = [], []
    T = 300
    for t in range(T):
        seed = sketch_seed(500 + t)
        Bq = oracle.f64_sketch(seed, d, zeta, A, mode=oracle.BQ)
        Bc = oracle.f64_sketch(seed, d, zeta, A, mode=oracle.BC)
        if t == 0:
            # P = B_q - B vanishes at zeta=4: multiplication by 1/2 is exact
            assert np.allclose(Bq, oracle.f64_sketch(seed, d, zeta, A), rtol=0, atol=1e-12)
        dc = Bc - Bq
        norms.append(float((dc ** 2).sum()))
        means.append(float(dc.mean()))
    norms = np.array(norms)
    z = (norms.mean() - sum_e2) / (norms.std(ddof=1) / math.sqrt(T))
    assert abs(z) < 4, (norms.mean(), sum_e2, z)
    # mean of Delta_c entries indistinguishable from 0 (BASELINE north_star)
    mm = np.array(means)
    assert abs(mm.mean()) / (mm.std(ddof=1) / math.sqrt(T)) < 4


def test_bq_differs_from_ideal_only_by_scale_rounding_at_zeta2():
    # zeta=2: s = fp32(1/sqrt2) is inexact, so P != 0 but tiny (reading R7: <= ~1e-7 relative)
    A = wl.gaussian(1024, 8, 32)
    seed = sketch_seed(40)
    B = oracle.f64_sketch(seed, 32, 2, A)
    Bq = oracle.f64_sketch(seed, 32, 2, A, mode=oracle.BQ)
    r = ev.rel_fro(Bq, B)
    assert 0 < r < 2e-7


def test_seq16_error_is_conversion_plus_accumulation():
    # D - B_c = Delta_a; with one contribution per bucket entry (m tiny, d huge, zeta=1) there is
    # nothing to accumulate: D == RN16 of the single product (0 + v = v) -> SEQ16 == B_c exactly
    A = wl.gaussian(16, 6, 33)
    seed = sketch_seed(41)
    b, _ = oracle.hashes(seed, 4096, 1, 16)
    assert len(set(b[:, 0].tolist())) == 16
    D = oracle.seq16_sketch(seed, 4096, 1, A)
    Bc = oracle.f64_sketch(seed, 4096, 1, A, mode=oracle.BC)
    assert np.array_equal(oracle.half_bits_to_f64(D), Bc)


def test_seq16_sr_uses_the_documented_bit_layout():
    # reading R14: R = splitmix64(sr_seed ^ ((i*zeta+j)*ceil(n/2) + pair)); bits 63..40 -> even column,
    # bits 39..16 -> odd column.  Singleton buckets make D == SR16(p, bits) directly.
    m, n, d, zeta = 12, 5, 8192, 2
    A = wl.gaussian(m, n, 34)
    seed, sr_seed = sketch_seed(42), sketch_seed(43)
    b, s = oracle.hashes(seed, d, zeta, m)
    assert len(set(b.ravel().tolist())) == m * zeta
    D = oracle.seq16_sketch(seed, d, zeta, A, rounding=oracle.SR, sr_seed=sr_seed)
    sc = oracle.scale_f32(zeta)
    npairs = (n + 1) // 2
    for i in range(m):
        for j in range(zeta):
            es = np.float32(-sc if s[i, j] else sc)
            for c in range(n):
                R = oracle.splitmix64(sr_seed ^ ((i * zeta + j) * npairs + c // 2))
                r24 = (R >> 16) & 0xFFFFFF if c & 1 else R >> 40
                want = oracle.sr16([np.float32(es * A[i, c])], [r24])[0]
                assert D[b[i, j], c] == want
    # and SR sketches are unbiased around B_q on average over sr seeds (loose statistical check)
    Bq = oracle.f64_sketch(seed, d, zeta, A, mode=oracle.BQ)
    acc = np.zeros_like(Bq)
    T = 200
    for t in range(T):
        acc += oracle.half_bits_to_f64(oracle.seq16_sketch(seed, d, zeta, A, rounding=oracle.SR, sr_seed=sketch_seed(900 + t)))
    nzmask = Bq != 0
    rel = np.abs(acc / T - Bq)[nzmask] / np.abs(Bq[nzmask])
    assert np.median(rel) < 2e-4 and rel.max() < 2e-3   # RN alone would sit at ~2.4e-4 median, fixed sign


def test_range_counts_match_numpy():
    A = np.concatenate([wl.gaussian(300, 8, 35, pow2=k) for k in (-24, -16, 0, 12, 17)])
    zeta = 4
    c = oracle.range_counts(zeta, A)
    p = np.abs(0.5 * A.astype(np.float64))
    with np.errstate(over="ignore", under="ignore"):
        h = (np.float32(0.5) * A).astype(np.float16)
    assert c["n_contrib"] == A.size * zeta
    assert c["n_sub"] == zeta * int(((p > 0) & (p < 2.0 ** -14)).sum())
    assert c["n_zero"] == zeta * int(((p > 0) & (h == 0)).sum())
    assert c["n_convinf"] == zeta * int(np.isinf(h).sum())
    assert c["n_zero"] > 0 and c["n_convinf"] > 0 and c["n_sub"] > c["n_zero"]


def test_proposition2_distortion_perturbation():
    # Prop. 2 Eq. (10): |eta(X)-eta(Y)| <= ||X-Y||_2 <= ||X-Y||_F,
    # on (F64 sketch, SEQ16 sketch) pairs mapped through R^-1
    m, n, d, zeta = 8192, 16, 64, 4
    A = wl.gaussian(m, n, 36)
    R = ev.gram_R([A[:3000], A[3000:]], n)
    assert np.allclose(np.abs(R), np.abs(np.linalg.qr(A.astype(np.float64), mode="r")), atol=1e-9)
    for t in range(5):
        seed = sketch_seed(60 + t)
        X = ev.distortion_operator(oracle.f64_sketch(seed, d, zeta, A), R)
        Y = ev.distortion_operator(oracle.half_bits_to_f64(oracle.seq16_sketch(seed, d, zeta, A)), R)
        lhs = abs(ev.eta_of(X) - ev.eta_of(Y))
        assert lhs <= np.linalg.norm(X - Y, 2) * (1 + 1e-12) <= np.linalg.norm(X - Y, "fro") * (1 + 1e-12)
        assert 0.05 < ev.eta_of(X) < 1.5     # d=4n sketch of a Gaussian subspace: eta ~ sqrt(n/d)
        assert ev.distortion(oracle.f64_sketch(seed, d, zeta, A), R) == ev.eta_of(X)


def test_sequential_fp16_error_grows_like_sqrt_depth():
    # SURVEY 8c "predicted conflicts": relF(SEQ16) ~ 1.44e-4 sqrt(L); checks the oracle reproduces
    # the order of magnitude at L = 512 and 4096 (the paper's operating depth)
    for m, want in ((4096, 3.4e-3), (32768, 9.9e-3)):
        A = wl.gaussian(m, 16, 37)
        seed = sketch_seed(70)
        B = oracle.f64_sketch(seed, 32, 4, A)
        D = oracle.half_bits_to_f64(oracle.seq16_sketch(seed, 32, 4, A))
        r = ev.rel_fro(D, B)
        assert want / 2 < r < want * 2, (m, r)
