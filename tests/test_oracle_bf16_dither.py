"""Pins for the oracle's NEXT-4 modes: the bfloat16 control and the
dither conversion of Eq. (6).  Committed before any kernel that implements them."""
import os

import numpy as np
import pytest

import oracle

NCPU = min(8, os.cpu_count() or 1)
UB = 2.0 ** -8     # bfloat16 unit roundoff
HB = 2.0 ** -133   # bfloat16 subnormal spacing
H = 2.0 ** -24     # binary16 subnormal spacing
M64 = (1 << 64) - 1
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ bfloat16 conversion
def test_bf16_rn_exhaustive_vs_integer_rule():
    bad, first = oracle.bf16_vs_bits(0, 1 << 32, 1, NCPU)   # every FP32 bit pattern
    assert bad == 0, hex(first)


def test_bf16_rn_vs_torch_bfloat16():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(0)
    x = rng.integers(0, 1 << 32, size=2_000_000, dtype=np.uint64).astype(np.uint32).view(np.float32)
    x = x[~np.isnan(x)]
    want = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(oracle.bf16_rn(x), want)
    y = np.ldexp(np.arange(0, 1 << 16, dtype=np.float32), -140)   # subnormal / tie region: multiples of 2^-140
    want = torch.from_numpy(y).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(oracle.bf16_rn(y), want)


def test_bf16_rn_is_odd_and_widening_is_exact():
    rng = np.random.default_rng(1)
    x = (rng.standard_normal(100000) * np.exp2(rng.integers(-120, 120, 100000))).astype(np.float32)
    assert np.array_equal(oracle.bf16_rn(-x), oracle.bf16_rn(x) ^ 0x8000)
    b = np.arange(1 << 16, dtype=np.uint16)
    fin = ((b >> 7) & 0xFF) != 0xFF
    wide = (b.astype(np.uint32) << 16).view(np.float32).astype(np.float64)   # a bfloat16 is the upper half of an FP32
    assert np.array_equal(oracle.bf16_bits_to_f64(b[fin]), wide[fin])
    assert np.array_equal(oracle.bf16_rn(wide[fin].astype(np.float32)), b[fin])   # round trip


def test_bf16_rn_edge_cases():
    f = np.float32
    assert oracle.bf16_rn([f(1.0)])[0] == 0x3F80
    assert oracle.bf16_rn([f(1.0 + 2.0 ** -8)])[0] == 0x3F80          # tie -> even
    assert oracle.bf16_rn([f(1.0 + 3 * 2.0 ** -8)])[0] == 0x3F82      # tie -> even (up)
    assert oracle.bf16_rn([np.nextafter(f(1.0 + 2.0 ** -8), f(2))])[0] == 0x3F81
    assert oracle.bf16_rn([f(65520.0)])[0] == 0x4780                  # finite where binary16 overflows
    assert oracle.bf16_rn([f(2.0 ** 20 * 1e3)])[0] & 0x7F80 != 0x7F80
    mx = np.uint32(0x7F7F0000).view(np.float32)                      # largest finite bfloat16
    assert oracle.bf16_rn([mx])[0] == 0x7F7F
    assert oracle.bf16_rn([np.finfo(np.float32).max])[0] == 0x7F80    # rounds up to inf
    assert oracle.bf16_rn([f(-np.inf)])[0] == 0xFF80
    assert oracle.bf16_rn([f(2.0 ** -133)])[0] == 0x0001              # subnormals kept
    assert oracle.bf16_rn([f(2.0 ** -134)])[0] == 0x0000              # half the spacing: tie -> even = 0
    assert oracle.bf16_rn([f(3 * 2.0 ** -134)])[0] == 0x0002          # 1.5 spacings -> 2 (even)
    assert oracle.bf16_rn([f(2.0 ** -126)])[0] == 0x0080              # smallest normal
    assert oracle.bf16_rn([f(2.0 ** -40)])[0] != 0                    # k = -40 of PAPER.md:394 is representable
    assert oracle.bf16_rn([f(-0.0)])[0] == 0x8000


# ------------------------------------------------------------------ bfloat16 accumulation step
def bfbits(x):
    return oracle.bf16_rn(np.asarray(x, dtype=np.float32))


def test_bf16_add_worked_example_at_u_2_pow_minus_8():
    # PAPER.md:257's example restated for u = 2^-8: at z = 1, adding +2^-8 rounds back to one (tie to even),
    # adding -2^-8 is exact (the spacing below one is 2^-8)
    one = 0x3F80
    assert oracle.bf16_add([one], bfbits([2.0 ** -8]))[0] == one
    r = oracle.bf16_add([one], bfbits([-(2.0 ** -8)]))[0]
    assert oracle.bf16_bits_to_f64([r])[0] == 1.0 - 2.0 ** -8


def test_bf16_add_vs_float_add_then_round():
    bad, first = oracle.bf16_add_vs_float(0, 7, NCPU)       # z: all 2^16; v: every seventh pattern
    assert bad == 0, hex(first)


def test_bf16_add_vs_torch_bfloat16():
    torch = pytest.importorskip("torch")
    rng = np.random.default_rng(2)
    z = rng.integers(0, 1 << 16, 2_000_000).astype(np.uint16)
    v = rng.integers(0, 1 << 16, 2_000_000).astype(np.uint16)
    tz = torch.from_numpy(z.view(np.int16)).view(torch.bfloat16)
    tv = torch.from_numpy(v.view(np.int16)).view(torch.bfloat16)
    want = (tz + tv).view(torch.int16).numpy().view(np.uint16)
    got = oracle.bf16_add(z, v)
    nan = np.isnan(oracle.bf16_bits_to_f64(want))
    assert np.array_equal(got[~nan], want[~nan])
    assert np.all(np.isnan(oracle.bf16_bits_to_f64(got[nan])))


def test_bf16_add_special_values():
    inf, ninf = 0x7F80, 0xFF80
    assert oracle.bf16_add([0x7F7F], [0x7F7F])[0] == inf
    assert np.isnan(oracle.bf16_bits_to_f64(oracle.bf16_add([inf], [ninf]))[0])
    assert oracle.bf16_add([0x0000], [0x8000])[0] == 0x0000
    assert oracle.bf16_add([0x3F80], [0xBF80])[0] == 0x0000
    assert oracle.bf16_add([0x0001], [0x0001])[0] == 0x0002           # subnormals kept
    assert oracle.bf16_add([0x0000], [0x1234])[0] == 0x1234
    # exponents more than 44 apart (the double sum is inexact): the result is the larger operand
    assert oracle.bf16_add([0x7F00], [0x0001])[0] == 0x7F00
    assert oracle.bf16_add([0x7F00], [0x8001])[0] == 0x7F00


def test_bf16_serial_accumulation_bound():
    # PAPER.md:259-263 with u = 2^-8: |z_L - sum v| <= L u/(1 - L u) sum|v| for L u < 1
    rng = np.random.default_rng(3)
    for L in (16, 100, 200):
        v = bfbits(rng.standard_normal((200, L)) * 0.5)
        z = np.zeros(200, dtype=np.uint16)
        for k in range(L):
            z = oracle.bf16_add(z, v[:, k])
        vv = oracle.bf16_bits_to_f64(v)
        exact = vv.sum(axis=1)
        bound = L * UB / (1 - L * UB) * np.abs(vv).sum(axis=1)
        err = np.abs(oracle.bf16_bits_to_f64(z) - exact)
        assert np.all(err <= bound)
        assert err.max() > 0.001 * bound.max()       # and it really is an 8-bit accumulation


def test_seqbf16_integer_valued_input_equals_f64_in_any_order():
    # entries in {-3..3}, zeta in {1, 4} (scale 1 or 1/2 exact): every partial sum is a multiple of 1/2
    # below 128, hence exact with an 8-bit significand in any order -> SEQ-BF16 == F64 bit for bit
    import workloads as wl

    for zeta, d, m in ((4, 64, 700), (1, 64, 900)):
        A = wl.integer_valued(m, 12, 5 + zeta)
        seed = wl.sketch_seed(11)
        want = oracle.f64_sketch(seed, d, zeta, A)
        assert np.abs(want).max() < 128
        got = oracle.seqbf16_sketch(seed, d, zeta, A)
        assert np.array_equal(oracle.bf16_bits_to_f64(got), want)
        # row ranges stream: two halves accumulated into one D give the same bits
        # (same ascending order) -- through the row_begin argument
    A = wl.gaussian(500, 6, 9)
    seed = wl.sketch_seed(12)
    B = oracle.f64_sketch(seed, 32, 4, A)
    D = oracle.bf16_bits_to_f64(oracle.seqbf16_sketch(seed, 32, 4, A))
    rel = np.linalg.norm(D - B) / np.linalg.norm(B)
    assert 1e-4 < rel < 3e-2                          # bf16-sized error (u = 3.9e-3), not binary16-sized (4.9e-4)
    D16 = oracle.half_bits_to_f64(oracle.seq16_sketch(seed, 32, 4, A))
    assert np.linalg.norm(D16 - B) < 0.5 * np.linalg.norm(D - B)


# ------------------------------------------------------------------ dither (Eq. 6)
def test_xorshift64_published_vector():
    for ln in open(os.path.join(GOLDEN, "xorshift64_vector.txt")):
        if ln.startswith("#") or not ln.strip():
            continue
        a, b = (int(t) for t in ln.split())
        assert oracle.xorshift64(a) == b


def test_dither_coefficient_is_the_papers_literal():
    c = oracle.dither_c()
    assert c == np.float32(0.00097656)                 # PAPER.md:201 "written as 0.00097656f"
    assert c < np.float32(2.0 ** -10) and abs(float(c) / 2.0 ** -10 - 1) < 1e-5   # "approximately 2^-10"


def _rand_p(rng, k, lo=-20, hi=15):
    return (rng.standard_normal(k) * np.exp2(rng.integers(lo, hi, k))).astype(np.float32)


def test_dither_reduces_to_rn_when_the_perturbation_vanishes():
    rng = np.random.default_rng(4)
    p = _rand_p(rng, 200000, -30, 17)
    r = rng.integers(0, 1 << 24, p.shape).astype(np.uint32)
    assert np.array_equal(oracle.dither16(p, r, c=0.0), oracle.rn16(p))               # c = 0
    mid = np.full(p.shape, 1 << 23, dtype=np.uint32)
    assert np.array_equal(oracle.dither16(p, mid), oracle.rn16(p))                    # u0 = 1/2
    assert np.array_equal(oracle.dither16(p, mid, c=0.3), oracle.rn16(p))


def test_dither_is_odd_monotone_and_stays_within_one_relative_half_width():
    rng = np.random.default_rng(5)
    p = _rand_p(rng, 100000)
    r = rng.integers(0, 1 << 24, p.shape).astype(np.uint32)
    q = oracle.dither16(p, r)
    assert np.array_equal(oracle.dither16(-p, r), q ^ 0x8000)                         # relative perturbation: odd in q
    # monotone in u0 for q > 0: a larger draw never gives a smaller result
    pp = np.abs(p[:20000]) + np.float32(1e-30)
    r2 = np.minimum(r[:20000] + rng.integers(0, 1 << 20, 20000).astype(np.uint32), (1 << 24) - 1).astype(np.uint32)
    a, b = oracle.half_bits_to_f64(oracle.dither16(pp, r[:20000])), oracle.half_bits_to_f64(oracle.dither16(pp, r2))
    assert np.all(b >= a)
    # |perturbation| <= c/2 |q|: the result lies between RN16 of the two extreme perturbed values (RN16 is monotone)
    c = float(oracle.dither_c())
    p64 = p.astype(np.float64)
    lo = oracle.half_bits_to_f64(oracle.rn16((p64 - np.abs(p64) * c * 0.5000001).astype(np.float32)))
    hi = oracle.half_bits_to_f64(oracle.rn16((p64 + np.abs(p64) * c * 0.5000001).astype(np.float32)))
    v = oracle.half_bits_to_f64(q)
    assert np.all((v >= lo) & (v <= hi))
    # sign of the perturbation: u0 = 0 moves a positive q down, u0 -> 1 moves it up (1.5 (1 -+ c/2) = 1.5 -+ 0.75 spacings)
    s = 2.0 ** -10
    assert oracle.half_bits_to_f64(oracle.dither16([np.float32(1.5)], [0]))[0] == 1.5 - s
    assert oracle.half_bits_to_f64(oracle.dither16([np.float32(1.5)], [(1 << 24) - 1]))[0] == 1.5 + s
    assert oracle.half_bits_to_f64(oracle.dither16([np.float32(-1.5)], [0]))[0] == -(1.5 - s)


@pytest.mark.parametrize("q", [1.0 + 0.3 * 2.0 ** -10, 1.5 + 0.3 * 2.0 ** -10, 1.999, 1000.123, 6.1e-5 * 1.37, 0.3 * 2.0 ** -14])
def test_dither_jump_probabilities_closed_form(q):
    # q' = q (1 + (u0 - 1/2) c) with u0 uniform on the 2^24-point grid: P(Q <= g) for a binary16 grid point g is
    # P(q' < g + spacing/2) = clamp(((g + s/2)/q - 1)/c + 1/2, 0, 1).  The FP32 roundings of Eq. (6) move q' by a few
    # 2^-24 q, i.e. the probability by <= ~2^-22/c ~ 2.5e-4.
    q = float(np.float32(q))
    c = float(oracle.dither_c())
    r = np.arange(1 << 24, dtype=np.uint32)
    out = oracle.half_bits_to_f64(oracle.dither16(np.full(r.shape, q, dtype=np.float32), r))
    vals, counts = np.unique(out, return_counts=True)
    assert 1 <= len(vals) <= 3
    cdf = np.cumsum(counts) / float(1 << 24)
    for g, got in zip(vals, cdf):
        nxt = oracle.half_bits_to_f64(oracle.rn16([np.float32(g)]) + np.uint16(1))[0]   # next grid point above g > 0
        want = min(1.0, max(0.0, ((g + (nxt - g) / 2) / q - 1.0) / c + 0.5))
        assert abs(got - want) < 6e-4, (g, got, want)
    # the width c q lies between one spacing (bottom of a binade) and two (top): "not uniformly one FP16 spacing"
    # (PAPER.md:205); in the subnormal range it is far below the spacing and dither is RN
    if q < 2.0 ** -14:
        assert len(vals) == 1 and vals[0] == oracle.half_bits_to_f64(oracle.rn16([np.float32(q)]))[0]


def test_dither_loses_tiny_terms_like_rn_and_is_nearly_unbiased_only_where_the_width_is_one_spacing():
    r = np.arange(0, 1 << 24, 7, dtype=np.uint32)
    # PAPER.md:384 "Relative dither also loses sufficiently small terms because its perturbation shrinks with their magnitude"
    tiny = np.full(r.shape, 2.0 ** -26, dtype=np.float32)
    assert not oracle.dither16(tiny, r).any()
    # just above a power of two the width c q is one spacing (up to 1e-3): mean error ~ 0; the same offset at the top
    # of the binade (width two spacings) is also nearly unbiased, in between it is not an SR but the
    # mean stays within half a spacing of q
    s = 2.0 ** -10
    for q, tol in ((1.0 + 0.3 * s, 2e-3), (1.25 + 0.3 * s, 0.5), (1.4142135, 0.5)):
        q = float(np.float32(q))
        out = oracle.half_bits_to_f64(oracle.dither16(np.full(r.shape, q, dtype=np.float32), r))
        assert abs(out.mean() - q) <= tol * s, (q, out.mean())


def _py_splitmix64(x):
    z = (x + 0x9E3779B97F4A7C15) & M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M64
    return z ^ (z >> 31)


def _py_xorshift64(x):
    x ^= (x << 13) & M64
    x ^= x >> 7
    x ^= (x << 17) & M64
    return x


def test_seq16_dither_mode_counter_layout_through_singleton_buckets():
    # reading R21: bits = xorshift64(splitmix64(sr_seed ^ ((i zeta + j) ceil(n/2) + pair))), 63..40 -> even column,
    # 39..16 -> odd column.  Re-derived with Python integers; a sketch entry hit once equals Q_dith(p) (0 + v = v).
    import workloads as wl

    m, n, d, zeta = 24, 7, 4096, 2
    seed, sr_seed = wl.sketch_seed(21), wl.sketch_seed(22)
    rng = np.random.default_rng(6)
    A = _rand_p(rng, m * n, -6, 6).reshape(m, n)
    b, sgn = oracle.hashes(seed, d, zeta, m)
    cnt = np.bincount(b.ravel(), minlength=d)
    D = oracle.seq16_sketch(seed, d, zeta, A, rounding=oracle.DITHER, sr_seed=sr_seed)
    sc = oracle.scale_f32(zeta)
    npairs = (n + 1) // 2
    checked = 0
    for i in range(m):
        for j in range(zeta):
            if cnt[b[i, j]] != 1:
                continue
            es = np.float32(-sc if sgn[i, j] else sc)
            p = (es * A[i]).astype(np.float32)
            r24 = np.empty(n, dtype=np.uint32)
            for c in range(n):
                R = _py_xorshift64(_py_splitmix64(sr_seed ^ ((i * zeta + j) * npairs + c // 2)))
                r24[c] = ((R >> 16) & 0xFFFFFF) if c & 1 else (R >> 40)
            assert np.array_equal(D[b[i, j]], oracle.dither16(p, r24)), (i, j)
            checked += 1
    assert checked > m * zeta * 0.9
    # and it differs from RN on this input
    hit = cnt > 0
    assert (D[hit] != oracle.seq16_sketch(seed, d, zeta, A)[hit]).mean() > 0.2
