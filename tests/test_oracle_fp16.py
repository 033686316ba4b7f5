"""Pins for the oracle's binary16 routines (conversion a4, accumulation step of a5, SR)."""
import os

import numpy as np
import pytest

import oracle

NCPU = min(8, os.cpu_count() or 1)
U = 2.0 ** -11   # unit roundoff
H = 2.0 ** -24   # subnormal spacing


def bits16(x):
    return np.asarray(x, dtype=np.float16).view(np.uint16)


def test_rn16_exhaustive_vs_f16c_hardware():
    if not oracle.has_f16c_crosscheck():
        pytest.skip("host CPU has no F16C")
    bad, first = oracle.rn16_vs_f16c(0, 1 << 32, 1, NCPU)  # every FP32 bit pattern
    assert bad == 0, hex(first)


def test_rn16_vs_numpy_float16():
    rng = np.random.default_rng(0)
    x = rng.integers(0, 1 << 32, size=2_000_000, dtype=np.uint64).astype(np.uint32).view(np.float32)
    x = x[~np.isnan(x)]
    with np.errstate(over="ignore"):
        want = x.astype(np.float16).view(np.uint16)
    assert np.array_equal(oracle.rn16(x), want)
    # dense sweep through the subnormal / tie region
    y = np.ldexp(np.arange(0, 1 << 16, dtype=np.float32), -29)  # multiples of 2^-29 up to 2^-13
    assert np.array_equal(oracle.rn16(y), y.astype(np.float16).view(np.uint16))


def test_rn16_is_odd():
    # PAPER.md:239 "RN is odd: Q(-q) = -Q(q)"
    rng = np.random.default_rng(1)
    x = (rng.standard_normal(100000) * np.exp2(rng.integers(-30, 18, 100000))).astype(np.float32)
    assert np.array_equal(oracle.rn16(-x), oracle.rn16(x) ^ 0x8000)


def test_rn16_edge_cases():
    f = np.float32
    # Cor. 3 / PAPER.md:293, :394: below h/2 -> 0; exactly h/2 = 2^-25 -> 0 (nearest even)
    assert oracle.rn16([f(2.0 ** -25)])[0] == 0x0000
    assert oracle.rn16([f(2.0 ** -25 * 0.999)])[0] == 0x0000
    assert oracle.rn16([np.nextafter(f(2.0 ** -25), f(1))])[0] == 0x0001
    assert oracle.rn16([f(3 * 2.0 ** -25)])[0] == 0x0002     # 1.5h -> 2h (even)
    assert oracle.rn16([f(5 * 2.0 ** -25)])[0] == 0x0002     # 2.5h -> 2h (even)
    assert oracle.rn16([f(2.0 ** -24)])[0] == 0x0001
    assert oracle.rn16([f(2.0 ** -14)])[0] == 0x0400         # smallest normal
    assert oracle.rn16([f(65504.0)])[0] == 0x7BFF
    assert oracle.rn16([f(65519.99)])[0] == 0x7BFF
    assert oracle.rn16([f(65520.0)])[0] == 0x7C00            # RN overflow -> inf (reading R9)
    assert oracle.rn16([f(-65520.0)])[0] == 0xFC00
    assert oracle.rn16([f(32768.0)])[0] == 0x7800            # PAPER.md:394 "still finite ... 32768"
    assert oracle.rn16([f(1.0 + 2.0 ** -11)])[0] == 0x3C00   # tie -> even
    assert oracle.rn16([f(1.0 + 3 * 2.0 ** -11)])[0] == 0x3C02
    assert oracle.rn16([f(np.inf)])[0] == 0x7C00
    assert oracle.rn16([f(-0.0)])[0] == 0x8000


def test_add16_paper_worked_example():
    # "at z=1, adding +2^-11 rounds back to one, whereas adding -2^-11 is exact"
    one = 0x3C00
    plus = bits16(2.0 ** -11)
    minus = bits16(-(2.0 ** -11))
    assert oracle.add16([one], [plus])[0] == one
    r = oracle.add16([one], [minus])[0]
    assert oracle.half_bits_to_f64([r])[0] == 1.0 - 2.0 ** -11


def test_add16_exhaustive_vs_f16c_hardware():
    if not oracle.has_f16c_crosscheck():
        pytest.skip("host CPU has no F16C")
    bad, first = oracle.add16_vs_f16c(0, 3, NCPU)  # z: all 2^16; v: every third pattern
    assert bad == 0, hex(first)


def test_add16_vs_numpy_float16():
    rng = np.random.default_rng(2)
    z = rng.integers(0, 1 << 16, 3_000_000).astype(np.uint16)
    v = rng.integers(0, 1 << 16, 3_000_000).astype(np.uint16)
    with np.errstate(over="ignore", invalid="ignore"):
        want = (z.view(np.float16) + v.view(np.float16)).view(np.uint16)
    got = oracle.add16(z, v)
    nan = np.isnan(want.view(np.float16))
    assert np.array_equal(got[~nan], want[~nan])
    assert np.all(np.isnan(got[nan].view(np.float16)))


def test_add16_special_values():
    inf, ninf = 0x7C00, 0xFC00
    assert oracle.add16([0x7BFF], [0x7BFF])[0] == inf               # running-sum overflow (reading R9)
    assert np.isnan(oracle.add16([inf], [ninf]).view(np.float16)[0])
    assert oracle.add16([0x0000], [0x8000])[0] == 0x0000            # (+0)+(-0)=+0 (reading R10)
    assert oracle.add16([0x3C00], [0xBC00])[0] == 0x0000            # x+(-x)=+0
    assert oracle.add16([0x0001], [0x0001])[0] == 0x0002            # subnormals kept (.noftz)
    assert oracle.add16([0x0000], [0x1234])[0] == 0x1234            # 0+v = v


def test_serial_accumulation_bound():
    # |z_L - sum v| <= L u/(1-L u) sum|v| for L u < 1
    rng = np.random.default_rng(3)
    for L in (16, 256, 1500):
        v = (rng.standard_normal((200, L)) * 0.5).astype(np.float16)
        z = np.zeros(200, dtype=np.uint16)
        for k in range(L):
            z = oracle.add16(z, v[:, k].view(np.uint16))
        exact = v.astype(np.float64).sum(axis=1)
        bound = L * U / (1 - L * U) * np.abs(v.astype(np.float64)).sum(axis=1)
        assert np.all(np.abs(oracle.half_bits_to_f64(z) - exact) <= bound)


# ------------------------------------------------------------------ stochastic conversion
def _sr_all_draws(p):
    r = np.arange(1 << 24, dtype=np.uint32)
    return oracle.sr16(np.full(r.shape, p, dtype=np.float32), r)


@pytest.mark.parametrize("p", [0.3, -1.7, 1000.123, 6.1e-5 * 0.37, 2.0 ** -20 * 1.3, -(2.0 ** -26) * 1.1])
def test_sr16_unbiased_over_all_draws(p):
    # "rounded to one of its neighboring FP16 values l<=q<=v, selecting v with
    # probability (q-l)/(v-l)"; the ideal rule has expectation q.  24-bit draws, centred (R13).
    p = float(np.float32(p))
    out = oracle.half_bits_to_f64(_sr_all_draws(p))
    vals = np.unique(out)
    assert len(vals) == 2
    lo, hi = (vals[0], vals[1]) if abs(vals[0]) < abs(vals[1]) else (vals[1], vals[0])
    assert abs(lo) < abs(p) < abs(hi)                       # the two neighbours bracket p
    w = abs(hi) - abs(lo)
    assert abs(out.mean() - p) <= 2.0 ** -25 * w + 1e-18    # probability quantised to 2^-24


def test_sr16_representable_unchanged_and_symmetric():
    rng = np.random.default_rng(4)
    h = rng.integers(0, 0x7C00, 5000).astype(np.uint16)
    x = h.view(np.float16).astype(np.float32)
    r = rng.integers(0, 1 << 24, 5000).astype(np.uint32)
    assert np.array_equal(oracle.sr16(x, r), h)             # "returned unchanged when q is representable"
    y = (rng.standard_normal(5000) * np.exp2(rng.integers(-28, 15, 5000))).astype(np.float32)
    assert np.array_equal(oracle.sr16(-y, r), oracle.sr16(y, r) ^ 0x8000)


def test_sr16_normal_range_matches_add_random_bits_then_truncate():
    # in the FP16 normal range t = frac13/2^13, so "u<t" == "carry out of frac13 + (~R13 & 0x1FFF)":
    # the textbook SR-by-truncation construction, retyped with integers.
    rng = np.random.default_rng(5)
    x = (rng.uniform(1, 2, 200000) * np.exp2(rng.integers(-14, 15, 200000))).astype(np.float32)
    x *= rng.choice([-1, 1], x.shape).astype(np.float32)
    r = rng.integers(0, 1 << 24, x.shape).astype(np.uint32)
    fb = x.view(np.uint32)
    mag = fb & 0x7FFFFFFF
    add = (~(r >> 11)) & 0x1FFF
    t = (mag + add) >> 13                                   # truncate 13 bits after adding
    e = (t >> 10).astype(np.int64) - 127 + 15
    h = ((e << 10) | (t & 0x3FF)).astype(np.uint16)
    h = np.where(e >= 31, 0x7C00, h).astype(np.uint16) | ((fb >> 16) & 0x8000).astype(np.uint16)
    assert np.array_equal(oracle.sr16(x, r), h)


@pytest.mark.parametrize("q", [2.0 ** -26, 0.3 * 2.0 ** -24, 0.9 * 2.0 ** -24])
def test_sr16_corollary3_variance(q):
    # Cor. 3 Eq. (12), k=0: for 0<|q|<h, E e = 0, E e^2 = h|q| - q^2
    q = float(np.float32(q))
    e = oracle.half_bits_to_f64(_sr_all_draws(q)) - q
    assert abs(e.mean()) <= 2.0 ** -25 * H
    assert abs((e ** 2).mean() - (H * q - q * q)) <= 2e-7 * H * q
    # RN in the same regime: below h/2 the contribution is erased, e = -q
    if q < H / 2:
        assert oracle.rn16([np.float32(q)])[0] == 0


def test_sr16_overflow_edge():
    f = np.float32
    assert oracle.sr16([f(65504.0)], [123])[0] == 0x7BFF
    assert oracle.sr16([f(70000.0)], [5])[0] == 0x7C00
    out = _sr_all_draws(65520.0)                            # halfway between 65504 and "65536"
    assert set(np.unique(out)) == {0x7BFF, 0x7C00}          # |l|=65504 -> v=inf allowed (R13)
    assert abs((out == 0x7C00).mean() - 0.5) < 1e-6
