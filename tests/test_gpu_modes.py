"""GPU parity tests of the other accumulation formats and conversion controls and of the fused
right-hand side (NEXT-1), through the C ABI against the CPU oracle on the same seeded inputs:
  bfloat16 accumulate .... bit-exact on inputs whose sums are exact in bfloat16; relF <= 1.5 x the
                                                 oracle's sequential-bfloat16 relF otherwise
  dither conversion, Eq. (6)  bit-exact through singleton buckets (0 + v = v)
  SR inside the tensor-memory kernel ........... bit-exact through singleton buckets
  FP32 accumulate in tensor memory ............. bit-exact on integer inputs, relF <= 1e-5 vs the FP64 oracle
  [A | b] in one pass ........... Sb bit-exact on integer inputs, relF <= 1e-5 otherwise; SA unchanged
"""
import numpy as np
import pytest

import evaluation as ev
import oracle
import workloads as wl
from workloads import sketch_seed

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

VID = {"auto": 0, "flat_pair": 1, "flat_vec": 2, "smem": 3, "generic": 4, "tmem": 5, "small": 6}


@pytest.fixture(scope="module")
def ss():
    import paper_2606_20195_b200 as ss_

    assert torch.cuda.is_available()
    return ss_


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def bits(t):
    """16-bit tensor (binary16 or bfloat16) -> uint16 bit patterns with -0 canonicalised to +0 (R10)."""
    b = t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()
    b[b == 0x8000] = 0
    return b


def col(b):
    """A vector as an [m, 1] matrix with unit column stride (numpy leaves a length-1 axis's stride arbitrary)."""
    out = np.empty((b.shape[0], 1), dtype=np.float32)
    out[:, 0] = b
    return out


def plan_ok(ss, sk, n, variant, f16, rounding=0, rows=None):
    try:
        sk.plan(n, f16=f16, rounding=rounding, variant=VID[variant], rows=rows or sk.m)
        return True
    except ss.SketchError as e:
        assert e.code == -6, e
        return False


# ------------------------------------------------------------------------------------ bfloat16
BF16_VARIANTS = ["auto", "flat_pair", "flat_vec", "tmem", "generic"]
# (m, n, d, zeta): mean depth m zeta / d <= 64, entries in {-1, 0, 1} scaled by 1 or 1/2: every partial sum is a multiple of
# 1/2 below 128 in magnitude, i.e. exact in bfloat16 (8 significant bits) in any order
BF16_EXACT = [(2048, 16, 128, 4), (1500, 64, 128, 1), (8191, 128, 512, 4), (8191, 256, 1024, 4), (16001, 256, 2048, 4), (3001, 24, 256, 4),
              (8191, 1024, 1024, 4), (4001, 192, 384, 1)]


@pytest.mark.parametrize("variant", BF16_VARIANTS)
@pytest.mark.parametrize("m,n,d,zeta", BF16_EXACT)
def test_bf16_exact_sums_bit_exact(ss, variant, m, n, d, zeta):
    A = wl.integer_valued(m, n, 200 + m % 89, lo=-1, hi=1)
    seed = sketch_seed(m + 7 * zeta)
    want = oracle.f64_sketch(seed, d, zeta, A)
    b, _ = oracle.hashes(seed, d, zeta, m)
    assert np.bincount(b.ravel(), minlength=d).max() * (0.5 if zeta == 4 else 1.0) < 128
    sk = ss.Sketch(m, d, zeta, seed)
    if not plan_ok(ss, sk, n, variant, 2):
        with pytest.raises(ss.SketchError) as ei:
            sk.apply_bf16acc(dev(A), variant=VID[variant])
        assert ei.value.code == -6
        pytest.skip("plan: variant %s cannot run the bfloat16 path at m=%d n=%d d=%d zeta=%d" % (variant, m, n, d, zeta))
    got = sk.apply_bf16acc(dev(A), variant=VID[variant])
    assert got.dtype == torch.bfloat16
    assert np.array_equal(oracle.bf16_bits_to_f64(bits(got)), want)
    assert np.array_equal(bits(got), oracle.seqbf16_sketch(seed, d, zeta, A))


@pytest.mark.parametrize("m,n,d,zeta", [(4096, 16, 32, 4), (50021, 64, 128, 4), (70001, 128, 256, 4), (30011, 256, 512, 4), (20011, 256, 2048, 8)])
def test_bf16_error_vs_sequential_oracle(ss, m, n, d, zeta):
    # bfloat16 keeps the range and gives up three bits: relF is ~8x the FP16 figure at the same depth
    A = wl.gaussian(m, n, 11)
    seed = sketch_seed(300 + m % 13)
    B = oracle.f64_sketch(seed, d, zeta, A)
    ref = ev.rel_fro(oracle.bf16_bits_to_f64(oracle.seqbf16_sketch(seed, d, zeta, A)), B)
    sk = ss.Sketch(m, d, zeta, seed)
    ran = []
    for variant in BF16_VARIANTS:
        if not plan_ok(ss, sk, n, variant, 2):
            continue
        got = sk.apply_bf16acc(dev(A), variant=VID[variant])
        r = ev.rel_fro(oracle.bf16_bits_to_f64(bits(got)), B)
        ran.append(variant)
        assert r <= 1.5 * ref, (variant, r, ref)
        assert r > 1e-4            # it really is a bfloat16 accumulation (conversion alone costs ~2^-9 / sqrt(3))
    assert {"auto", "flat_vec", "generic"} <= set(ran), ran


def test_bf16_keeps_the_range_fp16_loses(ss):
    # at scale 2^16 the FP16 sketch overflows, at 2^-30 it underflows to zero; bfloat16 does neither
    m, n, d, zeta = 1 << 16, 128, 256, 4
    seed = sketch_seed(41)
    sk = ss.Sketch(m, d, zeta, seed)
    for k in (16, -30):
        A = wl.gaussian(m, n, 3, pow2=k)
        B = oracle.f64_sketch(seed, d, zeta, A)
        h = sk.apply_f16acc(dev(A)).float()
        bf = sk.apply_bf16acc(dev(A))
        if k > 0:
            assert int((~torch.isfinite(h)).sum()) > 0.5 * d * n
        else:
            assert int(torch.count_nonzero(h)) == 0
        assert bool(torch.isfinite(bf.float()).all())
        assert ev.rel_fro(oracle.bf16_bits_to_f64(bits(bf)), B) < 5e-2


# ------------------------------------------------------------------------------------ conversion rules through singleton buckets
SPECIALS = np.array([
    2.0 ** -25, np.nextafter(np.float32(2.0 ** -25), np.float32(1)), 3 * 2.0 ** -25, 5 * 2.0 ** -25, 2.0 ** -24, 2.0 ** -14,
    np.nextafter(np.float32(2.0 ** -14), np.float32(0)), 65504.0, 65519.996, 65520.0, 70000.0, 1e30, 32768.0,
    1.0 + 2.0 ** -11, 1.0 + 3 * 2.0 ** -11, 0.0, 1e-30, 1e-42, 6.1e-5, 0.33333334, 1000.123,
    1.0 + 2.0 ** -11 - 2.0 ** -21, 1.0 + 2.0 ** -11 + 2.0 ** -21, 2048.0 + 1.0 - 2.0 ** -10, 65504.0 + 15.99,
], dtype=np.float32)

# (variant, m, n, d): d = 65536 makes nearly every row a singleton for the flat kernels; the tensor-memory kernel holds at most
# 512 sketch rows per block with one bucket group (per-contribution conversion), so there m is small against d / zeta
SINGLETON_CASES = [("auto", 48, 64, 65536), ("flat_pair", 48, 64, 65536), ("flat_vec", 48, 64, 65536), ("generic", 48, 63, 65536),
                   ("tmem", 24, 64, 512), ("tmem", 24, 128, 256), ("tmem", 24, 256, 128), ("tmem", 40, 512, 512), ("tmem", 24, 192, 96)]


@pytest.mark.parametrize("rounding", ["sr", "dither"])
@pytest.mark.parametrize("zeta", [1, 4, 2])
@pytest.mark.parametrize("variant,m,n,d", SINGLETON_CASES)
def test_sr_and_dither_conversion_bit_exact_singleton_buckets(ss, variant, m, n, d, zeta, rounding):
    # DESIGN.md R13/R14 (SR) and R20/R21 (dither): the GPU's integer rules and counter layout against the oracle's
    rnd, ornd = (ss.SR, oracle.SR) if rounding == "sr" else (ss.DITHER, oracle.DITHER)
    if d % zeta:
        pytest.skip("d % zeta")
    seed, sr_seed = sketch_seed(88 + zeta), sketch_seed(99)
    sk = ss.Sketch(m, d, zeta, seed)
    b, _ = oracle.hashes(seed, d, zeta, m)
    cnt = np.bincount(b.ravel(), minlength=d)
    rng = np.random.default_rng(6)
    A = rng.standard_normal((m, n)).astype(np.float32) * np.exp2(rng.integers(-40, 17, (m, n))).astype(np.float32)
    A[:, :SPECIALS.size] = SPECIALS[None, :]
    if not plan_ok(ss, sk, n, variant, 1, rnd):
        pytest.skip("plan: variant %s cannot run rounding %s at n=%d d=%d zeta=%d" % (variant, rounding, n, d, zeta))
    got = bits(sk.apply_f16acc(dev(A), rounding=rnd, sr_seed=sr_seed, variant=VID[variant]))
    want_all = oracle.seq16_sketch(seed, d, zeta, A, rounding=ornd, sr_seed=sr_seed)
    want_all[want_all == 0x8000] = 0
    rows = sorted({int(b[i, j]) for i in range(m) for j in range(zeta) if cnt[b[i, j]] == 1})
    assert len(rows) > m * zeta * 0.3
    assert np.array_equal(got[rows], want_all[rows])
    # the rule differs from RN on this input (otherwise the test proves nothing)
    rn = bits(sk.apply_f16acc(dev(A), variant=VID[variant]))
    assert (rn[rows] != got[rows]).mean() > (0.1 if rounding == "sr" else 0.005)


@pytest.mark.parametrize("rounding", ["sr", "dither"])
@pytest.mark.parametrize("m,n,d,zeta", [(30011, 128, 256, 4), (20011, 64, 128, 2), (25013, 256, 512, 8), (9001, 512, 128, 1)])
def test_sr_and_dither_in_tensor_memory_match_the_flat_kernels_statistically(ss, m, n, d, zeta, rounding):
    # the same per-contribution values (bit-exact above), another order of addition: relF within 1.5x of the oracle's order
    rnd, ornd = (ss.SR, oracle.SR) if rounding == "sr" else (ss.DITHER, oracle.DITHER)
    A = wl.gaussian(m, n, 17)
    seed, sr_seed = sketch_seed(400 + zeta), sketch_seed(401)
    B = oracle.f64_sketch(seed, d, zeta, A)
    ref = ev.rel_fro(oracle.half_bits_to_f64(oracle.seq16_sketch(seed, d, zeta, A, rounding=ornd, sr_seed=sr_seed)), B)
    sk = ss.Sketch(m, d, zeta, seed)
    assert plan_ok(ss, sk, n, "tmem", 1, rnd)
    for variant in ("tmem", "flat_vec"):
        got = sk.apply_f16acc(dev(A), rounding=rnd, sr_seed=sr_seed, variant=VID[variant])
        r = ev.rel_fro(oracle.half_bits_to_f64(bits(got)), B)
        assert r <= 1.5 * ref and r <= 5e-2, (variant, r, ref)


# ------------------------------------------------------------------------------------ FP32 accumulate in tensor memory
F32_TMEM = [(10007, 64, 128, 4), (33333, 128, 256, 4), (9999, 128, 256, 1), (5001, 256, 64, 4), (6007, 256, 512, 4), (6007, 256, 1024, 4),
            (5003, 512, 512, 4), (7001, 128, 1024, 4), (3001, 512, 128, 1), (2501, 1024, 512, 4), (2503, 384, 768, 4), (2503, 96, 96, 1),
            (4001, 32, 512, 2), (4001, 160, 320, 8)]


@pytest.mark.parametrize("m,n,d,zeta", F32_TMEM)
def test_f32_tensor_memory_integer_input_bit_exact(ss, m, n, d, zeta):
    A = wl.integer_valued(m, n, 100 + m % 97)
    seed = sketch_seed(m + zeta)
    sk = ss.Sketch(m, d, zeta, seed)
    if not plan_ok(ss, sk, n, "tmem", 0):
        pytest.skip("plan: the FP32 partial of n=%d d=%d zeta=%d does not fit tensor memory" % (n, d, zeta))
    got = sk.apply_f32acc(dev(A), variant=VID["tmem"]).cpu().numpy().astype(np.float64)
    want = oracle.f64_sketch(seed, d, zeta, A)
    if zeta in (1, 4):
        assert np.array_equal(got, want)
    else:
        assert ev.rel_fro(got, want) <= 1e-6


@pytest.mark.parametrize("m,n,d,zeta", [(50021, 64, 128, 4), (70001, 128, 256, 4), (30011, 256, 512, 4), (40009, 128, 256, 8), (30011, 512, 256, 2)])
def test_f32_tensor_memory_within_1e5_of_f64_oracle(ss, m, n, d, zeta):
    A = wl.gaussian(m, n, 21)
    seed = sketch_seed(500 + zeta)
    sk = ss.Sketch(m, d, zeta, seed)
    assert plan_ok(ss, sk, n, "tmem", 0)
    B = oracle.f64_sketch(seed, d, zeta, A)
    got = sk.apply_f32acc(dev(A), variant=VID["tmem"]).cpu().numpy()
    r = ev.rel_fro(got, B)
    assert r <= 1e-5, r
    # row ranges + accumulate + padded leading dimension
    Ap = np.zeros((m, n + 12), dtype=np.float32)
    Ap[:, :n] = A
    Ad = dev(Ap)[:, :n]
    cut = (m // 3) // 8 * 8 + 5
    out = sk.apply_f32acc(Ad[:cut], variant=VID["tmem"], row_begin=0, rows=cut)
    sk.apply_f32acc(Ad[cut:], out=out, variant=VID["tmem"], row_begin=cut, rows=m - cut, accumulate=True)
    assert ev.rel_fro(out.cpu().numpy(), B) <= 1e-5


# ------------------------------------------------------------------------------------ [A | b] in one pass
RHS_SHAPES = [(10007, 64, 128, 4, "auto"), (10007, 64, 128, 4, "tmem"), (33333, 128, 256, 4, "tmem"), (6007, 256, 1024, 4, "tmem"),
              (4099, 256, 2048, 4, "tmem"), (2501, 1024, 2048, 4, "tmem"), (9999, 128, 256, 1, "tmem"), (7001, 128, 512, 8, "tmem"),
              (5000, 24, 16, 4, "auto"), (3000, 63, 64, 2, "auto"), (40000, 64, 128, 4, "flat_vec"), (9000, 64, 128, 4, "smem")]


@pytest.mark.parametrize("f16", [True, False])
@pytest.mark.parametrize("m,n,d,zeta,variant", RHS_SHAPES)
def test_fused_rhs_integer_inputs_bit_exact(ss, m, n, d, zeta, variant, f16):
    # b in FP32 with the same map.  Integer b, zeta in {1, 4}: every FP32 partial sum is exact in any order
    A = wl.integer_valued(m, n, 31 + m % 7)
    b = wl.integer_valued(m, 1, 77 + m % 5, lo=-50, hi=50)[:, 0].copy()
    seed = sketch_seed(600 + m % 11)
    sk = ss.Sketch(m, d, zeta, seed)
    if not plan_ok(ss, sk, n, variant, int(f16)):
        pytest.skip("plan: variant %s cannot run n=%d d=%d zeta=%d f16=%s" % (variant, n, d, zeta, f16))
    fn = sk.apply_f16acc_with_rhs if f16 else sk.apply_f32acc_with_rhs
    SA, Sb = fn(dev(A), dev(b), variant=VID[variant])
    want_b = oracle.f64_sketch(seed, d, zeta, col(b))[:, 0]
    want_A = oracle.f64_sketch(seed, d, zeta, A)
    if zeta in (1, 4):
        assert np.array_equal(Sb.cpu().numpy().astype(np.float64), want_b)
        got_A = oracle.half_bits_to_f64(bits(SA)) if f16 else SA.cpu().numpy().astype(np.float64)
        assert np.array_equal(got_A, want_A)
    else:
        assert ev.rel_fro(Sb.cpu().numpy(), want_b) <= 1e-6
        assert ev.rel_fro(SA.float().cpu().numpy(), want_A) <= (5e-3 if f16 else 1e-6)
    # the unfused pair of calls gives the same Sb
    Sb2 = sk.apply_f32acc(dev(col(b)))[:, 0]
    assert ev.rel_fro(Sb.cpu().numpy(), Sb2.cpu().numpy()) <= 1e-6


@pytest.mark.parametrize("m,n,d,zeta", [(70001, 128, 256, 4), (30011, 256, 1024, 4), (20011, 1024, 2048, 4)])
def test_fused_rhs_generic_inputs_ranges_and_accumulate(ss, m, n, d, zeta):
    A, b, _ = wl.ls_system(m, n, 3)
    seed = sketch_seed(700 + n)
    sk = ss.Sketch(m, d, zeta, seed)
    want_b = oracle.f64_sketch(seed, d, zeta, col(b))[:, 0]
    B = oracle.f64_sketch(seed, d, zeta, A)
    Ad, bd = dev(A), dev(b)
    SA, Sb = sk.apply_f16acc_with_rhs(Ad, bd)
    assert ev.rel_fro(Sb.cpu().numpy(), want_b) <= 1e-5
    assert ev.rel_fro(oracle.half_bits_to_f64(bits(SA)), B) <= 5e-2
    # widen is exact
    W = ss.sketch_widen(SA)
    assert np.array_equal(W.cpu().numpy().astype(np.float64), oracle.half_bits_to_f64(bits(SA))) or np.array_equal(
        np.nan_to_num(W.cpu().numpy().astype(np.float64)), np.nan_to_num(oracle.half_bits_to_f64(bits(SA))))
    # two row ranges, the second accumulated
    cut = (m // 2) // 16 * 16 + 3
    SA2, Sb2 = sk.apply_f16acc_with_rhs(Ad[:cut], bd[:cut], row_begin=0, rows=cut)
    sk.apply_f16acc_with_rhs(Ad[cut:], bd[cut:], out=SA2, Sb=Sb2, row_begin=cut, rows=m - cut, accumulate=True)
    assert ev.rel_fro(Sb2.cpu().numpy(), want_b) <= 1e-5
    assert ev.rel_fro(oracle.half_bits_to_f64(bits(SA2)), B) <= 5e-2
    # FP32 pipeline arm
    SA32, Sb32 = sk.apply_f32acc_with_rhs(Ad, bd)
    assert ev.rel_fro(Sb32.cpu().numpy(), want_b) <= 1e-5
    assert ev.rel_fro(SA32.cpu().numpy(), B) <= 1e-5


def test_widen_bf16_and_f16_exact(ss):
    allbits = torch.arange(0, 65536, dtype=torch.int32).to(torch.int16).cuda()
    for dt, conv in ((torch.float16, oracle.half_bits_to_f64), (torch.bfloat16, oracle.bf16_bits_to_f64)):
        x = allbits.view(dt)
        w = ss.sketch_widen(x).cpu().numpy().astype(np.float64)
        want = conv(allbits.cpu().numpy().view(np.uint16))
        ok = np.isfinite(want)
        assert np.array_equal(w[ok], want[ok])
        assert np.array_equal(np.isnan(w), np.isnan(want)) and np.array_equal(np.isinf(w), np.isinf(want))


# ------------------------------------------------------------------------------------ the conversion step alone; hardware cvt.rs
def _probe(ss, p, r, kind):
    return ss.sketch_convert_probe(p, r, kind).cpu().numpy().view(np.uint16)


def test_conversion_probe_matches_the_oracle_rules(ss):
    # a4 in isolation against the oracle's scalar rules on 2^20 seeded values spanning every FP16 regime
    g = torch.Generator(device="cuda").manual_seed(5)
    k = 1 << 20
    p = (torch.randn(k, generator=g, device="cuda") * torch.exp2(torch.randint(-45, 20, (k,), generator=g, device="cuda").float())).contiguous()
    r = torch.randint(0, 1 << 24, (k,), generator=g, device="cuda", dtype=torch.int32)
    pn, rn = p.cpu().numpy(), r.cpu().numpy().astype(np.uint32)
    assert np.array_equal(_probe(ss, p, None, 0), oracle.rn16(pn))
    assert np.array_equal(_probe(ss, p, r, 1), oracle.sr16(pn, rn))
    assert np.array_equal(_probe(ss, p, r, 6), oracle.sr16(pn, rn))      # the library's pair conversion (hardware fast path
    assert np.array_equal(_probe(ss, p, r, 7), oracle.sr16(pn, rn))      # on the normal grid): both halves
    assert np.array_equal(_probe(ss, p, r, 2), oracle.dither16(pn, rn))
    assert np.array_equal(_probe(ss, p, None, 3), oracle.bf16_rn(pn))


def test_hardware_cvt_rs_against_the_sr_rule(ss, capsys):
    """the hardware cvt.rs.f16x2.f32 may replace the integer rule R13 only if bit-identical.  2^30 samples:
    on the FP16 NORMAL grid (13 discarded bits) the instruction is rule R13 with r24's top 13 bits = the complement of 13
    bits of its 16-bit random field; below 2^-14 (more discarded bits than the field has) it is NOT -- counter-example
    printed -- so the library uses it exactly on that grid and keeps the integer rule elsewhere (R22); the hybrid is
    checked against the rule on every one of the 2^30 samples."""
    g = torch.Generator(device="cuda").manual_seed(9)
    chunk, chunks = 1 << 26, 16
    found, sub_mismatch, example = None, 0, None
    normal_total = sub_total = 0
    for c in range(chunks):
        bitsr = torch.randint(-(1 << 31), (1 << 31) - 1, (chunk,), generator=g, device="cuda", dtype=torch.int64).to(torch.int32)
        mant = torch.randint(0, 1 << 23, (chunk,), generator=g, device="cuda", dtype=torch.int32)
        # exponents: 2^-30 .. 2^16 (biased 97 .. 143), random sign
        ex = torch.randint(97, 144, (chunk,), generator=g, device="cuda", dtype=torch.int32)
        sg = torch.randint(0, 2, (chunk,), generator=g, device="cuda", dtype=torch.int32)
        p = ((sg << 31) | (ex << 23) | mant).view(torch.float32).contiguous()
        hw = {4: ss.sketch_convert_probe(p, bitsr, 4), 5: ss.sketch_convert_probe(p, bitsr, 5)}
        normal = (p.abs() >= 2.0 ** -14) & (p.abs() < 65504.0)
        sub = p.abs() < 2.0 ** -14
        cands = {}
        for half, shift in ((4, 0), (5, 16)):
            field = (bitsr >> shift) & 0xFFFF
            for name, rnd13 in (("top13", field >> 3), ("low13", field & 0x1FFF)):
                r24 = (((~rnd13) & 0x1FFF) << 11) | 0x7FF      # low 11 bits do not matter on the normal grid
                mine = ss.sketch_convert_probe(p, r24.to(torch.int32).contiguous(), 1)
                cands[(half, name)] = (int((mine != hw[half])[normal].sum()), int((mine != hw[half])[sub].sum()), mine)
        if found is None:
            ok = [k for k, v in cands.items() if v[0] == 0]
            assert ok, {k: v[:2] for k, v in cands.items()}
            found = ok
        for k in found:
            assert cands[k][0] == 0, (k, cands[k][:2])
        # the library's pair conversion (kinds 6 / 7: cvt.rs where both values are on the normal grid, rule R13 elsewhere) must
        # equal rule R13 (kind 1) on EVERY sample, whatever the regime
        r24 = (bitsr & 0xFFFFFF).contiguous()
        rule = ss.sketch_convert_probe(p, r24, 1)
        assert bool((ss.sketch_convert_probe(p, r24, 6) == rule).all()) and bool((ss.sketch_convert_probe(p, r24, 7) == rule).all())
        normal_total += int(normal.sum())
        sub_total += int(sub.sum())
        k0 = found[0]
        sub_mismatch += cands[k0][1]
        if example is None and cands[k0][1]:
            idx = int(((cands[k0][2] != hw[k0[0]]) & sub).nonzero()[0])
            example = (float(p[idx]), int(bitsr[idx]) & 0xFFFFFFFF, int(hw[k0[0]][idx]) & 0xFFFF, int(cands[k0][2][idx]) & 0xFFFF)
    with capsys.disabled():
        print("\ncvt.rs.f16x2.f32 vs R13: mapping(s) %s identical on %d normal-grid samples; below 2^-14: %d of %d differ; first counter-example "
              "(p, rbits, hardware, R13) = %s" % (found, normal_total, sub_mismatch, sub_total, example))
    assert normal_total > 6e8
    # the outcome this build records: identical on the normal grid, not below it
    assert sub_mismatch > 0
