"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json:north_star's:
  hash .................. bit-exact
  integer-valued input .. bit-exact (FP16 and FP32, every variant)
  FP32 accumulate ....... rel. Frobenius error <= 1e-5 vs the FP64 oracle
  FP16 RN ............... relF <= 1.5 x the oracle's sequential-FP16 relF on that input, and <= 5e-2
"""
import numpy as np
import pytest

import evaluation as ev
import oracle
import workloads as wl
from workloads import sketch_seed

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ss():
    import paper_2606_20195_b200 as ss_

    assert torch.cuda.is_available()
    return ss_


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def bits(t):
    """FP16 tensor -> uint16 bit patterns with -0 canonicalised to +0 (R10)."""
    b = t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()
    b[b == 0x8000] = 0
    return b


F16_VARIANTS = ["auto", "flat_pair", "flat_vec", "smem", "tmem", "small", "generic"]
F32_VARIANTS = ["auto", "flat_pair", "flat_vec", "generic"]
VID = {"auto": 0, "flat_pair": 1, "flat_vec": 2, "smem": 3, "generic": 4, "tmem": 5, "small": 6}


def feasible(ss, sk, A, variant, f16=True, **kw):
    """The host-side plan decides whether a forced variant can run this shape (SKETCH_ERR_UNSUPPORTED = -6 comes from
    make_plan only); any other error is a failure."""
    plan_kw = {k: v for k, v in kw.items() if k in ("row_begin", "rows", "replicas", "hash_mode", "grid_ctas", "tmem_group_mode")}
    plan_kw.setdefault("rows", int(A.shape[0]))
    rounding = kw.get("rounding", 0)
    try:
        sk.plan(int(A.shape[1]), lda=int(A.stride(0)) if A.shape[0] > 1 else int(A.shape[1]), f16=f16, rounding=rounding,
                variant=VID[variant], **plan_kw)
        return True
    except ss.SketchError as e:
        assert e.code == -6, e
        return False


def apply16(ss, sk, A, variant="auto", **kw):
    """Forced variant: must run iff the plan says it can; an infeasible (variant, shape) must fail with -6 and is skipped
    with its reason.  A -6 / -7 on a feasible plan is a test failure."""
    if not feasible(ss, sk, A, variant, True, **kw):
        with pytest.raises(ss.SketchError) as ei:
            sk.apply_f16acc(A, variant=VID[variant], **kw)
        assert ei.value.code == -6
        pytest.skip("plan: variant %s cannot run m=%d n=%d d=%d zeta=%d rounding=%d" % (variant, sk.m, A.shape[1], sk.d, sk.zeta, kw.get("rounding", 0)))
    return sk.apply_f16acc(A, variant=VID[variant], **kw)


def apply32(ss, sk, A, variant="auto", **kw):
    if not feasible(ss, sk, A, variant, False, **kw):
        with pytest.raises(ss.SketchError) as ei:
            sk.apply_f32acc(A, variant=VID[variant], **kw)
        assert ei.value.code == -6
        pytest.skip("plan: variant %s cannot run the FP32 path at n=%d d=%d zeta=%d" % (variant, A.shape[1], sk.d, sk.zeta))
    return sk.apply_f32acc(A, variant=VID[variant], **kw)


# ------------------------------------------------------------------------------------ hash (a1)
@pytest.mark.parametrize("m,d,zeta,seed", [
    (4096, 32, 4, 0), (4096, 32, 1, 0), (1 << 20, 128, 4, 1), (100003, 256, 8, 0xDEADBEEF),
    (5000, 30, 3, sketch_seed(1)), (70000, 1 << 20, 2, sketch_seed(2)), (777, 2048, 16, sketch_seed(3)),
])
def test_hashes_bit_exact(ss, m, d, zeta, seed):
    sk = ss.Sketch(m, d, zeta, seed)
    b, s = sk.hashes_dump()
    ob, osn = oracle.hashes(seed, d, zeta, m)
    assert np.array_equal(b.cpu().numpy(), ob)
    assert np.array_equal(s.cpu().numpy(), osn)


def test_hashes_full_size_config5_sampled(ss):
    # BASELINE config 5: m = 2^25, d = 256, zeta = 4 -> 2^27 (row, block) pairs; oracle checks sampled rows,
    # structure checked everywhere
    m, d, zeta, seed = 1 << 25, 256, 4, sketch_seed(5)
    sk = ss.Sketch(m, d, zeta, seed)
    b, s = sk.hashes_dump()
    db = d // zeta
    j = torch.arange(zeta, device="cuda", dtype=torch.int32)[None, :]
    assert bool(((b >= j * db) & (b < (j + 1) * db)).all())          # one bucket per block
    cnt = torch.bincount(b.reshape(-1).long(), minlength=d).double()
    assert abs(float(cnt.mean()) - m * zeta / d) < 1e-6               # mean depth m*zeta/d
    assert float(((cnt - cnt.mean()) ** 2 / cnt.mean()).sum()) < d + 6 * (2 * d) ** 0.5
    for r0 in (0, 12345678, m - 4096):
        ob, osn = oracle.hashes(seed, d, zeta, 4096, row_begin=r0)
        assert np.array_equal(b[r0:r0 + 4096].cpu().numpy(), ob)
        assert np.array_equal(s[r0:r0 + 4096].cpu().numpy(), osn)


# ------------------------------------------------------------------------------------ exact cases
SHAPES_EXACT = [
    # (m, n, d, zeta)   -- config 1, then shapes spanning several tiles with ragged tails
    (4096, 16, 32, 4), (4096, 16, 32, 1), (10007, 64, 128, 4), (33333, 128, 256, 4), (9999, 128, 256, 1),
    (5001, 256, 64, 4), (777, 24, 16, 4), (3000, 8, 8, 1),
    # config-4 shaped sketches (256 KiB - 1 MiB): bucket groups and column slices of the tensor-memory kernel
    (6007, 256, 512, 4), (6007, 256, 1024, 4), (4099, 256, 2048, 4), (5003, 512, 512, 4), (7001, 128, 1024, 4),
    (3001, 512, 128, 1),
    # up to eight column slices: the paper's width n = 1024 while the sketch fits, widths that are not 64 * 2^k
    (2501, 1024, 512, 4), (2501, 1024, 1024, 4), (2503, 384, 768, 4), (2503, 320, 640, 4), (2503, 192, 96, 1),
]


@pytest.mark.parametrize("variant", F16_VARIANTS)
@pytest.mark.parametrize("m,n,d,zeta", SHAPES_EXACT)
def test_f16_integer_input_bit_exact(ss, variant, m, n, d, zeta):
    # scale 1/2 (zeta=4) or 1 is exact; entries in {-3..3}; sums stay exact FP16 in any order
    A = wl.integer_valued(m, n, 100 + m % 97)
    seed = sketch_seed(m + zeta)
    want = oracle.f64_sketch(seed, d, zeta, A)
    assert np.abs(want).max() < 1024
    sk = ss.Sketch(m, d, zeta, seed)
    got = apply16(ss, sk, dev(A), variant)
    assert np.array_equal(oracle.half_bits_to_f64(bits(got)), want)
    assert np.array_equal(bits(got), oracle.seq16_sketch(seed, d, zeta, A))


@pytest.mark.parametrize("variant", F32_VARIANTS)
@pytest.mark.parametrize("m,n,d,zeta", SHAPES_EXACT)
def test_f32_integer_input_bit_exact(ss, variant, m, n, d, zeta):
    A = wl.integer_valued(m, n, 100 + m % 97)
    seed = sketch_seed(m + zeta)
    want = oracle.f64_sketch(seed, d, zeta, A)
    sk = ss.Sketch(m, d, zeta, seed)
    got = apply32(ss, sk, dev(A), variant)
    assert np.array_equal(got.cpu().numpy().astype(np.float64), want)


@pytest.mark.parametrize("zeta", [2, 8, 3, 16])
def test_other_sparsities_against_f64(ss, zeta):
    # zeta in {2,8}: irrational scale -> tolerance test; zeta=3,16 run the generic kernel
    m, n, d = 20011, 64, 48 * zeta
    A = wl.gaussian(m, n, 200 + zeta)
    seed = sketch_seed(300 + zeta)
    B = oracle.f64_sketch(seed, d, zeta, A)
    sk = ss.Sketch(m, d, zeta, seed)
    assert ev.rel_fro(sk.apply_f32acc(dev(A)).cpu().numpy(), B) <= 1e-5
    D16 = oracle.half_bits_to_f64(oracle.seq16_sketch(seed, d, zeta, A))
    ref = ev.rel_fro(D16, B)
    ran = []
    for variant in F16_VARIANTS:
        if not feasible(ss, sk, dev(A), variant):
            continue
        got = sk.apply_f16acc(dev(A), variant=VID[variant])
        ran.append(variant)
        r = ev.rel_fro(oracle.half_bits_to_f64(bits(got)), B)
        assert r <= 1.5 * ref and r <= 5e-2, (variant, r, ref)
    assert "auto" in ran and "generic" in ran and (zeta not in (2, 8) or {"flat_vec", "tmem"} <= set(ran)), ran


# ------------------------------------------------------------------------------------ tolerance cases
SHAPES_TOL = [(4096, 16, 32, 4), (4096, 16, 32, 1), (50021, 64, 128, 4), (70001, 128, 256, 4), (30011, 256, 512, 4)]


@pytest.mark.parametrize("m,n,d,zeta", SHAPES_TOL)
def test_f32_within_1e5_of_f64_oracle(ss, m, n, d, zeta):
    A = wl.gaussian(m, n, m % 89)
    seed = sketch_seed(m)
    B = oracle.f64_sketch(seed, d, zeta, A)
    sk = ss.Sketch(m, d, zeta, seed)
    for variant in F32_VARIANTS:
        got = sk.apply_f32acc(dev(A), variant=VID[variant]).cpu().numpy()
        assert ev.rel_fro(got, B) <= 1e-5, variant


@pytest.mark.parametrize("m,n,d,zeta", SHAPES_TOL)
def test_f16_rn_error_vs_sequential_oracle(ss, m, n, d, zeta):
    A = wl.gaussian(m, n, m % 89)
    seed = sketch_seed(m)
    B = oracle.f64_sketch(seed, d, zeta, A)
    ref = ev.rel_fro(oracle.half_bits_to_f64(oracle.seq16_sketch(seed, d, zeta, A)), B)
    sk = ss.Sketch(m, d, zeta, seed)
    ran = []
    for variant in F16_VARIANTS:
        if not feasible(ss, sk, dev(A), variant):
            continue
        got = sk.apply_f16acc(dev(A), variant=VID[variant])
        ran.append(variant)
        r = ev.rel_fro(oracle.half_bits_to_f64(bits(got)), B)
        assert r <= 1.5 * ref and r <= 5e-2, (variant, r, ref)
        assert r > 0.02 * ref      # it really is an FP16 accumulation, not a widened one
    assert {"auto", "flat_vec", "flat_pair", "generic"} <= set(ran), ran


# ------------------------------------------------------------------------------------ conversion through the ABI
def _singleton_setup(ss, zeta, d, m, n, seed):
    sk = ss.Sketch(m, d, zeta, seed)
    b, s = oracle.hashes(seed, d, zeta, m)
    cnt = np.bincount(b.ravel(), minlength=d)
    return sk, b, s, cnt


SPECIALS = np.array([
    2.0 ** -25, np.nextafter(np.float32(2.0 ** -25), np.float32(1)), 3 * 2.0 ** -25, 5 * 2.0 ** -25, 2.0 ** -24, 2.0 ** -14,
    np.nextafter(np.float32(2.0 ** -14), np.float32(0)), 65504.0, 65519.996, 65520.0, 70000.0, 1e30, 32768.0,
    1.0 + 2.0 ** -11, 1.0 + 3 * 2.0 ** -11, 0.0, 1e-30, 1e-42, 6.1e-5, 0.33333334, 1000.123,
], dtype=np.float32)


@pytest.mark.parametrize("variant", F16_VARIANTS)
@pytest.mark.parametrize("zeta", [1, 4])
def test_rn_conversion_edge_cases_singleton_buckets(ss, variant, zeta):
    # m small, d large: a sketch entry hit once equals RN16(s*a) bit-exactly (0 + v = v)
    m, n, d = 64, 64, 65536
    seed = sketch_seed(77 + zeta)
    sk, b, s, cnt = _singleton_setup(ss, zeta, d, m, n, seed)
    rng = np.random.default_rng(5)
    A = rng.standard_normal((m, n)).astype(np.float32) * np.exp2(rng.integers(-30, 18, (m, n))).astype(np.float32)
    A[:, :SPECIALS.size] = SPECIALS[None, :] * np.where(rng.random((m, 1)) < 0.5, -1, 1).astype(np.float32)
    got = bits(apply16(ss, sk, dev(A), variant))
    sc = oracle.scale_f32(zeta)
    checked = 0
    for i in range(m):
        for j in range(zeta):
            if cnt[b[i, j]] == 1:
                es = np.float32(-sc if s[i, j] else sc)
                want = oracle.rn16(es * A[i])
                want[want == 0x8000] = 0
                assert np.array_equal(got[b[i, j]], want), (i, j)
                checked += 1
    assert checked > m * zeta * 0.9


@pytest.mark.parametrize("variant", F16_VARIANTS)
@pytest.mark.parametrize("zeta", [1, 4, 2])
def test_sr_conversion_bit_exact_singleton_buckets(ss, variant, zeta):
    # DESIGN.md R13/R14: the GPU's integer SR rule and counter layout against the oracle's real-number rule
    m, n, d = 48, 64, 65536
    seed, sr_seed = sketch_seed(88 + zeta), sketch_seed(99)
    sk, b, s, cnt = _singleton_setup(ss, zeta, d, m, n, seed)
    rng = np.random.default_rng(6)
    A = rng.standard_normal((m, n)).astype(np.float32) * np.exp2(rng.integers(-40, 17, (m, n))).astype(np.float32)
    A[:, :SPECIALS.size] = SPECIALS[None, :]
    got = bits(apply16(ss, sk, dev(A), variant, rounding=ss.SR, sr_seed=sr_seed))
    want_all = oracle.seq16_sketch(seed, d, zeta, A, rounding=oracle.SR, sr_seed=sr_seed)
    want_all[want_all == 0x8000] = 0
    rows = [b[i, j] for i in range(m) for j in range(zeta) if cnt[b[i, j]] == 1]
    assert len(rows) > m * zeta * 0.9
    assert np.array_equal(got[rows], want_all[rows])
    # SR differs from RN on this input (otherwise the test proves nothing)
    rn = bits(apply16(ss, sk, dev(A), variant))
    assert (rn[rows] != got[rows]).mean() > 0.1


def test_sr_is_unbiased_where_rn_erases(ss):
    # Cor. 3: contributions below h/2 vanish under RN but survive in expectation under SR
    m, n, d, zeta = 1 << 16, 64, 128, 4
    A = wl.gaussian(m, n, 7, pow2=-27)            # |s*a| ~ 2^-28 << h/2 (RN -> nonzero needs |g| > 8)
    seed = sketch_seed(123)
    sk = ss.Sketch(m, d, zeta, seed)
    Ad = dev(A)
    assert int(torch.count_nonzero(sk.apply_f16acc(Ad))) == 0       # RN erases everything
    B = oracle.f64_sketch(seed, d, zeta, A)
    acc = np.zeros_like(B)
    T = 8
    for t in range(T):
        acc += oracle.half_bits_to_f64(bits(sk.apply_f16acc(Ad, rounding=ss.SR, sr_seed=sketch_seed(1000 + t))))
    corr = float((acc * B).sum() / np.sqrt((acc * acc).sum() * (B * B).sum()))
    scale = float((acc / T * B).sum() / (B * B).sum())
    assert corr > 0.3 and 0.6 < scale < 1.4, (corr, scale)


# ------------------------------------------------------------------------------------ ABI features
@pytest.mark.parametrize("variant", F16_VARIANTS)
def test_row_ranges_accumulate_and_lda(ss, variant):
    m, n, d, zeta = 20000, 64, 128, 4
    A = wl.integer_valued(m, n, 11)
    seed = sketch_seed(55)
    want = oracle.f64_sketch(seed, d, zeta, A)
    sk = ss.Sketch(m, d, zeta, seed)
    # padded leading dimension
    Ap = torch.full((m, n + 8), float("nan"), device="cuda")
    Ap[:, :n] = dev(A)
    # the privatised kernel needs row ranges that start on a multiple of 4 (aligned row groups); ragged ends are fine
    cuts = ((0, 36), (36, 12000), (12000, m)) if variant == "smem" else ((0, 37), (37, 12001), (12001, m))
    out = None
    for k, (r0, r1) in enumerate(cuts):
        out = apply16(ss, sk, Ap[r0:r1, :n], variant, out=out, row_begin=r0, accumulate=k > 0)
    assert np.array_equal(oracle.half_bits_to_f64(bits(out)), want)
    if variant == "auto":   # auto falls back to the flat kernel for a range that starts off the 4-row grid
        assert sk.plan(n, row_begin=37, rows=100)["variant"] == "flat_vec" and sk.plan(n, row_begin=36, rows=100)["variant"] == "smem"
        assert sk.plan(n)["variant"] == "tmem"          # large enough ranges go to tensor memory, any row_begin
    out32 = None
    for k, (r0, r1) in enumerate(((0, 37), (37, 12001), (12001, m))):
        out32 = sk.apply_f32acc(Ap[r0:r1, :n], out=out32, row_begin=r0, accumulate=k > 0,
                                variant=VID[variant] if variant not in ("smem", "tmem", "small") else 0)
    assert np.array_equal(out32.cpu().numpy().astype(np.float64), want)


@pytest.mark.parametrize("d", [512, 1024, 2048])
def test_tmem_column_slices_row_ranges_accumulate_and_lda(ss, d):
    # config-4 shaped sketches: bucket groups (d = 512) and column slices across CTAs (d = 1024, 2048) of the
    # tensor-memory kernel, on a padded leading dimension, in three row ranges accumulated into one sketch
    m, n, zeta = 9001, 256, 4
    A = wl.integer_valued(m, n, 13)
    seed = sketch_seed(56 + d)
    want = oracle.f64_sketch(seed, d, zeta, A)
    sk = ss.Sketch(m, d, zeta, seed)
    assert sk.plan(n)["variant"] == "tmem"
    Ap = torch.full((m, n + 12), float("nan"), device="cuda")
    Ap[:, :n] = dev(A)
    out = None
    for k, (r0, r1) in enumerate(((0, 37), (37, 4001), (4001, m))):
        out = apply16(ss, sk, Ap[r0:r1, :n], "tmem", out=out, row_begin=r0, accumulate=k > 0)
    assert np.array_equal(oracle.half_bits_to_f64(bits(out)), want)
    # Gaussian input: north-star tolerances
    G = wl.gaussian(m, n, 14)
    B = oracle.f64_sketch(seed, d, zeta, G)
    ref = ev.rel_fro(oracle.half_bits_to_f64(oracle.seq16_sketch(seed, d, zeta, G)), B)
    got = ev.rel_fro(oracle.half_bits_to_f64(bits(apply16(ss, sk, dev(G), "tmem"))), B)
    assert got <= 1.5 * ref and got <= 5e-2, (got, ref)


def test_tmem_wide_rows_on_a_padded_leading_dimension(ss):
    # strided tiles come through a 2-D tensor map whose box is at most 256 elements wide: n = 512 / 1024 with lda > n must
    # pick more column slices than the contiguous case does, and still be exact
    m, zeta = 4001, 4
    for n, d in ((512, 128), (1024, 256), (256, 64)):
        A = wl.integer_valued(m, n, 15)
        seed = sketch_seed(600 + n)
        want = oracle.f64_sketch(seed, d, zeta, A)
        sk = ss.Sketch(m, d, zeta, seed)
        Ap = torch.full((m, n + 4), float("nan"), device="cuda")
        Ap[:, :n] = dev(A)
        for view in (Ap[:, :n], dev(A)):
            got = apply16(ss, sk, view, "tmem")
            assert np.array_equal(oracle.half_bits_to_f64(bits(got)), want), (n, view.stride(0))


def test_odd_n_and_poor_alignment_take_the_generic_path(ss):
    m, d, zeta = 3001, 64, 4
    seed = sketch_seed(66)
    sk = ss.Sketch(m, d, zeta, seed)
    for n in (1, 3, 257 // 8 + 1, 20):
        A = wl.integer_valued(m, n, 12 + n)
        want = oracle.f64_sketch(seed, d, zeta, A)
        # view offset by one float: only 4-byte aligned
        buf = torch.zeros(m * n + 1, device="cuda")
        buf[1:] = dev(A).reshape(-1)
        Av = buf[1:].view(m, n)
        assert np.array_equal(oracle.half_bits_to_f64(bits(sk.apply_f16acc(Av))), want)
        assert np.array_equal(sk.apply_f32acc(Av).cpu().numpy().astype(np.float64), want)
    assert sk.plan(3)["variant"] == "generic"


def test_precomputed_hash_mode_matches_on_the_fly(ss):
    m, n, d, zeta = 40013, 128, 256, 4
    seed = sketch_seed(67)
    sk = ss.Sketch(m, d, zeta, seed)
    A = wl.integer_valued(m, n, 13)
    want = oracle.f64_sketch(seed, d, zeta, A)
    Ad = dev(A)
    for variant in ("flat_vec", "flat_pair"):
        got = sk.apply_f16acc(Ad, variant=VID[variant], hash_mode=2)
        assert np.array_equal(oracle.half_bits_to_f64(bits(got)), want)
        got32 = sk.apply_f32acc(Ad, variant=VID[variant], hash_mode=2)
        assert np.array_equal(got32.cpu().numpy().astype(np.float64), want)
    # wide packed entries (d > 32768)
    sk2 = ss.Sketch(5000, 1 << 17, 4, seed)
    A2 = wl.integer_valued(5000, 64, 14)
    got = sk2.apply_f16acc(dev(A2), variant=VID["flat_vec"], hash_mode=2)
    assert np.array_equal(oracle.half_bits_to_f64(bits(got)), oracle.f64_sketch(seed, 1 << 17, 4, A2))


def test_host_entry_points_match_device_entry_points(ss):
    m, n, d, zeta = 300007, 128, 256, 4     # > 1 staging chunk is exercised by the chunking inside (256 MiB)
    seed = sketch_seed(68)
    sk = ss.Sketch(m, d, zeta, seed)
    A = wl.integer_valued(m, n, 15)
    want = oracle.f64_sketch(seed, d, zeta, A, threads=8)
    Ah = torch.from_numpy(A).pin_memory()
    got = sk.apply_f16acc_host(Ah)
    assert np.array_equal(oracle.half_bits_to_f64(bits(got)), want)
    got32 = sk.apply_f32acc_host(Ah)
    assert np.array_equal(got32.numpy().astype(np.float64), want)


def test_replica_counts_and_grids(ss):
    m, n, d, zeta = 25013, 64, 128, 4
    seed = sketch_seed(69)
    sk = ss.Sketch(m, d, zeta, seed)
    A = wl.integer_valued(m, n, 16)
    want = oracle.f64_sketch(seed, d, zeta, A)
    Ad = dev(A)
    for P in (1, 2, 7, 64):
        for grid in (0, 1, 5, 333):
            got = sk.apply_f16acc(Ad, variant=VID["flat_vec"], replicas=P, grid_ctas=grid)
            assert np.array_equal(oracle.half_bits_to_f64(bits(got)), want), (P, grid)
    for variant in ("smem", "tmem"):
        for grid in (1, 3, 148, 1000):
            got = sk.apply_f16acc(Ad, variant=VID[variant], grid_ctas=grid)
            assert np.array_equal(oracle.half_bits_to_f64(bits(got)), want), (variant, grid)


def test_tiny_and_degenerate_inputs(ss):
    seed = sketch_seed(70)
    # one row, one column
    sk = ss.Sketch(1, 4, 4, seed)
    A = np.array([[3.0]], dtype=np.float32)
    want = oracle.f64_sketch(seed, 4, 4, A)
    assert np.array_equal(oracle.half_bits_to_f64(bits(sk.apply_f16acc(dev(A)))), want)
    assert np.array_equal(sk.apply_f32acc(dev(A)).cpu().numpy().astype(np.float64), want)
    # empty row range: complete-sketch semantics give zeros; accumulate leaves B alone
    sk = ss.Sketch(100, 32, 4, seed)
    A = dev(wl.integer_valued(100, 16, 1))
    out = torch.full((32, 16), 7.0, dtype=torch.float16, device="cuda")
    lib = ss.lib()
    import ctypes as C
    o = ss.SketchOpts(0, 0, 0, 1, 100, 0, 0, 0)   # row_begin = m -> zero rows, accumulate
    st = torch.cuda.current_stream().cuda_stream
    assert lib.sketch_apply_f16acc_ex(sk._h, A.data_ptr(), 16, 16, out.data_ptr(), 0, 0, C.byref(o), st) == 0
    torch.cuda.synchronize()
    assert bool((out == 7).all())
    o = ss.SketchOpts(0, 0, 0, 0, 100, 0, 0, 0)
    assert lib.sketch_apply_f16acc_ex(sk._h, A.data_ptr(), 16, 16, out.data_ptr(), 0, 0, C.byref(o), st) == 0
    torch.cuda.synchronize()
    assert bool((out == 0).all())
    # d = zeta (one row per block): every contribution of a block lands in one row
    sk = ss.Sketch(5000, 4, 4, seed)
    A = wl.integer_valued(5000, 64, 2, lo=-1, hi=1)
    want = oracle.f64_sketch(seed, 4, 4, A)
    assert np.array_equal(oracle.half_bits_to_f64(bits(sk.apply_f16acc(dev(A)))), want)


def test_subnormal_scale_is_exact_in_any_order(ss):
    # config 5, k = -24: contributions are 0, +-h, +-2h; partial sums are integer multiples of h,
    # exact up to 2048h in any order -> GPU FP16 == oracle SEQ16 bit for bit (and != 0: .noftz matters)
    m, n, d, zeta = 1 << 18, 64, 128, 4
    A = wl.gaussian(m, n, 17, pow2=-24)
    seed = sketch_seed(71)
    want = oracle.seq16_sketch(seed, d, zeta, A)
    mag = oracle.half_bits_to_f64(want) / 2.0 ** -24
    assert np.abs(mag).max() < 2048 and np.count_nonzero(want) > 0.9 * want.size
    sk = ss.Sketch(m, d, zeta, seed)
    want[want == 0x8000] = 0
    for variant in ("tmem", "smem", "small", "flat_vec", "flat_pair"):
        assert np.array_equal(bits(sk.apply_f16acc(dev(A), variant=VID[variant])), want), variant


def test_overflow_saturates_like_the_oracle(ss):
    # config 5, k = +12: running sums leave the FP16 range and stick at +-inf.  No single contribution
    # converts to inf, so a flat running sum never makes NaN; hierarchical variants can (+inf partial
    # plus -inf partial = NaN, reading R9).  Order-dependent, so compare the class, not the bits.
    m, n, d, zeta = 1 << 16, 64, 128, 4
    A = wl.gaussian(m, n, 18, pow2=12)
    seed = sketch_seed(72)
    sk = ss.Sketch(m, d, zeta, seed)
    want = oracle.half_bits_to_f64(oracle.seq16_sketch(seed, d, zeta, A))
    assert not np.isnan(want).any()
    over_want = (~np.isfinite(want)).mean()
    # the exact sums have std ~ 2^12 * 0.5 * sqrt(2048) = 9.3e4 > 65504: a large share overflows
    assert 0.2 < over_want < 0.95
    B = oracle.f64_sketch(seed, d, zeta, A)
    for variant, kw in (("tmem", {}), ("smem", {}), ("flat_vec", {"replicas": 1}), ("flat_vec", {"replicas": 8})):
        got = oracle.half_bits_to_f64(bits(sk.apply_f16acc(dev(A), variant=VID[variant], **kw)))
        over = (~np.isfinite(got)).mean()
        assert abs(over - over_want) < 0.3, (variant, over, over_want)
        if kw.get("replicas") == 1:
            assert not np.isnan(got).any()
        fin = np.isfinite(got)
        assert fin.sum() > 0 and ev.rel_fro(got[fin], B[fin]) < 0.2


# ------------------------------------------------------------------------------------ error contract
def test_forced_variant_fails_iff_the_plan_says_so_and_auto_never_does(ss):
    seed = sketch_seed(73)
    # a sketch far beyond tensor memory / shared memory: forced privatised variants are refused by the PLAN (no launch,
    # B untouched), AUTO runs the flat kernel
    m, n, d, zeta = 3000, 1024, 8192, 4
    sk = ss.Sketch(m, d, zeta, seed)
    A = dev(wl.integer_valued(m, n, 21))
    out = torch.full((d, n), 7.0, dtype=torch.float16, device="cuda")
    before = ss.sketch_launch_count()
    for variant in ("tmem", "smem", "small"):
        with pytest.raises(ss.SketchError) as ei:
            sk.plan(n, variant=VID[variant])
        assert ei.value.code == -6
        with pytest.raises(ss.SketchError) as ei:
            sk.apply_f16acc(A, out=out, variant=VID[variant])
        assert ei.value.code == -6
    assert ss.sketch_launch_count() == before and bool((out == 7).all())
    assert sk.plan(n)["variant"] == "flat_vec"
    got = sk.apply_f16acc(A)
    assert np.array_equal(oracle.half_bits_to_f64(bits(got)), oracle.f64_sketch(seed, d, zeta, wl.integer_valued(m, n, 21)))
    # SR / dither / FP32 on the RN-only privatised variants (the tensor-memory kernel has every mode), odd n on the vector variants
    sk2 = ss.Sketch(5000, 256, 4, seed)
    A2 = dev(wl.integer_valued(5000, 128, 22))
    for variant in ("smem", "small"):
        for rnd in (ss.SR, ss.DITHER):
            with pytest.raises(ss.SketchError) as ei:
                sk2.apply_f16acc(A2, variant=VID[variant], rounding=rnd, sr_seed=1)
            assert ei.value.code == -6
        with pytest.raises(ss.SketchError) as ei:
            sk2.apply_f32acc(A2, variant=VID[variant])
        assert ei.value.code == -6
        with pytest.raises(ss.SketchError) as ei:
            sk2.apply_bf16acc(A2, variant=VID[variant])
        assert ei.value.code == -6
    # per-contribution conversion keeps one bucket group in tensor memory: d = 1024 at n = 128 needs two -> refused for SR only
    sk3 = ss.Sketch(5000, 1024, 4, seed)
    sk3.apply_f16acc(A2, variant=VID["tmem"])
    with pytest.raises(ss.SketchError) as ei:
        sk3.apply_f16acc(A2, variant=VID["tmem"], rounding=ss.SR, sr_seed=1)
    assert ei.value.code == -6
    # a rounding rule that does not exist, or one on the wrong element type
    with pytest.raises(ss.SketchError) as ei:
        sk2.apply_f16acc(A2, rounding=3)
    assert ei.value.code == -1
    A3 = dev(wl.integer_valued(5000, 33, 23))
    for variant in ("flat_vec", "flat_pair", "tmem", "smem", "small"):
        with pytest.raises(ss.SketchError) as ei:
            sk2.apply_f16acc(A3, variant=VID[variant])
        assert ei.value.code == -6
    # AUTO over a sweep of awkward shapes: always a plan, never -6
    for (mm, nn, dd, zz) in ((10, 1, 3, 3), (100, 7, 14, 7), (5000, 66, 132, 4), (5000, 1088, 64, 1), (200, 4096, 8, 8), (70, 130, 52, 2)):
        skx = ss.Sketch(mm, dd, zz, seed)
        Ax = wl.integer_valued(mm, nn, 24)
        assert skx.plan(nn)["variant"] in VID
        if zz in (1, 4):
            assert np.array_equal(oracle.half_bits_to_f64(bits(skx.apply_f16acc(dev(Ax)))), oracle.f64_sketch(seed, dd, zz, Ax))


@pytest.mark.parametrize("n,zeta", [(64000, 1), (64000, 4), (32002, 1), (32002, 8), (20000, 2), (100000, 4)])
def test_very_wide_rows_index_exactly(ss, n, zeta):
    # the flat kernels split a macro step of 32/zeta rows into chunks with a multiply-high division that is exact only for
    # (32/zeta) (n/VEC)^2 <= 2^32; wider rows must take the exact division (n/VEC = 16000, 16001, 20000, 50000 used to fail)
    m, d = 131, 8 * zeta
    A = wl.integer_valued(m, n, 31, lo=-1, hi=1)
    seed = sketch_seed(74 + zeta)
    sk = ss.Sketch(m, d, zeta, seed)
    Ad = dev(A)
    if zeta in (1, 4):
        want = oracle.f64_sketch(seed, d, zeta, A)
        for variant in ("flat_vec", "flat_pair"):
            assert np.array_equal(oracle.half_bits_to_f64(bits(apply16(ss, sk, Ad, variant))), want), variant
            assert np.array_equal(apply32(ss, sk, Ad, variant).cpu().numpy().astype(np.float64), want), variant
    else:
        G = wl.gaussian(m, n, 32)
        B = oracle.f64_sketch(seed, d, zeta, G)
        for variant in ("flat_vec", "flat_pair"):
            assert ev.rel_fro(apply32(ss, sk, dev(G), variant).cpu().numpy(), B) <= 1e-5
            assert ev.rel_fro(oracle.half_bits_to_f64(bits(apply16(ss, sk, dev(G), variant))), B) <= 5e-3


def test_odd_sized_sketch_never_touches_memory_past_B(ss):
    # d * n odd: the last element has no partner word inside B: it is added by a 16-bit CAS, partial sketches
    # and host-path slots are padded to 16 bytes
    seed = sketch_seed(75)
    for (m, n, d, zeta) in ((4000, 3, 5, 1), (4000, 7, 9, 3), (4000, 1, 7, 7)):
        A = wl.integer_valued(m, n, 33, lo=-1, hi=1)
        want = oracle.f64_sketch(seed, d, zeta, A) if zeta == 1 else None
        sk = ss.Sketch(m, d, zeta, seed)
        for P in (1, 3):
            buf = torch.full((d * n + 9,), 7.0, dtype=torch.float16, device="cuda")
            out = buf[: d * n].view(d, n)
            sk.apply_f16acc(dev(A), out=out, replicas=P)
            torch.cuda.synchronize()
            assert bool((buf[d * n:] == 7).all()), (m, n, d, zeta, P)
            if want is not None:
                assert np.array_equal(oracle.half_bits_to_f64(bits(out)), want)
            else:
                B = oracle.f64_sketch(seed, d, zeta, A)
                assert ev.rel_fro(oracle.half_bits_to_f64(bits(out)), B) <= 5e-3
    # host entry point with an odd sketch and more than one 256 MiB chunk (slot 1 used to be 2-byte aligned only)
    m, n, d, zeta = 23_000_000, 3, 5, 1
    rng = np.random.default_rng(34)
    A = (rng.random((m, n)) < 0.001).astype(np.float32)
    sk = ss.Sketch(m, d, zeta, seed)
    got = sk.apply_f16acc_host(torch.from_numpy(A))
    assert np.array_equal(oracle.half_bits_to_f64(bits(got)), oracle.f64_sketch(seed, d, zeta, A, threads=8))
    # an empty A through the binding is the empty range, not "all m rows"
    empty = torch.empty((0, 16), dtype=torch.float32, device="cuda")
    sk = ss.Sketch(100, 32, 4, seed)
    assert int(torch.count_nonzero(sk.apply_f16acc(empty, rows=0))) == 0


# ------------------------------------------------------------------------------------ stream semantics
@pytest.mark.parametrize("m,n,d,zeta,pad", [
    (4096, 16, 32, 4, 0),        # c1: launch-bound variants (SMALL / flat straight into B)
    (1 << 17, 64, 128, 4, 0),    # c2-shaped: tensor memory, contiguous tiles; FP32 through replicated partials + fold
    (20000, 256, 1024, 4, 0),    # tensor memory, two column slices: the cached tensor-map path
    (20000, 128, 256, 4, 8),     # padded leading dimension: tensor-map path
    (9000, 20, 16, 2, 0),        # flat FP16 with replicas
])
def test_applies_are_asynchronous_capturable_and_allocation_free(ss, m, n, d, zeta, pad):
    # SURVEY.md:309-310: "asynchronous on the given stream, never synchronises, never allocates per call".  A CUDA graph
    # capture (global mode) fails on any synchronisation or allocation inside the captured region, so: one warm-up call on
    # a non-default stream (first-use scratch allocation is allowed there), then capture f16acc + f32acc, replay, compare.
    seed = sketch_seed(76 + n)
    sk = ss.Sketch(m, d, zeta, seed)
    exact = zeta in (1, 4)
    gen = (lambda s_: wl.integer_valued(m, n, s_)) if exact else (lambda s_: wl.gaussian(m, n, s_))
    A1, A2 = gen(41), gen(42)
    buf = torch.zeros((m, n + pad), device="cuda")
    A = buf[:, :n]
    A.copy_(dev(A1))
    out16 = torch.empty((d, n), dtype=torch.float16, device="cuda")
    out32 = torch.empty((d, n), dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        sk.apply_f16acc(A, out=out16)
        sk.apply_f32acc(A, out=out32)
    side.synchronize()
    launches0 = ss.sketch_launch_count()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        sk.apply_f16acc(A, out=out16)
        sk.apply_f32acc(A, out=out32)
    per_capture = ss.sketch_launch_count() - launches0
    assert per_capture >= 2
    out16.fill_(3)
    out32.fill_(3)
    A.copy_(dev(A2))                      # the graph reads the buffers, not a snapshot
    for _ in range(10):
        g.replay()
    torch.cuda.synchronize()
    assert ss.sketch_launch_count() - launches0 == per_capture          # replays go through no library call
    B = oracle.f64_sketch(seed, d, zeta, A2)
    if exact:
        assert np.array_equal(oracle.half_bits_to_f64(bits(out16)), B)
        assert np.array_equal(out32.cpu().numpy().astype(np.float64), B)
    else:
        assert ev.rel_fro(out32.cpu().numpy(), B) <= 1e-5
        assert ev.rel_fro(oracle.half_bits_to_f64(bits(out16)), B) <= 5e-3


def test_capture_allocates_nothing_and_captured_scratch_survives_regrowth(ss):
    # include/sparse_sketch.h "CUDA graphs": (1) a capture that would have to create library scratch fails with
    # SKETCH_ERR_CAPTURE (-10) instead of running cudaMalloc inside the capture; (2) a scratch buffer a graph was captured
    # with is kept until sketch_destroy even when a later eager apply on another stream needs a larger one, so the replay
    # after that regrowth still reads and writes live memory.  Flat FP16 with 8 partial sketches = the scratch path.
    m, n, n_big, d, zeta = 20000, 64, 512, 128, 4
    seed = sketch_seed(91)
    sk = ss.Sketch(m, d, zeta, seed)
    A1, A2, A3 = wl.integer_valued(m, n, 51), wl.integer_valued(m, n, 52), wl.integer_valued(m, n_big, 53)
    A = dev(A1)
    out = torch.empty((d, n), dtype=torch.float16, device="cuda")
    side, other = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    kw = dict(variant=VID["flat_vec"], replicas=8)
    pl = sk.plan(n, **kw)
    assert pl["variant"] == "flat_vec" and pl["replicas"] == 8
    # (1) first use inside a capture: refused, nothing launched
    g0 = torch.cuda.CUDAGraph()
    launches0 = ss.sketch_launch_count()
    code, text = None, ""
    with torch.cuda.graph(g0, stream=side):
        out.zero_()                                   # keeps the aborted capture non-empty
        try:
            sk.apply_f16acc(A, out=out, **kw)
        except ss.SketchError as e:
            code, text = e.code, str(e)
    assert code == -10 and "capture" in text
    assert ss.sketch_launch_count() == launches0
    del g0
    # the same for the packed hash array (hash_mode 2) and for building it explicitly
    g0 = torch.cuda.CUDAGraph()
    codes = []
    with torch.cuda.graph(g0, stream=side):
        out.zero_()
        for call in (lambda: sk.apply_f16acc(A, out=out, variant=VID["flat_vec"], replicas=1, hash_mode=2), lambda: sk.precompute_hashes(stream=side)):
            try:
                call()
                codes.append(0)
            except ss.SketchError as e:
                codes.append(e.code)
    assert codes == [-10, -10]
    del g0
    # (2) warm-up outside, capture, replay
    with torch.cuda.stream(side):
        sk.apply_f16acc(A, out=out, **kw)
    side.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        sk.apply_f16acc(A, out=out, **kw)
    A.copy_(dev(A2))
    out.fill_(3)
    g.replay()
    torch.cuda.synchronize()
    want2 = oracle.f64_sketch(seed, d, zeta, A2)
    assert np.array_equal(oracle.half_bits_to_f64(bits(out)), want2)
    # an eager apply with eight times the columns on another stream: the handle's partial-sketch buffer has to grow
    Ab = dev(A3)
    with torch.cuda.stream(other):
        big = sk.apply_f16acc(Ab, variant=VID["flat_vec"], replicas=8)
    other.synchronize()
    assert np.array_equal(oracle.half_bits_to_f64(bits(big)), oracle.f64_sketch(seed, d, zeta, A3))
    # churn the allocator so that a freed buffer would have been handed out again and overwritten
    junk = [torch.full((1 << 18,), 7.0, device="cuda") for _ in range(16)]
    torch.cuda.synchronize()
    for _ in range(3):
        out.fill_(3)
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(oracle.half_bits_to_f64(bits(out)), want2)
    del junk, g
    sk.close()


def test_one_handle_on_two_streams_keeps_its_scratch_ordered(ss):
    # the replicated partial sketches and the packed hash array belong to the handle; applies on different streams are
    # ordered behind each other's use of them
    m, n, d, zeta = 60000, 64, 128, 4
    seed = sketch_seed(77)
    sk = ss.Sketch(m, d, zeta, seed)
    A1, A2 = wl.integer_valued(m, n, 43), wl.integer_valued(m, n, 44)
    want1, want2 = oracle.f64_sketch(seed, d, zeta, A1), oracle.f64_sketch(seed, d, zeta, A2)
    d1, d2 = dev(A1), dev(A2)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    o1 = [torch.empty((d, n), dtype=torch.float32, device="cuda") for _ in range(12)]
    o2 = [torch.empty((d, n), dtype=torch.float16, device="cuda") for _ in range(12)]
    for k in range(12):
        with torch.cuda.stream(s1):
            sk.apply_f32acc(d1, out=o1[k], replicas=8)                                   # memset + RED + fold of s->rep
        with torch.cuda.stream(s2):
            sk.apply_f16acc(d2, out=o2[k], variant=VID["flat_vec"], replicas=5, hash_mode=2)   # s->rep again, and s->packed
    torch.cuda.synchronize()
    for k in range(12):
        assert np.array_equal(o1[k].cpu().numpy().astype(np.float64), want1), k
        assert np.array_equal(oracle.half_bits_to_f64(bits(o2[k])), want2), k


# ------------------------------------------------------------------------------------ full sizes
# BASELINE.json's full shapes in the launch configuration bench.py times (AUTO through the C ABI, resident input).
# The oracle cannot redo 16 GiB in seconds, so it recomputes SAMPLED COLUMNS of the sketch (S acts on every column
# independently: column c of S A is S applied to column c of A) from the same bytes, copied back from the device.
FULL_SIZES = [
    # (name, m, n, d, zeta, expected AUTO variant)
    ("c5", 1 << 25, 128, 256, 4, "tmem"),
    ("c4-512", 1 << 23, 256, 512, 4, "tmem"),
    ("c4", 1 << 23, 256, 1024, 4, "tmem"),
    ("c4-2048", 1 << 23, 256, 2048, 4, "tmem"),
    ("e1", 1 << 21, 1024, 2048, 4, "tmem"),
    ("e1-d4096", 1 << 21, 1024, 4096, 4, "flat_vec"),
    ("c3", 1 << 22, 128, 256, 4, "tmem"),
]


def _sample_cols(n):
    # both halves of a half2 pair, lane and warp / column-slice boundaries, the last pair
    c = {0, 1, 62, 63, 64, 65, n // 2 - 1, n // 2, n - 2, n - 1}
    c |= {64 * k + (7 * k + 3) % 64 for k in range(n // 64)}      # one column in every 64-feature slice (column slices / warps)
    return [x for x in sorted(c) if 0 <= x < n]


@pytest.mark.parametrize("name,m,n,d,zeta,variant", FULL_SIZES)
def test_full_size_sampled_columns(ss, name, m, n, d, zeta, variant):
    free, _ = torch.cuda.mem_get_info()
    if free < m * n * 4 * 1.3:
        pytest.skip("not enough device memory for %s" % name)
    seed = sketch_seed(900 + d)
    sk = ss.Sketch(m, d, zeta, seed)
    assert sk.plan(n)["variant"] == variant
    cols = _sample_cols(n)
    threads = min(32, __import__("os").cpu_count() or 1)
    # (1) integer-valued sparse input: every FP16 partial sum exact in any order -> bit-exact on the sampled columns,
    #     FP16 and FP32 paths; the unsampled columns must at least agree between the two GPU paths exactly
    A = wl.sparse_signs_device(m, n, 31, torch.device("cuda"))
    got16 = sk.apply_f16acc(A)
    got32 = sk.apply_f32acc(A)
    Ac = np.ascontiguousarray(A[:, cols].cpu().numpy())
    want = oracle.f64_sketch(seed, d, zeta, Ac, threads=threads)
    assert np.abs(want).max() < 1024
    assert np.array_equal(oracle.half_bits_to_f64(bits(got16[:, cols])), want)
    assert np.array_equal(got32[:, cols].cpu().numpy().astype(np.float64), want)
    assert bool((got16.float() == got32).all())
    del got16, got32
    # (2) Gaussian input: north-star ceilings on the sampled columns
    A.normal_(generator=torch.Generator(device="cuda").manual_seed(32))
    got16 = sk.apply_f16acc(A)
    got32 = sk.apply_f32acc(A)
    Ac = np.ascontiguousarray(A[:, cols].cpu().numpy())
    B = oracle.f64_sketch(seed, d, zeta, Ac, threads=threads)
    r16 = ev.rel_fro(oracle.half_bits_to_f64(bits(got16[:, cols])), B)
    r32 = ev.rel_fro(got32[:, cols].cpu().numpy(), B)
    print("%s: relF f16 %.3e, f32 %.3e on %d sampled columns" % (name, r16, r32, len(cols)))
    assert r32 <= 1e-5, r32
    # FP16: never above 5e-2 (north star).  The flat kernel keeps one running sum per entry and replica, the
    # privatised kernels a two-level hierarchy; both stay far below at these depths (L = 2^14 .. 2^19)
    assert r16 <= 5e-2, r16
    if name in ("c5", "e1"):
        # the relative half of the north-star rule at the headline size: on two sampled columns (one column pair) the GPU's
        # hierarchical FP16 sum is no further from FP64 than 1.5 x the oracle's own sequential-FP16 sum of the same bytes
        two = [0, 1]
        seq = oracle.half_bits_to_f64(_seq16_columns(seed, d, zeta, np.ascontiguousarray(Ac[:, two])))
        ref = ev.rel_fro(seq, B[:, two])
        r2 = ev.rel_fro(oracle.half_bits_to_f64(bits(got16[:, [cols[k] for k in two]])), B[:, two])
        print("%s: relF on columns 0-1: gpu f16 %.3e, sequential-FP16 oracle %.3e" % (name, r2, ref))
        assert cols[0] == 0 and cols[1] == 1 and r2 <= 1.5 * ref, (r2, ref)


def _seq16_columns(seed, d, zeta, Ac, **kw):
    """Sequential-FP16 oracle on sampled columns, one host thread per column (columns are independent: each entry keeps
    its ascending (i, j) order)."""
    from concurrent.futures import ThreadPoolExecutor

    cols = [np.ascontiguousarray(Ac[:, c:c + 1]) for c in range(Ac.shape[1])]
    with ThreadPoolExecutor(max_workers=min(len(cols), __import__("os").cpu_count() or 1)) as ex:
        outs = list(ex.map(lambda a: oracle.seq16_sketch(seed, d, zeta, a, **kw), cols))
    return np.concatenate(outs, axis=1)


def test_config5_range_and_rounding_sweep_full_size(ss):
    # BASELINE.json configs[4] at its full size (m = 2^25, n = 128, d = 256, zeta = 4, 16 GiB): A = N(0,1) 2^k for
    # k in {-24, -16, 0, +8, +12}, RN and SR, in the launch configuration bench.py times.  Sampled columns against the oracle:
    #   k = -24 RN : bit-exact against the SEQUENTIAL FP16 oracle (every partial sum is an integer multiple of h, exact in
    #                any order while it stays within +-2048 h; SURVEY 8c conflict 3)
    #   k = -16, 0 : relF <= 5e-2 against FP64, RN and SR
    #   k = +8, +12: share of non-finite entries in the oracle's class (order-dependent: +-0.3), finite entries within 0.2
    m, n, d, zeta = 1 << 25, 128, 256, 4
    free, _ = torch.cuda.mem_get_info()
    if free < m * n * 4 * 1.2:
        pytest.skip("not enough device memory for config 5")
    seed, sr_seed = sketch_seed(905), sketch_seed(906)
    sk = ss.Sketch(m, d, zeta, seed)
    A = wl.gaussian_device(m, n, 4, torch.device("cuda"))
    cols = [0, 1, 63, 64, 127]
    threads = min(32, __import__("os").cpu_count() or 1)
    Ac = np.ascontiguousarray(A[:, cols].cpu().numpy())
    B0 = oracle.f64_sketch(seed, d, zeta, Ac, threads=threads)       # S (2^k A) = 2^k S A exactly
    prev = 0
    for k in (-24, -16, 0, 8, 12):
        A.mul_(float(2.0 ** (k - prev)))                              # exact in FP32
        prev = k
        want = B0 * 2.0 ** k
        Ack = np.ldexp(Ac, k).astype(np.float32)
        for rounding in (ss.RN, ss.SR):
            got = sk.apply_f16acc(A, rounding=rounding, sr_seed=sr_seed)
            g = oracle.half_bits_to_f64(bits(got[:, cols]))
            fin = np.isfinite(g)
            if k == -24 and rounding == ss.RN:
                seq = _seq16_columns(seed, d, zeta, Ack)
                mag = np.abs(oracle.half_bits_to_f64(seq)) / 2.0 ** -24
                seq[seq == 0x8000] = 0
                inside = mag < 2000                                    # an entry that left +-2048 h may differ (rare)
                assert inside.mean() > 0.99
                assert np.array_equal(bits(got[:, cols])[inside], seq[inside])
                assert np.count_nonzero(seq) > 0.9 * seq.size          # .noftz: subnormal sums survive
            elif k in (-16, 0):
                assert fin.all()
                r = ev.rel_fro(g, want)
                print("c5 k=%d rounding=%d: relF %.3e" % (k, rounding, r))
                assert r <= 5e-2, (k, rounding, r)
            elif k in (8, 12) and rounding == ss.RN:
                seq = oracle.half_bits_to_f64(_seq16_columns(seed, d, zeta, Ack))
                over_want, over = (~np.isfinite(seq)).mean(), (~fin).mean()
                print("c5 k=%d: non-finite share gpu %.3f, sequential oracle %.3f" % (k, over, over_want))
                assert abs(over - over_want) <= 0.3, (k, over, over_want)
                assert (over_want > 0.3) == (over > 0.3)
                if fin.any() and k == 8:
                    assert ev.rel_fro(g[fin], want[fin]) < 0.2
            elif k == -24:                                             # SR keeps tiny terms in expectation (Cor. 3)
                assert fin.all() and np.count_nonzero(g) > 0.5 * g.size


@pytest.mark.parametrize("zeta", [1, 2, 8])
def test_config3_sparsity_and_coherence_sweep_full_size(ss, zeta):
    # BASELINE.json configs[2] at its full size (m = 2^22, n = 128, d = 256) for the sparsities the round-1 full-size test
    # left out, and every alpha of the heavy-row generator; sampled columns against the FP64 oracle
    m, n, d = 1 << 22, 128, 256
    seed = sketch_seed(910 + zeta)
    sk = ss.Sketch(m, d, zeta, seed)
    assert sk.plan(n)["variant"] == "tmem"
    cols = _sample_cols(n)
    threads = min(32, __import__("os").cpu_count() or 1)
    if zeta == 1:   # scale 1: exact arithmetic on the sparse integer input
        A = wl.sparse_signs_device(m, n, 35, torch.device("cuda"))
        want = oracle.f64_sketch(seed, d, zeta, np.ascontiguousarray(A[:, cols].cpu().numpy()), threads=threads)
        g16, g32 = sk.apply_f16acc(A), sk.apply_f32acc(A)
        assert np.array_equal(oracle.half_bits_to_f64(bits(g16[:, cols])), want)
        assert np.array_equal(g32[:, cols].cpu().numpy().astype(np.float64), want)
        assert bool((g16.float() == g32).all())
        del A, g16, g32
    for alpha in (0.0, 0.5, 1.0):
        A = wl.heavy_rows_device(m, n, alpha, 36, torch.device("cuda"))
        B = oracle.f64_sketch(seed, d, zeta, np.ascontiguousarray(A[:, cols].cpu().numpy()), threads=threads)
        r16 = ev.rel_fro(oracle.half_bits_to_f64(bits(sk.apply_f16acc(A)[:, cols])), B)
        r32 = ev.rel_fro(sk.apply_f32acc(A)[:, cols].cpu().numpy(), B)
        print("c3 zeta=%d alpha=%.1f: relF f16 %.3e f32 %.3e" % (zeta, alpha, r16, r32))
        assert r32 <= 1e-5 and r16 <= 5e-2, (zeta, alpha, r16, r32)
        del A


# ------------------------------------------------------------------------------------ geometry sweep
def _geometry_cases():
    rng = np.random.default_rng(20260611)
    cases = []
    for n in (64, 128, 192, 256, 384, 512, 1024):   # 192, 384: three column slices; sketches beyond TMEM are skipped
        for zeta in (1, 2, 4, 8):
            for d_over_zeta in (8, 32, 64, 128, 256, 512):
                cases.append((int(rng.integers(600, 2600)), n, zeta * d_over_zeta, zeta))
    idx = rng.permutation(len(cases))[:72]
    return [cases[i] for i in sorted(idx)]


@pytest.mark.parametrize("m,n,d,zeta", _geometry_cases())
def test_tmem_geometry_sweep(ss, m, n, d, zeta):
    # every geometry the tensor-memory kernel can take (X, S, bucket groups, column slices, chained / deferral groups,
    # 16- to 128-row stages), forced, against the oracle: bit-exact where the arithmetic is exact in any order
    # (zeta in {1, 4}), within 2e-3 of FP64 where the scale is irrational (zeta in {2, 8}; L <= 64 terms)
    seed = sketch_seed(7000 + m + d)
    sk = ss.Sketch(m, d, zeta, seed)
    exact = zeta in (1, 4)
    A = wl.integer_valued(m, n, m) if exact else wl.gaussian(m, n, m)
    got = apply16(ss, sk, dev(A), "tmem")
    want = oracle.f64_sketch(seed, d, zeta, A)
    if exact:
        assert np.array_equal(oracle.half_bits_to_f64(bits(got)), want)
    else:
        assert ev.rel_fro(oracle.half_bits_to_f64(bits(got)), want) <= 2e-3


# bucket-group geometries under every group mode (sketch_opts_t::tmem_group_mode): chained, deferral with groups of 4 / 8
# rows.  Small d / zeta makes rows of one group collide often, which is what the chains and the deferral lists exist for.
@pytest.mark.parametrize("mode", [1, 2, 3])
@pytest.mark.parametrize("m,n,d,zeta", [
    (5003, 256, 256, 4),      # X = 4, two bucket groups of two blocks, d / zeta = 64: a clash in most groups
    (4999, 256, 1024, 4),     # c4's geometry: X = 2, four bucket groups, two column slices
    (6007, 256, 2048, 4),     # c4-2048's: X = 1, 128-row stages, four column slices
    (2203, 1024, 2048, 4),    # e1's: sixteen column slices
    (5501, 256, 512, 8),      # zeta = 8: four bucket groups of two blocks, d / zeta = 64
    (7001, 128, 384, 4),      # d / zeta = 96: groups of 8 allowed (>= 72)
    (3301, 512, 1024, 2),     # two bucket groups of one block
])
def test_tmem_group_modes(ss, m, n, d, zeta, mode):
    seed = sketch_seed(7100 + m)
    sk = ss.Sketch(m, d, zeta, seed)
    try:
        sk.plan(n, variant=VID["tmem"], tmem_group_mode=mode)
    except ss.SketchError:
        pytest.skip("plan: no tensor-memory geometry for n=%d d=%d zeta=%d" % (n, d, zeta))
    exact = zeta in (1, 4)
    A = wl.integer_valued(m, n, m) if exact else wl.gaussian(m, n, m)
    Ad = dev(A)
    want = oracle.f64_sketch(seed, d, zeta, A)
    for grid in (0, 3 * 16):        # the full grid, and a few CTAs with many stages each
        got = sk.apply_f16acc(Ad, variant=VID["tmem"], tmem_group_mode=mode, grid_ctas=grid)
        if exact:
            assert np.array_equal(oracle.half_bits_to_f64(bits(got)), want), (mode, grid)
        else:
            assert ev.rel_fro(oracle.half_bits_to_f64(bits(got)), want) <= 2e-3, (mode, grid)


def test_stream_probe_reads_and_returns(ss):
    # step a2 in isolation (sketch_stream_probe): both kinds run to completion on a buffer with a ragged tail and on an
    # empty one, leave the data untouched, and report the bytes they read
    x = torch.arange(3 * (1 << 20) + 100, dtype=torch.float32, device="cuda")
    ref = x.clone()
    assert ss.sketch_stream_probe(x, 0) == x.numel() * 4 // 32 * 32
    assert ss.sketch_stream_probe(x, 1) == x.numel() * 4 // 32768 * 32768
    assert ss.sketch_stream_probe(x[:4096], 1, grid_ctas=7) == 4096 * 4 // 32768 * 32768 == 0
    torch.cuda.synchronize()
    assert torch.equal(x, ref)


# small sketches (a quarter of a warp's tensor-memory region or less): AUTO's replicated-rows mode -- every row of a group adds
# into its own private copy, the copies are summed at the flush -- against the chained groups (tmem_group_mode = 1) and the oracle
@pytest.mark.parametrize("m,n,d,zeta", [
    (9001, 64, 128, 4),       # c2's geometry: X = 1, four copies of a 128-row partial
    (6011, 64, 64, 8),        # zeta = 8: two copies
    (7013, 128, 64, 2),       # X = 2, one feature slice
    (5003, 256, 32, 1),       # X = 1, four feature slices (column offsets relative to the warp's region)
])
def test_tmem_replicated_rows(ss, m, n, d, zeta):
    seed = sketch_seed(7200 + m)
    sk = ss.Sketch(m, d, zeta, seed)
    exact = zeta in (1, 4)
    A = wl.integer_valued(m, n, m) if exact else wl.gaussian(m, n, m)
    Ad = dev(A)
    want = oracle.f64_sketch(seed, d, zeta, A)
    # irrational scale: the north star's rule against the sequential-FP16 oracle (L = m zeta / d is up to 750 terms here)
    tol16 = None if exact else 1.5 * ev.rel_fro(oracle.half_bits_to_f64(oracle.seq16_sketch(seed, d, zeta, A)), want)
    for mode in (0, 1):
        for grid in (0, 5):
            got16 = sk.apply_f16acc(Ad, variant=VID["tmem"], tmem_group_mode=mode, grid_ctas=grid)
            got32 = sk.apply_f32acc(Ad, variant=VID["tmem"], tmem_group_mode=mode, grid_ctas=grid)
            if exact:
                assert np.array_equal(oracle.half_bits_to_f64(bits(got16)), want), (mode, grid)
                assert np.array_equal(got32.cpu().numpy().astype(np.float64), want), (mode, grid)
            else:
                assert ev.rel_fro(oracle.half_bits_to_f64(bits(got16)), want) <= tol16, (mode, grid)
                assert ev.rel_fro(got32.cpu().numpy(), want) <= 1e-5, (mode, grid)
