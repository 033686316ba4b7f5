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


def apply16(ss, sk, A, variant="auto", **kw):
    try:
        return sk.apply_f16acc(A, variant=VID[variant], **kw)
    except ss.SketchError as e:
        if e.code == -6:
            pytest.skip("variant %s does not support this shape" % variant)
        raise


def apply32(ss, sk, A, variant="auto", **kw):
    try:
        return sk.apply_f32acc(A, variant=VID[variant], **kw)
    except ss.SketchError as e:
        if e.code == -6:
            pytest.skip("variant %s does not support this shape" % variant)
        raise


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
    for variant in F16_VARIANTS:
        try:
            got = sk.apply_f16acc(dev(A), variant=VID[variant])
        except ss.SketchError as e:
            assert e.code == -6
            continue
        r = ev.rel_fro(oracle.half_bits_to_f64(bits(got)), B)
        assert r <= 1.5 * ref and r <= 5e-2, (variant, r, ref)


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
    for variant in F16_VARIANTS:
        try:
            got = sk.apply_f16acc(dev(A), variant=VID[variant])
        except ss.SketchError as e:
            assert e.code == -6
            continue
        r = ev.rel_fro(oracle.half_bits_to_f64(bits(got)), B)
        assert r <= 1.5 * ref and r <= 5e-2, (variant, r, ref)
        assert r > 0.02 * ref      # it really is an FP16 accumulation, not a widened one


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
    c = sorted({0, 1, 62, 63, 64, 65, n // 2 - 1, n // 2, n - 2, n - 1})
    return [x for x in c if 0 <= x < n]


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
