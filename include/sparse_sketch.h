/* sparse_sketch.h -- C ABI of the B200 (sm_100a) sparse-sketch library.
 *
 * The library forms B = S*A for a tall FP32 row-major matrix A (m x n, m >> n)
 * under CountSketch (zeta = 1) and SparseStack (zeta stacked CountSketch blocks
 * of d/zeta rows each, entries +-1/sqrt(zeta)):
 *     PAPER.md:59-65, Eq. (1)  (arxiv 2606.20195, Sec. II-A).
 * The bucket / sign map is the counter hash fixed by BASELINE.json:north_star
 * (instantiating PAPER.md:59; readings R1-R4 in DESIGN.md):
 *     h       = splitmix64(seed ^ (i*zeta + j))        i = global row, j = block, 0-based
 *     bucket  = j*(d/zeta) + (((h >> 32) * (d/zeta)) >> 32)
 *     signbit = h & 1                                   0 -> +1, 1 -> -1
 *
 * Conventions for every entry point
 *   - returns SKETCH_OK (0) or a negative SKETCH_ERR_* code; never throws, never aborts;
 *   - "dev" pointers are CUDA device pointers on the current device, "host" pointers are
 *     host memory; the caller owns every buffer and the stream it passes; the library owns
 *     the handle, its scratch (replicated partial sketches, optional packed hash array,
 *     staging buffers) and frees them in sketch_destroy;
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  apply/dump calls
 *     are asynchronous on that stream and never synchronise, except a call that has to grow a
 *     scratch buffer (cudaMalloc; the first call of a shape, outside any capture) and the *_host
 *     entry points (which return after the result is in host memory);
 *   - A is never modified; one handle may be applied to any number of matrices with any n
 *     (S is d x m, independent of n), e.g. A in FP16 and b in FP32 with the same map as in
 *     PAPER.md:356 / Table I.
 *   - a handle must not be used from two host threads at once.
 *   - CUDA graphs (stream capture).  Every device-buffer apply can be captured, with two rules.  (1) Nothing is allocated
 *     inside a capture: if the call would have to create or grow a library-owned scratch buffer (the partial sketches of
 *     the FLAT / GENERIC variants with replicas > 1, those of a fused right-hand side, the packed hash array of the SMEM
 *     variant / hash_mode 2) it fails with SKETCH_ERR_CAPTURE and enqueues nothing that uses it -- run the same apply once
 *     outside the capture first (the *_noalloc entry point and the TMEM / SMALL variants without a right-hand side use
 *     none).  (2) The graph holds the scratch pointers it was captured with.  The library keeps such a buffer alive until
 *     sketch_destroy even when a later call needs a larger one (it then allocates a second buffer), so a replay never
 *     touches freed memory; but the stream ordering the library provides between applies on different streams does not
 *     extend to replays, which go through no library call: order every replay against other work on the same handle
 *     yourself (one stream, or events), or give each graph a handle of its own.  Destroy the graph before the handle.
 */
#ifndef SPARSE_SKETCH_H_
#define SPARSE_SKETCH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sketch sketch_t; /* opaque, library-owned */

/* error codes */
#define SKETCH_OK 0
#define SKETCH_ERR_INVALID (-1)     /* m<=0, d<=0, zeta<1, n<=0, rows<0, row range outside [0,m), bad enum */
#define SKETCH_ERR_NULL (-2)        /* a required pointer is NULL */
#define SKETCH_ERR_DIVISIBILITY (-3)/* d % zeta != 0 ("Let d be divisible by zeta") */
#define SKETCH_ERR_LDA (-4)         /* lda < n */
#define SKETCH_ERR_ALIGNMENT (-5)   /* A or B not 4-byte aligned (the 16-bit sketches too: their REDs work on 4-byte words) */
#define SKETCH_ERR_UNSUPPORTED (-6) /* the forced variant cannot run this shape (AUTO never returns it) */
#define SKETCH_ERR_CUDA (-7)        /* CUDA runtime error; text via sketch_last_error() */
#define SKETCH_ERR_NOMEM (-8)       /* host or device allocation failed */
#define SKETCH_ERR_CAPTURE (-10)    /* a library-owned scratch buffer would have to be created or grown inside a stream
                                       capture (see "CUDA graphs" above); text in sketch_last_error() */
#define SKETCH_ERR_SCRATCH_LIMIT (-9) /* sketch_apply_f16acc_noalloc only: two partial sketches of this d x n do not fit
                                         the built-in scratch (SKETCH_NOALLOC_SCRATCH_BYTES); sizes in sketch_last_error() */

/* conversion rule of the FP16 path (Sec. III-D) */
#define SKETCH_RN 0 /* round-to-nearest-even, __float2half semantics */
#define SKETCH_SR 1 /* stochastic conversion with counter-based bits (readings R13, R14) */
#define SKETCH_DITHER 2 /* dither conversion, Eq. (6): RN16(q + (u0 - 1/2) c q), c = 0.00097656f, u0 a 24-bit variate,
                           every operation one FP32 rounding (readings R20, R21) */

/* kernel variants (all compute the same sums; they differ in where partial sums live) */
#define SKETCH_VARIANT_AUTO 0      /* chosen per shape from measurement */
#define SKETCH_VARIANT_FLAT_PAIR 1 /* paper's Listing 1/2 restated: one column (f32) / column pair (f16) per
                                      lane, one result-discarding RED per contribution */
#define SKETCH_VARIANT_FLAT_VEC 2  /* widest vector RED the shape allows (16-byte REDG: 8 halves / 4 floats) */
#define SKETCH_VARIANT_SMEM 3      /* shared-memory-privatised partial sketch per CTA, flushed with vector RED */
#define SKETCH_VARIANT_GENERIC 4   /* any n / any alignment scalar fallback (one lane per element) */
#define SKETCH_VARIANT_TMEM 5      /* tensor-memory-privatised partial sketch per warp (tcgen05.ld / tcgen05.st read-
                                      modify-write), A staged by TMA, hashes computed on the fly by a producer
                                      warp; every accumulation mode (FP16 RN / SR / dither, bfloat16, FP32);
                                      zeta in {1,2,4,8}, n = 32*FW*X*S*CS with FW = 2 features per 32-bit word for
                                      the 16-bit sketches and 1 for FP32, X, S in {1,2,4}, CS in 1..16,
                                      BQ in {1,2,4} bucket groups dividing zeta (SR / dither: BQ = 1), S*BQ <= 4 and
                                      (d/BQ)*X <= 512 (e.g. FP16 n = 256: d <= 2048), lda % 4 == 0,
                                      A and B 16-byte aligned, rows < 2^31 when lda != n / CS (2-D tensor-map
                                      coordinates).
                                      Overflow signature: partial sums live per warp and meet at the flush, so a
                                      sketch entry whose partials overflowed to +inf in one warp and -inf in
                                      another comes back NaN, where one running sum (FLAT with replicas = 1, or
                                      the sequential order) sticks at +-inf.  Both are legal orders (reading R9);
                                      count non-finite entries, not infinities, when comparing with PAPER.md:394 */
#define SKETCH_VARIANT_SMALL 6     /* per-warp shared-memory partial sketches for small inputs and narrow matrices:
                                      FP16-RN, zeta in {1,2,4,8}, n and lda even, A 8-byte aligned,
                                      8*d*n*2 bytes of shared memory (AUTO picks it for launch-bound inputs) */

typedef struct sketch_opts {
  int32_t variant;    /* SKETCH_VARIANT_* */
  int32_t replicas;   /* FLAT variants: number P of L2-resident partial sketches the CTAs are spread over,
                         summed by a reduce kernel (0 = auto: as many as 16 MiB of scratch and 1/8 of A's bytes hold, at
                         most 256 -- a two-level sum, which is what keeps a flat FP16 scatter accurate; 1 = RED straight
                         into B) */
  int32_t hash_mode;  /* 0 = auto, 1 = hash on the fly inside the scatter kernel, 2 = read the packed array
                         built by sketch_precompute_hashes (built on demand) */
  int32_t accumulate; /* 0 = complete sketch: B is zero-initialised by the call;
                         1 = add this row range's contributions into the existing B */
  int64_t row_begin;  /* global index of the first row stored at A (rows are hashed by global index) */
  int64_t rows;       /* number of rows at A; 0 = m - row_begin */
  int32_t grid_ctas;  /* 0 = auto; tuning / tests only */
  int32_t tmem_group_mode; /* 0 = auto; tuning / tests only, TMEM variant: 1 = chained groups (every geometry), 2 / 3 =
                              deferral with groups of 4 / 8 rows (bucket-group geometries; ignored where the geometry has
                              no such mode).  AUTO also has replicated rows for sketches a quarter of a warp's
                              tensor-memory region or smaller */
} sketch_opts_t;

/* ---- handle ------------------------------------------------------------------------------- */

/* Create the sketch S in R^{d x m} with zeta nonzeros per column.
 * m: rows of the matrices it will be applied to; d: sketch rows, d % zeta == 0; seed: full 64 bits
 * (use full-width seeds: seeds that differ only in low bits alias, R15).
 * *out receives the handle.  No device memory is allocated here. */
int sketch_create(int64_t m, int32_t d, int32_t zeta, uint64_t seed, sketch_t** out);

/* Free the handle and all library-owned device/host scratch.  NULL is accepted. */
int sketch_destroy(sketch_t* s);

/* ---- hash stage ------------------------------------------------------------- */

/* Write bucket[i*zeta + j] (int32, in [j*d/zeta, (j+1)*d/zeta)) and signbit[i*zeta + j] (uint8, the raw
 * h & 1) for all i in [0,m), j in [0,zeta) to DEVICE buffers of m*zeta elements each. */
int sketch_hashes_dump(const sketch_t* s, int32_t* bucket_dev, uint8_t* signbit_dev, void* stream);

/* Build (once) the packed per-(row,block) hash array the hash_mode=2 kernels read; m*zeta entries, library-owned:
 * uint16 = bucket | reload<<14 | signbit<<15 in the sub-step order of the SMEM variant (entry (row, t) at row*zeta + t holds
 * block (row mod R + t) mod zeta, R = min(zeta, 4)) when zeta is 1, 2, 4 or 8 and d <= 2047, else uint32 = bucket | signbit<<31
 * at row*zeta + j.  Counted in "complete sketch" time by bench.py when that mode is used.  Not inside a stream
 * capture (SKETCH_ERR_CAPTURE): the handle would count the array as built while the graph has yet to run. */
int sketch_precompute_hashes(sketch_t* s, void* stream);

/* ---- scatter kernels ------------------------------------------------- */

/* FP32-accumulate baseline (Listing 1; Table I "FP32 path").
 * A_dev: m x n FP32 row-major with leading dimension lda >= n (elements); B_dev: d x n FP32 row-major
 * (leading dimension n), overwritten with S*A.  Products and sums are FP32; the global RED used for
 * FP32 flushes FP32 subnormals (SASS REDG.E.ADD.F32.FTZ). */
int sketch_apply_f32acc(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, float* B_dev,
                        void* stream);

/* FP16-accumulate path (PAPER.md:114-136, Listing 2; :140-165; :175-187): per contribution
 * p = fp32(+-s * a), v = RN16(p) (or SR16), B16[bucket, c] = RN16(B16[bucket, c] + v), each FP16 component
 * independently, subnormals kept (.noftz), overflow -> +-inf.  The order of the additions is unspecified
 * ("Parallel atomic updates may also realize different orders").
 * B_dev: d x n IEEE binary16 row-major, overwritten.  rounding: SKETCH_RN / SKETCH_SR / SKETCH_DITHER; sr_seed is
 * used by SR and dither only.  Any n >= 1 is accepted (odd n runs the scalar GENERIC variant). */
int sketch_apply_f16acc(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev,
                        int rounding, uint64_t sr_seed, void* stream);

/* bfloat16-accumulate control (PAPER.md:382 Fig. 7, :396 "BF16 ... wider range"): the FP16 path with bfloat16 in
 * place of binary16 -- p = fp32(+-s * a), v = RN_bf16(p), B[bucket, c] = RN_bf16(B[bucket, c] + v), subnormals kept.
 * B_dev: d x n bfloat16 row-major, overwritten.  RN conversion only. */
int sketch_apply_bf16acc(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev, void* stream);

/* Same, with explicit options (variant override, row range, accumulate-into-B).  opts == NULL means
 * all-zero options, i.e. exactly the calls above. */
int sketch_apply_f32acc_ex(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, float* B_dev,
                           const sketch_opts_t* opts, void* stream);
int sketch_apply_f16acc_ex(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev,
                           int rounding, uint64_t sr_seed, const sketch_opts_t* opts, void* stream);

int sketch_apply_bf16acc_ex(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev,
                            const sketch_opts_t* opts, void* stream);

/* ---- for callers that must not allocate device memory ---------------------------------------- */

/* Size of the scratch array built into the library's device image.  Every GPU on which the library's module is loaded
 * holds this much for as long as the process lives, whether or not the entry point below is ever called. */
#define SKETCH_NOALLOC_SCRATCH_BYTES (8u << 20) /* 8 MiB */

/* sketch_apply_f16acc for programs that cannot call cudaMalloc while they run.
 *
 * Who that is: an application that gave all device memory to its own pool at start-up (nothing is left for us to
 * allocate, and going around its pool defeats its accounting); a latency-bound or certified pipeline whose device memory
 * map is frozen after initialisation (cudaMalloc / cudaFree synchronise the whole device, and an allocation that can fail
 * in steady state is not acceptable there); a plug-in running inside a host program that forbids allocation in its
 * callbacks.  Every other apply in this header may grow a library-owned buffer on some call; this one never does: it
 * calls no cudaMalloc, no cudaFree and no routine that allocates on its behalf.
 *
 * What it computes: the complete FP16-accumulate sketch B = S*A of all m rows (Listing 2), exactly as
 * sketch_apply_f16acc_ex does with variant = SKETCH_VARIANT_FLAT_VEC (SKETCH_VARIANT_GENERIC where n, lda or the
 * alignment rule out vector REDs) and several L2-resident partial sketches: the same kernels, the same conversions
 * (rounding = SKETCH_RN / SKETCH_SR / SKETCH_DITHER, sr_seed as there) and the same FP16 RN adds; only the home of the
 * partial sketches differs -- a fixed array inside the library instead of a buffer from cudaMalloc.  It is not the
 * fastest path for shapes the tensor-memory kernel takes (that kernel needs no scratch either: plain sketch_apply_f16acc
 * already allocates nothing for those shapes as long as no right-hand side is fused).
 * A_dev, B_dev, lda, stream: as for sketch_apply_f16acc; the caller passes (and owns) input and output as usual.
 *
 * Limit: two partial sketches must fit the array, i.e. 2 * roundup8(d * n) * 2 bytes <= SKETCH_NOALLOC_SCRATCH_BYTES
 * (d * n <= 2 097 152, e.g. d = 2048 at n = 1024).  Larger sketches are refused with SKETCH_ERR_SCRATCH_LIMIT before
 * anything is enqueued; sketch_last_error() then carries the sizes.  Within the limit it uses as many partial sketches
 * as fit, at most 256.
 *
 * First call on a device: looks up the array's device address (cudaGetSymbolAddress, with that device current; this
 * can make the CUDA runtime load the library's module there) and caches it per device ordinal (ordinals 0..63).  Make that
 * first call during your own initialisation, on every device you will use, and before any stream capture begins.
 *
 * Sharing: there is ONE array per device, shared by every handle, stream and host thread of the process, and it keeps
 * whatever the previous call left in it.  Each call zeroes the part it is about to use, on `stream`, before its kernels.
 * Two calls whose GPU work can overlap (different streams without an ordering between them, or two host threads) add
 * into the same partial sketches and both results are garbage: order such calls yourself (same stream, or an event). */
int sketch_apply_f16acc_noalloc(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev, int rounding,
                                uint64_t sr_seed, void* stream);

/* ---- least-squares front end (PAPER.md:356 Sec. V-D; :312) ---------------------------------- */

/* One pass over the rows for [A | b]: "We sketch A in the chosen precision and b in FP32 with the same map"
 * (PAPER.md:356).  A as sketch_apply_f16acc (RN) / sketch_apply_f32acc; b_dev: FP32 vector, element k = the right-hand
 * side of row (row_begin + k); Sb32_dev: d FP32 values, overwritten with S*b (or added to, with opts->accumulate):
 * Sb[bucket(i, j)] += fp32(+-s * b_i), FP32 products and sums in unspecified order, same map as A.
 * Where the tensor-memory variant runs, the lanes that hash a row also add its b contributions (no second pass,
 * no second hash); other variants run a one-column FP32 scatter behind the first.  opts may be NULL. */
int sketch_apply_f16acc_with_rhs(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, const float* b_dev,
                                 void* B16_dev, float* Sb32_dev, const sketch_opts_t* opts, void* stream);
int sketch_apply_f32acc_with_rhs(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, const float* b_dev,
                                 float* B32_dev, float* Sb32_dev, const sketch_opts_t* opts, void* stream);

/* "widen FP16 SA exactly" ("layout/promotion"): out_dev[k] = fp32(B16_dev[k]) for k < count, exact for
 * every binary16 (is_bf16 = 0) or bfloat16 (is_bf16 = 1) value.  Device pointers; asynchronous on `stream`. */
int sketch_widen(const void* B16_dev, int64_t count, int is_bf16, float* out_dev, void* stream);

/* End-to-end entry points with HOST buffers: A_host (m x n, lda) is streamed to the device in row chunks
 * through two library-owned staging buffers (copy of chunk k+1 overlaps the kernels of chunk k), sketched
 * with the kernels above (row_begin / accumulate), and B_host (d x n) is written before the call returns.
 * Pinned (page-locked) host memory is needed for the copies to overlap; pageable memory works, slower. */
int sketch_apply_f32acc_host(const sketch_t* s, const float* A_host, int32_t n, int64_t lda,
                             float* B_host, const sketch_opts_t* opts);
int sketch_apply_f16acc_host(const sketch_t* s, const float* A_host, int32_t n, int64_t lda, void* B_host,
                             int rounding, uint64_t sr_seed, const sketch_opts_t* opts);

/* ---- measurement support ------------------------------------------------------------------- */

/* L2 atomic-throughput probe (the second term of the roofline): issues `iters` rounds of
 * result-discarding REDs with the scatter kernels' address pattern (a random bucket row per lane group,
 * consecutive lanes on consecutive columns of a d x n sketch) from register values, with no A loads.
 * kind: 0 = f16x2 (4 B), 1 = v2.f16x2 (8 B), 2 = v4.f16x2 (16 B), 3 = f32 (4 B), 4 = v2.f32, 5 = v4.f32.
 * Candidates for sketches beyond tensor memory, same pattern: 6 = plain (non-atomic) L2 read-modify-write of 16 bytes
 * per lane (ld.global.cg / HADD2 / st.global.cg; hazards ignored: an upper bound); 7 / 8 = TMA bulk reduction
 * (cp.reduce.async.bulk ... add.noftz.f16 / add.f32) of min(row, 2 KiB) bytes from shared memory per warp and round,
 * counted in 16-byte units (n * elem % 16 == 0 required).
 * sketch_dev: scratch of replicas*d*n*elem bytes.  Asynchronous on `stream`; time it with CUDA events.
 * *red_ops_out (host, may be NULL) receives the number of lane-level RED operations issued. */
int sketch_red_probe(void* sketch_dev, int32_t d, int32_t n, int32_t kind, int32_t replicas,
                     int32_t grid_ctas, int32_t iters, uint64_t* red_ops_out, void* stream);

/* Read-only streaming probe (step a2 in isolation): reads `bytes` (multiple of 32 KiB is read in full; a tail is skipped)
 * from src_dev once and discards them -- kind 0: 256-bit no-allocate / evict-first loads, grid-stride over grid_ctas CTAs of
 * 256 threads; kind 1: TMA bulk copies of 32 KiB into a 4-slot shared-memory ring per CTA (k_tmem's producer with the
 * consumers removed; use one CTA per SM).  Time it with CUDA events: bytes / time is the rate at which this GPU delivers a
 * buffer that is read and never written, the ceiling of any complete sketch; bench.py prints it beside the COPY rate of
 * MEASURED_PEAKS.json that roofline.frac is quoted against.  src_dev 32-byte aligned; sink_dev: 8 device bytes or NULL
 * (never written in practice).  Asynchronous on `stream`. */
int sketch_stream_probe(const void* src_dev, int64_t bytes, int32_t kind, int32_t grid_ctas, void* sink_dev, void* stream);

/* The conversion step in isolation, for tests: out_dev[k] (16-bit pattern) = conversion of p_dev[k] under
 * kind with the random bits rbits_dev[k]:  0 = RN16;  1 = SR16, reading R13 with r24 = rbits & 0xFFFFFF
 * (PAPER.md:203-207);  2 = dither, Eq. (6), same r24;  3 = bfloat16 RN;  4 / 5 = the hardware
 * cvt.rs.f16x2.f32 d, a, b, rbits with p in both sources: the half converted from b / from a;  6 / 7 = the library's SR pair
 * conversion with p and r24 in both halves (low / high half).  The two agree on the FP16 normal grid [2^-14, 65504) under a
 * fixed bit mapping and differ below 2^-14 (tests/test_gpu_modes.py, R22), so the library's SR kernels use the
 * hardware instruction exactly where both values of a pair lie on that grid and the integer rule 1 everywhere else.  Shown
 * by test, not proved: kinds 6 / 7 equal kind 1 on 2^30 random samples (tests/test_gpu_modes.py) and equal the oracle's
 * SR16 on 2^26 random samples plus every FP32 value in windows around 2^-14, 65504, 65520, 2^-24 and 2^-25
 * (tests/test_gpu_add_paths.py).  rbits_dev may be NULL for kinds 0 and 3.  Device pointers. */
int sketch_convert_probe(const float* p_dev, const uint32_t* rbits_dev, int64_t count, int32_t kind, uint16_t* out_dev,
                         void* stream);

/* Which variant / replica count / hash mode AUTO resolves to for this shape; host-only, no launch.
 * is_f16: 0 = f32acc, 1 = f16acc, 2 = bf16acc.  Any out pointer may be NULL. */
int sketch_plan(const sketch_t* s, int32_t n, int64_t lda, int is_f16, int rounding, const sketch_opts_t* opts,
                int32_t* variant_out, int32_t* replicas_out, int32_t* hash_mode_out, int32_t* grid_out);

/* Number of kernels this library has launched since load (for bench.py's `gpu_launches`). */
uint64_t sketch_launch_count(void);

/* Static text for a SKETCH_ERR_* code; and the text of the last CUDA error seen by this thread. */
const char* sketch_strerror(int code);
const char* sketch_last_error(void);

/* "sparse_sketch <major>.<minor> sm_100a" */
const char* sketch_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPARSE_SKETCH_H_ */
