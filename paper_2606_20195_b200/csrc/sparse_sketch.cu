// sparse_sketch.cu -- C ABI (include/sparse_sketch.h), handle, variant selection and launches.
// Host logic only; every step of the hot path runs in the kernels of kernel_*.cuh (launched via launch.h).
#include "../../include/sparse_sketch.h"

#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "kernel_misc.cuh"
#include "launch.h"

namespace {

std::atomic<uint64_t> g_launches{0};
thread_local char g_last_error[512] = "";

int cuda_fail(cudaError_t e, const char* what) {
  snprintf(g_last_error, sizeof(g_last_error), "%s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
  return SKETCH_ERR_CUDA;
}
#define CU_TRY(call)                                      \
  do {                                                    \
    cudaError_t _e = (call);                              \
    if (_e != cudaSuccess) return cuda_fail(_e, #call);   \
  } while (0)

inline int launch_check(const char* what) {
  g_launches.fetch_add(1, std::memory_order_relaxed);
  cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? SKETCH_OK : cuda_fail(e, what);
}

}  // namespace

struct sketch {
  int64_t m;
  int32_t d, zeta;
  uint32_t db;
  uint64_t seed;
  float scale;
  // device properties (filled lazily on first device use)
  int dev_ready;
  int sm_count;
  int smem_optin;    // max dynamic smem per block
  int smem_per_sm;
  // library-owned scratch
  void* rep;  size_t rep_bytes;        // replicated partial sketches
  void* sbrep; size_t sbrep_bytes;     // replicated FP32 sketches of a fused right-hand side
  void* packed; size_t packed_bytes; int packed_width;  // 0 = none, 2 = 16-bit entries in sub-step order, 4 = plain 32-bit
  void* stage[2]; size_t stage_bytes;  // host-path staging
  void* bdev; size_t bdev_bytes;
  cudaStream_t st_copy, st_comp;
  cudaEvent_t ev_copied[2], ev_done[2];
  int host_ready;
  // stream ordering of the library-owned scratch (rep, packed): the last stream that used it and an event recorded
  // behind that use; an apply on another stream waits for the event first
  cudaStream_t scratch_stream;
  cudaEvent_t ev_scratch;
  int scratch_busy;   // 0 = never used, 1 = ev_scratch is valid
  // stream capture: a captured apply bakes the scratch pointers into its graph, so a buffer a capture has used is pinned --
  // when a later call needs a larger one, the old buffer is retired (kept until sketch_destroy), never freed under the graph
  int rep_pinned, sbrep_pinned, packed_pinned;
  struct Retired {
    void* buf;
    Retired* next;
  }* retired;
  // tensor maps of the strided / column-sliced tensor-memory launches, keyed by what they encode (a handle is applied
  // to the same few matrices over and over: the hot call then does no encoding)
  struct TmapSlot {
    const float* A;
    int64_t lda, rows;
    int32_t n, n_cta, box_rows;
    CUtensorMap map;
  } tmaps[8];
  int tmap_count, tmap_next;
};

namespace {

struct Plan {
  int variant, vec, replicas, hash_mode, grid, wpc, zeta_t;
  size_t smem_bytes;
  int64_t rows_per_cta;
  int64_t rows_main;  // smem variant: rows handled by k_smem (multiple of its ring rows); the rest go to k_flat
  sk::TmemShape tm;   // tmem variant: geometry
  int tm_mode;        // tmem variant: TM_* accumulation mode
};

// tensor-memory accumulation mode of (sketch element type, conversion rule)
inline int tmem_mode_of(int out, int rounding) {
  return out == sk::OUT_F32 ? sk::TM_F32 : out == sk::OUT_BF16 ? sk::TM_BF16
       : rounding == SKETCH_SR ? sk::TM_F16_SR : rounding == SKETCH_DITHER ? sk::TM_F16_DITHER : sk::TM_F16;
}

int ensure_device(sketch* s) {
  if (s->dev_ready) return SKETCH_OK;
  int dev = 0;
  CU_TRY(cudaGetDevice(&dev));
  CU_TRY(cudaDeviceGetAttribute(&s->sm_count, cudaDevAttrMultiProcessorCount, dev));
  CU_TRY(cudaDeviceGetAttribute(&s->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  CU_TRY(cudaDeviceGetAttribute(&s->smem_per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
  s->dev_ready = 1;
  return SKETCH_OK;
}

// Grow a library-owned buffer to `want` bytes.  Inside a stream capture nothing may be allocated or freed: a buffer that
// is large enough is marked pinned (the graph now refers to it), one that is not makes the call fail with
// SKETCH_ERR_CAPTURE.  Outside a capture a pinned buffer that must grow is retired instead of freed.
int ensure_scratch(sketch* s, void** buf, size_t* have, size_t want, bool capturing = false, int* pinned = nullptr) {
  if (*have >= want) {
    if (capturing && pinned) *pinned = 1;
    return SKETCH_OK;
  }
  if (capturing) {
    snprintf(g_last_error, sizeof(g_last_error),
             "a library-owned scratch buffer would have to grow from %zu to %zu bytes inside a stream capture; run the same "
             "apply once outside the capture first", *have, want);
    return SKETCH_ERR_CAPTURE;
  }
  if (*buf) {
    if (pinned && *pinned) {
      sketch::Retired* r = new (std::nothrow) sketch::Retired;
      if (!r) return SKETCH_ERR_NOMEM;
      r->buf = *buf;
      r->next = s->retired;
      s->retired = r;
      *pinned = 0;
    } else {
      CU_TRY(cudaFree(*buf));
    }
    *buf = nullptr;
    *have = 0;
  }
  cudaError_t e = cudaMalloc(buf, want);
  if (e == cudaErrorMemoryAllocation) {
    cudaGetLastError();
    return SKETCH_ERR_NOMEM;
  }
  if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc(scratch)");
  *have = want;
  return SKETCH_OK;
}

// Grid cap of the grid-stride helper kernels that take no handle (widen, conversion probe): 16 CTAs per SM of the
// current device, the SM count asked once per device ordinal.
int grid_cap_current_device() {
  static std::atomic<int> sms[64];
  int dev = 0, n = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 1024;
  n = sms[dev].load(std::memory_order_relaxed);
  if (n == 0) {
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return 1024;
    sms[dev].store(n, std::memory_order_relaxed);
  }
  return n * 16;
}

inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }
inline bool zeta_templated(int z) { return z == 1 || z == 2 || z == 4 || z == 8; }
inline bool rot_ok(const sketch* s) { return zeta_templated(s->zeta) && s->d <= sk::smem_max_bucket(); }

bool smem_feasible(const sketch* s, int n, int64_t lda, const void* A, const void* B, size_t* bytes) {
  if (!rot_ok(s)) return false;
  if (n % 64 != 0 || n / 64 > 16) return false;
  const int vec = 2 * sk::smem_step_rows(s->zeta);  // columns per lane: 8 / 4 / 2
  if (lda % vec != 0 || !aligned(A, 4 * (size_t)vec) || !aligned(B, 16)) return false;
  size_t b = ((size_t)s->d + 1) * n * 2;  // partial sketch + the dummy row d
  if (b > (size_t)s->smem_optin) return false;
  *bytes = b;
  return true;
}

bool tmem_feasible(const sketch* s, int n, int64_t lda, int64_t rows, const void* A, const void* B, int gm_force, int mode,
                   sk::TmemShape* h) {
  if (!zeta_templated(s->zeta)) return false;
  if (!sk::tmem_shape(n, s->d, s->zeta, lda, gm_force, mode, h)) return false;
  if (lda % 4 != 0 || !aligned(A, 16) || !aligned(B, 16)) return false;  // TMA bulk copies: 16-byte granules
  if (lda != n / h->CS && !sk::tmem_tensor_map_ok(lda, rows, n / h->CS)) return false;   // the 2-D tensor-map path
  return sk::tmem_smem_bytes_for(s->zeta, n / h->CS, h->BQ, h->GM, mode) <= (size_t)s->smem_optin;
}

int flat_vec_for(bool f16 /* a 16-bit sketch */, int n, int64_t lda, const void* A, const void* B, int want_max) {
  const int cands_h[3] = {8, 4, 2};
  const int cands_f[4] = {4, 2, 1, 0};  // FP32: one 16-byte RED per lane is the widest single transaction
  const int* c = f16 ? cands_h : cands_f;
  int nc = f16 ? 3 : 3;
  for (int k = 0; k < nc; ++k) {
    int v = c[k];
    if (v > want_max) continue;
    size_t eb = f16 ? 2 : 4;
    if (n % v == 0 && lda % v == 0 && aligned(A, 4 * (size_t)v) && aligned(B, eb * v)) return v;
  }
  return 0;
}

int make_plan(sketch* s, int n, int64_t lda, const void* A, const void* B, int out, int rounding,
              const sketch_opts_t* o, int64_t rows, Plan* p) {
  const bool f16 = out != sk::OUT_F32;                              // a 16-bit sketch
  const bool h16rn = out == sk::OUT_F16 && rounding == SKETCH_RN;   // the FP16-RN hot path
  int rc = ensure_device(s);
  if (rc) return rc;
  memset(p, 0, sizeof(*p));
  int want = o ? o->variant : SKETCH_VARIANT_AUTO;
  if (want < 0 || want > SKETCH_VARIANT_SMALL) return SKETCH_ERR_INVALID;
  p->hash_mode = (o && o->hash_mode) ? o->hash_mode : 1;
  if (p->hash_mode != 1 && p->hash_mode != 2) return SKETCH_ERR_INVALID;
  if (f16 && !h16rn) p->hash_mode = 1;   // bfloat16 / SR / dither kernels hash on the fly
  size_t sm_bytes = 0;
  // the privatised kernel is FP16-RN with precomputed hashes; its R-row steps must be aligned in the global
  // row index.  Everything else (FP32, SR, odd shapes) runs the flat / generic kernels.
  const int64_t rb0 = o ? o->row_begin : 0;
  bool sm_ok = h16rn && smem_feasible(s, n, lda, A, B, &sm_bytes) &&
               (rb0 % sk::smem_step_rows(s->zeta) == 0);
  sk::TmemShape tm = {0, 0, 0, 0, 0, 0};
  const int gm_force = (o ? o->tmem_group_mode : 0) - 1;
  const int tm_mode = tmem_mode_of(out, rounding);
  bool tm_ok = tmem_feasible(s, n, lda, rows, A, B, gm_force, tm_mode, &tm);
  // per-warp shared-memory partials (kernel_small.cuh)
  const size_t small_bytes = (size_t)sk::small_warps() * s->d * n * 2;
  bool small_ok = h16rn && zeta_templated(s->zeta) && n % 2 == 0 && lda % 2 == 0 && aligned(A, 8) &&
                  small_bytes <= (size_t)s->smem_optin;
  int vmax = flat_vec_for(f16, n, lda, A, B, 8);
  int vpair = flat_vec_for(f16, n, lda, A, B, f16 ? 2 : 1);
  // the flat kernels index the chunks of a (32 / zeta)-row macro step with 32 bits
  bool zt = zeta_templated(s->zeta) && (int64_t)n * (32 / (zeta_templated(s->zeta) ? s->zeta : 1)) < (1ll << 31);

  int v = want;
  if (v == SKETCH_VARIANT_AUTO) {
    // measured on B200 (profiles/r01_variant_sweep.md): with one contribution per element (zeta = 1) the
    // 16-byte REDs of the flat kernel stay under the L2 atomic rate and beat the privatised kernel, whose
    // one-row steps are issue-bound; from zeta = 2 on the privatised kernel wins wherever it fits
    // the tensor-memory kernel (profiles/r01_tmem_*.md) beats both wherever it fits; below ~4 MiB of A the
    // launch is latency-bound and the lighter kernels win
    // (64-feature column slices cut into bucket groups of several blocks -- d = 640 at n = 320 -- measured 2.69 TB/s
    // against 2.80 TB/s of the flat REDs; with one block per warp they get 128-row stages and win: d = 2048 at n = 256
    // 2.99 vs 2.74 TB/s; without bucket groups -- d = 384 at n = 192 -- the same slices run at 4.65 TB/s)
    // (the FP32 path privatised in tensor memory beats its flat REDs -- 1.4 TB/s is the L2-atomic ceiling of an FP32
    // zeta = 4 scatter -- with up to two bucket groups: c5 3.4 vs 12.1 ms, c4-512 2.3 vs 6.0 ms; with four, every warp
    // converts the whole FP32 tile for itself and the kernel loses: c4 7.0, n = 1024 / d = 1024 7.2 vs 6.0 ms flat)
    // (at zeta = 8 the flat REDs carry twice the payload: n = 1024, d = 2048 runs 4.68 ms in tensor memory against 6.04 ms flat)
    // (per-contribution conversion -- SR, dither -- is integer-ALU work: 2^33 counter hashes and conversions at c5.  The flat
    // kernel spreads it over 64 warps per SM and runs 29 ms (SR) / 22 ms (dither); the tensor-memory kernel has four consumer
    // warps per SM and takes 218 / 92 ms (profiles/r02_sr_dither.md).  AUTO therefore keeps SR and dither on the flat REDs
    // and gets the accuracy of a two-level sum from many L2-resident partial sketches instead, see the replica rule below)
    const bool perj = out == sk::OUT_F16 && rounding != SKETCH_RN;
    if (tm_ok && !perj && (f16 ? (s->zeta > 4 || !(tm.X * tm.S == 1 && tm.BQ > 1 && tm.BQ != s->zeta)) : tm.BQ <= 2) && rows * (int64_t)n > (1 << 20))
      v = SKETCH_VARIANT_TMEM;
    else if (sm_ok && s->zeta >= 2) v = SKETCH_VARIANT_SMEM;
    // launch-bound inputs into a sketch of a few KiB: the flat REDs queue ~1000 deep on each L2 sector (c1: 10 us);
    // per-warp shared-memory partials need no such queue
    else if (small_ok && small_bytes <= 64 * 1024 && rows * (int64_t)n <= (1 << 20)) v = SKETCH_VARIANT_SMALL;
    else if (zt && vmax) v = SKETCH_VARIANT_FLAT_VEC;
    else v = SKETCH_VARIANT_GENERIC;
  }
  if (v == SKETCH_VARIANT_SMEM && !sm_ok) return SKETCH_ERR_UNSUPPORTED;
  if (v == SKETCH_VARIANT_TMEM && !tm_ok) return SKETCH_ERR_UNSUPPORTED;
  if (v == SKETCH_VARIANT_SMALL && !small_ok) return SKETCH_ERR_UNSUPPORTED;
  if (v == SKETCH_VARIANT_FLAT_VEC && !(zt && vmax)) return SKETCH_ERR_UNSUPPORTED;
  if (v == SKETCH_VARIANT_FLAT_PAIR && !(zt && vpair)) return SKETCH_ERR_UNSUPPORTED;
  p->variant = v;
  p->zeta_t = s->zeta;

  if (v == SKETCH_VARIANT_TMEM) {
    p->hash_mode = 1;  // the producer warp hashes on the fly
    p->replicas = 1;
    p->tm = tm;
    p->tm_mode = tm_mode;
    p->wpc = tm.NW + 1;
    p->smem_bytes = sk::tmem_smem_bytes_for(s->zeta, n / tm.CS, tm.BQ, tm.GM, tm_mode);
    const int T = sk::tmem_rows_per_stage(n / tm.CS, tm.BQ, s->zeta);
    int64_t stages = (rows + T - 1) / T;
    // one CTA per SM (it owns all 512 TMEM columns); gridDim.y = CS column slices share a row range
    int64_t grid = s->sm_count / tm.CS;
    if (o && o->grid_ctas > 0) grid = (o->grid_ctas + tm.CS - 1) / tm.CS;
    if (grid > stages) grid = stages;
    if (grid < 1) grid = 1;
    p->grid = (int)grid;
    return SKETCH_OK;
  }

  if (v == SKETCH_VARIANT_SMALL) {
    p->hash_mode = 1;
    p->replicas = 1;
    p->wpc = sk::small_warps();
    p->smem_bytes = small_bytes;
    const int64_t rb = 16;   // rows per step of k_small (two batches of 8; 2 x 4 at zeta = 8)
    // one step per warp while that keeps the grid at <= 32 CTAs: every CTA ends with d*n/2 REDs into the same few
    // L2 sectors, which is the queue this kernel exists to avoid
    int64_t rpw = (rows + 32 * (int64_t)p->wpc - 1) / (32 * (int64_t)p->wpc);
    rpw = (rpw + rb - 1) / rb * rb;
    if (rpw < rb) rpw = rb;
    int64_t grid = (rows + rpw * p->wpc - 1) / (rpw * p->wpc);
    if (o && o->grid_ctas > 0) {
      grid = o->grid_ctas;
      rpw = (rows + grid * p->wpc - 1) / (grid * p->wpc);
      rpw = (rpw + rb - 1) / rb * rb;
      if (rpw < rb) rpw = rb;
    }
    if (grid < 1) grid = 1;
    p->grid = (int)grid;
    p->rows_per_cta = rpw;   // rows per WARP for this variant
    return SKETCH_OK;
  }

  if (v == SKETCH_VARIANT_SMEM) {
    p->hash_mode = 2;  // always the precomputed entries
    p->vec = 2 * sk::smem_step_rows(s->zeta);
    p->wpc = n / 64;
    p->smem_bytes = sm_bytes;
    p->replicas = 1;
    int per_sm = (int)((size_t)s->smem_per_sm / (sm_bytes + 1024));
    if (per_sm < 1) per_sm = 1;
    int max_warps_per_sm = 64 / p->wpc;
    if (per_sm > max_warps_per_sm) per_sm = max_warps_per_sm;
    if (per_sm > 32) per_sm = 32;
    int64_t grid = (int64_t)s->sm_count * per_sm;
    if (o && o->grid_ctas > 0) grid = o->grid_ctas;
    // every CTA gets a whole number of loop iterations (two load batches); the kernel itself masks the
    // steps past the end of the range
    const int64_t ring = sk::smem_ring_rows(s->zeta, p->wpc);
    const int64_t rows_main = rows;
    p->rows_main = rows_main;
    int64_t rpc = (rows_main + grid - 1) / grid;
    rpc = (rpc + ring - 1) / ring * ring;
    if (rpc < ring) rpc = ring;
    grid = (rows_main + rpc - 1) / rpc;
    if (grid < 1) grid = 1;
    p->grid = (int)grid;
    p->rows_per_cta = rpc;
    return SKETCH_OK;
  }

  if (v == SKETCH_VARIANT_GENERIC) {
    p->vec = 1;
    p->hash_mode = 1;
  } else {
    p->vec = (v == SKETCH_VARIANT_FLAT_PAIR) ? vpair : vmax;
  }
  int P = (o && o->replicas > 0) ? o->replicas : 0;
  if (P == 0) {
    // auto: as many L2-resident partial sketches as 16 MiB of scratch hold, at most 256.  Eight spread the same-line RED
    // traffic over L2; more cost nothing (c5 FP16-RN: 6.93 ms with 8, 6.06 ms with 128 - 256) and shorten every running sum
    // -- each partial sums 1/P of the contributions, the fold adds P partials -- which is what keeps a flat FP16 scatter
    // inside the north star's 5e-2 (c5: relF 3.8e-2 with 8 partials, 7e-3 with 256; profiles/r02_sr_dither.md);
    // launch-bound inputs (c1: 12.3 us with P = 1 vs 13.6 us with the fold kernel) RED straight into B
    size_t one = (size_t)s->d * n * (f16 ? 2 : 4);
    size_t cap = (16u << 20) / (one ? one : 1);
    const size_t by_input = (size_t)(rows * (int64_t)n * 4 / 8) / (one ? one : 1);   // zeroing + folding them stays under 1/8 of A's bytes
    if (cap > by_input) cap = by_input;
    P = (int)(cap < 1 ? 1 : cap > 256 ? 256 : cap);
    if (rows * (int64_t)n <= (1 << 20)) P = 1;
  }
  if (P > 4096) P = 4096;
  p->replicas = P;
  int64_t work_warps;
  if (v == SKETCH_VARIANT_GENERIC) {
    work_warps = (rows * (int64_t)n + 31) / 32;
  } else {
    int hb = 32 / s->zeta;
    work_warps = (rows + hb - 1) / hb;
  }
  int64_t grid = (work_warps + 7) / 8;
  int64_t cap = (int64_t)s->sm_count * 8;
  if (grid > cap) grid = cap;
  if (grid < 1) grid = 1;
  if (o && o->grid_ctas > 0) grid = o->grid_ctas;
  p->grid = (int)grid;
  (void)rounding;
  return SKETCH_OK;
}

// elements between two partial sketches / result slots: padded to 16 bytes so that every partial keeps the vector-RED
// alignment of the first (d * n may be odd)
inline int64_t padded_count(int64_t count) { return (count + 7) / 8 * 8; }

sk::ScatterArgs make_args(const sketch* s, const float* A, int n, int64_t lda, void* B, int64_t row_begin,
                          int64_t rows, uint64_t sr_seed, int vec) {
  sk::ScatterArgs a;
  a.A = A;
  a.lda = lda;
  a.row_begin = row_begin;
  a.rows = rows;
  a.B = B;
  a.replica_stride = padded_count((int64_t)s->d * n);
  a.replicas = 1;
  a.odd_tail = -1;
  a.n = n;
  a.zeta = s->zeta;
  a.db = s->db;
  a.seed = s->seed;
  a.sr_seed = sr_seed;
  a.scale = s->scale;
  a.cpr = (uint32_t)(n / (vec > 0 ? vec : 1));
  // c / cpr by multiply-high: with magic = ceil(2^32 / cpr), umulhi(c, magic) is exact while c * (magic * cpr - 2^32) <
  // 2^32; the excess is below cpr and c below (32 / zeta) * cpr, so (32 / zeta) * cpr^2 <= 2^32 suffices.  Wider rows
  // (n ~ 16k and up) divide.
  const uint64_t cmax = (uint64_t)(32 / (s->zeta <= 32 ? (s->zeta > 0 ? s->zeta : 1) : 32)) * a.cpr;
  a.cpr_magic = (a.cpr <= 1) ? 0u : (cmax * a.cpr <= (1ull << 32)) ? (uint32_t)(((1ull << 32) + a.cpr - 1) / a.cpr) : 0xFFFFFFFFu;
  a.packed = nullptr;
  return a;
}

// Every feasibility condition is decided on the host by make_plan, before anything is enqueued: a failing launch is
// a CUDA error (SKETCH_ERR_CUDA, text in sketch_last_error), never "unsupported".
int launched(cudaError_t e, const char* what) {
  if (e != cudaSuccess) return cuda_fail(e, what);
  g_launches.fetch_add(1, std::memory_order_relaxed);
  return SKETCH_OK;
}

// Order the library-owned scratch behind its previous use when the caller switches streams.  Inside a stream capture
// nothing is recorded or waited for (events cannot cross a capture): replays of a captured apply that uses scratch must
// be ordered by the caller against every other apply on the handle (include/sparse_sketch.h, "CUDA graphs").
int scratch_acquire(sketch* s, cudaStream_t st, bool* capturing) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  CU_TRY(cudaStreamIsCapturing(st, &cs));
  *capturing = cs != cudaStreamCaptureStatusNone;
  if (*capturing) return SKETCH_OK;
  if (s->scratch_busy && s->scratch_stream != st) CU_TRY(cudaStreamWaitEvent(st, s->ev_scratch, 0));
  return SKETCH_OK;
}
int scratch_release(sketch* s, cudaStream_t st, bool capturing) {
  if (capturing) return SKETCH_OK;
  if (!s->ev_scratch) CU_TRY(cudaEventCreateWithFlags(&s->ev_scratch, cudaEventDisableTiming));
  CU_TRY(cudaEventRecord(s->ev_scratch, st));
  s->scratch_stream = st;
  s->scratch_busy = 1;
  return SKETCH_OK;
}

constexpr int kSbReplicas = 64;   // partial FP32 sketches of a fused right-hand side

// fold P partial sketches (k_reduce_replicas) in the sketch's own element type
int fold_replicas(int out, const void* rep, int64_t stride, int P, void* B, int64_t count, int accumulate, int grid, cudaStream_t st) {
  if (out == sk::OUT_F16) sk::k_reduce_replicas<sk::OUT_F16><<<grid, 256, 0, st>>>(rep, stride, P, B, count, accumulate);
  else if (out == sk::OUT_BF16) sk::k_reduce_replicas<sk::OUT_BF16><<<grid, 256, 0, st>>>(rep, stride, P, B, count, accumulate);
  else sk::k_reduce_replicas<sk::OUT_F32><<<grid, 256, 0, st>>>(rep, stride, P, B, count, accumulate);
  return launch_check("k_reduce_replicas");
}

// tensor map of a strided / column-sliced tensor-memory launch, from the handle's cache
int tensor_map_for(sketch* s, const float* A, int n, int64_t lda, int64_t rows, int n_cta, int box_rows, const CUtensorMap** out) {
  for (int k = 0; k < s->tmap_count; ++k) {
    const sketch::TmapSlot& t = s->tmaps[k];
    if (t.A == A && t.lda == lda && t.rows == rows && t.n == n && t.n_cta == n_cta && t.box_rows == box_rows) {
      *out = &t.map;
      return SKETCH_OK;
    }
  }
  const int slot = s->tmap_next;
  sketch::TmapSlot& t = s->tmaps[slot];
  cudaError_t e = sk::tmem_make_tensor_map(A, n, lda, rows, n_cta, box_rows, &t.map);
  if (e != cudaSuccess) return cuda_fail(e, "cuTensorMapEncodeTiled");
  t.A = A; t.lda = lda; t.rows = rows; t.n = n; t.n_cta = n_cta; t.box_rows = box_rows;
  s->tmap_next = (slot + 1) % 8;
  if (s->tmap_count < 8) ++s->tmap_count;
  *out = &t.map;
  return SKETCH_OK;
}

// a1 in its precomputed form.  16-bit entries in sub-step order (kernel_smem.cuh) when zeta is templated and the
// sketch fits the 15-bit bucket field, else plain 32-bit entries (bucket | sign<<31).  force: re-run the kernel.
int ensure_packed(sketch* s, cudaStream_t st, bool force, bool capturing) {
  if (s->packed_width && !force) {
    if (capturing) s->packed_pinned = 1;
    return SKETCH_OK;
  }
  if (capturing) {
    // the array would be filled when the graph is replayed, not now, while the handle already counted it as built
    snprintf(g_last_error, sizeof(g_last_error),
             "the packed hash array cannot be built inside a stream capture; call sketch_precompute_hashes (or run the same "
             "apply once) before capturing");
    return SKETCH_ERR_CAPTURE;
  }
  int rc = ensure_device(s);
  if (rc) return rc;
  const bool rot = rot_ok(s);
  const int64_t total = s->m * (int64_t)s->zeta;
  rc = ensure_scratch(s, &s->packed, &s->packed_bytes, (size_t)total * (rot ? 2 : 4), false, &s->packed_pinned);
  if (rc) return rc;
  int64_t blocks = rot ? (s->m / 28 + 1 + 7) / 8 : (total + 255) / 256;  // rot: one warp per 28 rows, 8 warps per block
  int64_t cap = (int64_t)s->sm_count * 16;
  int grid = (int)(blocks < cap ? blocks : cap);
  if (grid < 1) grid = 1;
  if (rot) {
    rc = launched(sk::launch_hash_pack_rot(s->seed, s->zeta, s->m, s->db, (uint16_t*)s->packed, grid, st), "k_hash_pack_rot");
  } else {
    sk::k_hash_pack32<<<grid, 256, 0, st>>>(s->seed, total, (uint32_t)s->zeta, s->db, (uint32_t*)s->packed);
    rc = launch_check("k_hash_pack32");
  }
  if (rc) return rc;
  s->packed_width = rot ? 2 : 4;
  return SKETCH_OK;
}

int validate_apply(const sketch* s, const void* A, int32_t n, int64_t lda, const void* B, bool f16,
                   const sketch_opts_t* o, int64_t* row_begin, int64_t* rows) {
  if (!s || !B) return SKETCH_ERR_NULL;
  if (n <= 0) return SKETCH_ERR_INVALID;
  if (lda < n) return SKETCH_ERR_LDA;
  if (!aligned(A, 4) || !aligned(B, 4)) return SKETCH_ERR_ALIGNMENT;  // f16: packed RED works on 4-byte words
  (void)f16;
  int64_t rb = o ? o->row_begin : 0;
  int64_t r = o ? o->rows : 0;
  if (o && (o->tmem_group_mode < 0 || o->tmem_group_mode > 3)) return SKETCH_ERR_INVALID;
  if (rb < 0 || r < 0 || rb > s->m) return SKETCH_ERR_INVALID;
  if (r == 0) r = s->m - rb;
  if (rb + r > s->m) return SKETCH_ERR_INVALID;
  if (!A && r > 0) return SKETCH_ERR_NULL;   // an empty row range reads nothing: A may be NULL (an empty tensor has no storage)
  *row_begin = rb;
  *rows = r;
  return SKETCH_OK;
}

// The fused right-hand side (rhs, Sb): b[rows] FP32 is sketched with the same map into Sb[d] FP32.  The
// tensor-memory kernel does it in the same pass (its producer lanes hold every row's hashes); the other variants run a
// second, one-column FP32 scatter behind the first.
int apply_device(const sketch_t* cs, const float* A, int32_t n, int64_t lda, void* B, int out, int rounding,
                 uint64_t sr_seed, const sketch_opts_t* o, void* stream, const float* rhs = nullptr, float* Sb = nullptr) {
  sketch* s = const_cast<sketch*>(cs);
  const bool f16 = out != sk::OUT_F32;   // a 16-bit sketch
  int64_t row_begin = 0, rows = 0;
  int rc = validate_apply(s, A, n, lda, B, f16, o, &row_begin, &rows);
  if (rc) return rc;
  if ((rhs == nullptr) != (Sb == nullptr)) return SKETCH_ERR_NULL;
  if (rhs && (!aligned(rhs, 4) || !aligned(Sb, 4))) return SKETCH_ERR_ALIGNMENT;
  if (out == sk::OUT_F16 ? (rounding != SKETCH_RN && rounding != SKETCH_SR && rounding != SKETCH_DITHER) : rounding != SKETCH_RN)
    return SKETCH_ERR_INVALID;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  Plan p;
  rc = make_plan(s, n, lda, A, B, out, rounding, o, rows, &p);
  if (rc) return rc;
  const int accumulate = o ? o->accumulate : 0;
  const size_t elem = f16 ? 2 : 4;
  const size_t out_bytes = (size_t)s->d * n * elem;

  if (rhs && p.variant != SKETCH_VARIANT_TMEM) {
    sketch_opts_t ob;
    memset(&ob, 0, sizeof(ob));
    ob.accumulate = accumulate;
    ob.row_begin = row_begin;
    ob.rows = rows;
    if (rows == 0) {   // the ABI reads rows = 0 as "through row m - 1": an empty range only zero-fills
      if (!accumulate) CU_TRY(cudaMemsetAsync(Sb, 0, (size_t)s->d * 4, st));
    } else {
      rc = apply_device(cs, rhs, 1, 1, Sb, sk::OUT_F32, SKETCH_RN, 0, &ob, stream);
      if (rc) return rc;
    }
  }

  if (p.variant == SKETCH_VARIANT_TMEM) {
    if (!accumulate) CU_TRY(cudaMemsetAsync(B, 0, out_bytes, st));  // a0
    if (rhs && rows == 0 && !accumulate) CU_TRY(cudaMemsetAsync(Sb, 0, (size_t)s->d * 4, st));
    if (rows > 0) {
      sk::TmemArgs g;
      g.s = make_args(s, A, n, lda, B, row_begin, rows, sr_seed, 1);
      g.d = s->d;
      g.rhs = rhs;
      g.Sb = nullptr;
      g.sb_stride = 0;
      g.sb_replicas = 1;
      bool capturing = false;
      if (rhs) {
        // FP32 REDs of the m zeta contributions of b into kSbReplicas partial sketches (same-address traffic in L2 spread
        // over as many lines; every running sum that much shorter), folded into Sb behind the kernel
        rc = scratch_acquire(s, st, &capturing);
        if (rc) return rc;
        g.sb_stride = padded_count(s->d);
        g.sb_replicas = kSbReplicas;
        rc = ensure_scratch(s, &s->sbrep, &s->sbrep_bytes, (size_t)g.sb_stride * 4 * kSbReplicas, capturing, &s->sbrep_pinned);
        if (rc) return rc;
        g.Sb = static_cast<float*>(s->sbrep);
        CU_TRY(cudaMemsetAsync(s->sbrep, 0, (size_t)g.sb_stride * 4 * kSbReplicas, st));
      }
      const CUtensorMap* tmap = nullptr;
      const int n_cta = n / p.tm.CS;
      if (lda != n_cta) {
        rc = tensor_map_for(s, A, n, lda, rows, n_cta, sk::tmem_rows_per_stage(n_cta, p.tm.BQ, s->zeta), &tmap);
        if (rc) return rc;
      }
      rc = launched(sk::launch_tmem(g, s->zeta, p.tm_mode, p.tm, tmap, p.grid, st), "k_tmem");
      if (rc) return rc;
      if (rhs) {
        int grid = (s->d + 255) / 256;
        sk::k_reduce_replicas<sk::OUT_F32><<<grid, 256, 0, st>>>(s->sbrep, g.sb_stride, kSbReplicas, Sb, s->d, accumulate);
        rc = launch_check("k_reduce_replicas (rhs)");
        if (rc) return rc;
        rc = scratch_release(s, st, capturing);
        if (rc) return rc;
      }
    }
    return SKETCH_OK;
  }

  if (p.variant == SKETCH_VARIANT_SMALL) {
    if (!accumulate) CU_TRY(cudaMemsetAsync(B, 0, out_bytes, st));  // a0
    if (rows > 0) {
      sk::SmallArgs g;
      g.s = make_args(s, A, n, lda, B, row_begin, rows, sr_seed, 2);
      g.rows_per_warp = p.rows_per_cta;
      g.d = s->d;
      rc = launched(sk::launch_small_f16(g, s->zeta, p.grid, p.smem_bytes, st), "k_small");
      if (rc) return rc;
    }
    return SKETCH_OK;
  }

  if (p.variant == SKETCH_VARIANT_SMEM) {
    if (!accumulate) CU_TRY(cudaMemsetAsync(B, 0, out_bytes, st));  // a0
    if (p.rows_main > 0) {
      sk::SmemArgs g;
      g.s = make_args(s, A, n, lda, B, row_begin, p.rows_main, sr_seed, p.vec);
      g.rows_per_cta = p.rows_per_cta;
      g.d = s->d;
      g.zero = 0u;
      bool capturing = false;
      rc = scratch_acquire(s, st, &capturing);
      if (rc) return rc;
      rc = ensure_packed(s, st, false, capturing);
      if (rc) return rc;
      g.s.packed = s->packed;
      rc = launched(sk::launch_smem_f16(g, s->zeta, p.wpc, p.grid, p.smem_bytes, st), "k_smem");
      if (rc) return rc;
      rc = scratch_release(s, st, capturing);
      if (rc) return rc;
    }
    return SKETCH_OK;
  }

  // flat / generic: RED into B itself (P == 1) or into P partial sketches folded afterwards
  void* target = B;
  int P = p.replicas;
  const int64_t count = (int64_t)s->d * n;
  const int64_t pstride = padded_count(count);      // elements between partial sketches
  const bool packed_hashes = p.hash_mode == 2 && p.variant != SKETCH_VARIANT_GENERIC;
  const bool uses_scratch = P > 1 || packed_hashes;
  bool capturing = false;
  if (uses_scratch) {
    rc = scratch_acquire(s, st, &capturing);
    if (rc) return rc;
  }
  if (P > 1) {
    rc = ensure_scratch(s, &s->rep, &s->rep_bytes, (size_t)pstride * elem * P, capturing, &s->rep_pinned);
    if (rc) return rc;
    target = s->rep;
    CU_TRY(cudaMemsetAsync(target, 0, (size_t)pstride * elem * P, st));
  } else if (!accumulate) {
    CU_TRY(cudaMemsetAsync(B, 0, out_bytes, st));
  }
  int pw = 0;
  if (packed_hashes) {
    rc = ensure_packed(s, st, false, capturing);
    if (rc) return rc;
    pw = s->packed_width;
  }
  if (rows > 0) {
    sk::ScatterArgs a = make_args(s, A, n, lda, target, row_begin, rows, sr_seed, p.vec);
    a.replicas = P;
    a.packed = pw ? s->packed : nullptr;
    if (p.variant == SKETCH_VARIANT_GENERIC) {
      if (f16 && P == 1 && (count & 1)) a.odd_tail = count - 1;
      rc = launched(sk::launch_generic(a, out, rounding, p.grid, st), "k_generic");
    } else if (out == sk::OUT_F32) {
      rc = launched(sk::launch_flat_f32(a, s->zeta, p.vec, pw, p.grid, st), "k_flat<f32>");
    } else if (out == sk::OUT_BF16) {
      rc = launched(sk::launch_flat_bf16(a, s->zeta, p.vec, p.grid, st), "k_flat<bf16>");
    } else {
      rc = launched(sk::launch_flat_f16(a, s->zeta, p.vec, rounding, pw, p.grid, st), "k_flat<f16>");
    }
    if (rc) return rc;
  }
  if (P > 1) {
    int grid = (int)((count + 255) / 256);
    if (grid > s->sm_count * 8) grid = s->sm_count * 8;
    rc = fold_replicas(out, target, pstride, P, B, count, accumulate, grid, st);
    if (rc) return rc;
  }
  if (uses_scratch) {
    rc = scratch_release(s, st, capturing);
    if (rc) return rc;
  }
  return SKETCH_OK;
}

int ensure_host_path(sketch* s) {
  if (s->host_ready) return SKETCH_OK;
  CU_TRY(cudaStreamCreateWithFlags(&s->st_copy, cudaStreamNonBlocking));
  CU_TRY(cudaStreamCreateWithFlags(&s->st_comp, cudaStreamNonBlocking));
  for (int k = 0; k < 2; ++k) {
    CU_TRY(cudaEventCreateWithFlags(&s->ev_copied[k], cudaEventDisableTiming));
    CU_TRY(cudaEventCreateWithFlags(&s->ev_done[k], cudaEventDisableTiming));
  }
  s->host_ready = 1;
  return SKETCH_OK;
}

int apply_host_impl(sketch* s, const float* A, int32_t n, int64_t lda, void* B, int out, int rounding, uint64_t sr_seed,
                    const sketch_opts_t* o, int64_t rb, int64_t rows) {
  int rc;
  const size_t elem = out != sk::OUT_F32 ? 2 : 4;
  const size_t out_bytes = (size_t)s->d * n * elem;
  const size_t slot_bytes = (size_t)padded_count((int64_t)s->d * n) * elem;   // 16-byte aligned slots (d * n may be odd)
  // staging: two buffers of ~256 MiB, whole rows, row count a multiple of 32
  const size_t row_bytes = (size_t)n * 4;
  int64_t chunk_rows = (int64_t)((256u << 20) / row_bytes);
  chunk_rows = chunk_rows / 32 * 32;
  if (chunk_rows < 32) chunk_rows = 32;
  if (chunk_rows > rows) chunk_rows = (rows + 31) / 32 * 32;
  const size_t chunk_bytes = (size_t)chunk_rows * row_bytes;
  if (s->stage_bytes < chunk_bytes) {
    for (int k = 0; k < 2; ++k) {
      size_t have = s->stage[k] ? s->stage_bytes : 0;
      rc = ensure_scratch(s, &s->stage[k], &have, chunk_bytes);
      if (rc) return rc;
    }
    s->stage_bytes = chunk_bytes;
  }
  // one partial sketch per row chunk (slot k mod kSlots), folded once at the end: the chunk level of the
  // accumulation hierarchy.  Adding every chunk into ONE FP16 sketch would put #chunks x #CTAs partial sums
  // on a single running sum (measured at c5: relF 2.5e-2 instead of 7e-3).
  const int64_t nchunks = rows > 0 ? (rows + chunk_rows - 1) / chunk_rows : 0;
  const int64_t kSlots = nchunks < 64 ? (nchunks > 0 ? nchunks : 1) : 64;
  rc = ensure_scratch(s, &s->bdev, &s->bdev_bytes, slot_bytes * (size_t)(kSlots + 1));
  if (rc) return rc;
  char* const slots = static_cast<char*>(s->bdev);            // [kSlots][padded d*n]
  char* const result = slots + slot_bytes * (size_t)kSlots;    // [d][n]
  sketch_opts_t oo;
  memset(&oo, 0, sizeof(oo));
  if (o) oo = *o;
  const int user_acc = o ? o->accumulate : 0;
  if (user_acc) CU_TRY(cudaMemcpyAsync(result, B, out_bytes, cudaMemcpyHostToDevice, s->st_comp));
  if (nchunks == 0) CU_TRY(cudaMemsetAsync(slots, 0, out_bytes, s->st_comp));
  int64_t k = 0;
  for (int64_t r0 = 0; r0 < rows; r0 += chunk_rows, ++k) {
    int64_t nr = rows - r0 < chunk_rows ? rows - r0 : chunk_rows;
    int b = (int)(k & 1);
    if (k >= 2) CU_TRY(cudaStreamWaitEvent(s->st_copy, s->ev_done[b], 0));
    const float* src = A + r0 * lda;
    if (lda == n) CU_TRY(cudaMemcpyAsync(s->stage[b], src, (size_t)nr * row_bytes, cudaMemcpyHostToDevice, s->st_copy));
    else CU_TRY(cudaMemcpy2DAsync(s->stage[b], row_bytes, src, (size_t)lda * 4, row_bytes, (size_t)nr, cudaMemcpyHostToDevice, s->st_copy));
    CU_TRY(cudaEventRecord(s->ev_copied[b], s->st_copy));
    CU_TRY(cudaStreamWaitEvent(s->st_comp, s->ev_copied[b], 0));
    oo.row_begin = rb + r0;
    oo.rows = nr;
    oo.accumulate = k >= kSlots ? 1 : 0;
    rc = apply_device(s, (const float*)s->stage[b], n, n, slots + slot_bytes * (size_t)(k % kSlots), out, rounding, sr_seed, &oo,
                      s->st_comp);
    if (rc) return rc;
    CU_TRY(cudaEventRecord(s->ev_done[b], s->st_comp));
  }
  {
    const int64_t count = (int64_t)s->d * n;
    int grid = (int)((count + 255) / 256);
    if (grid > s->sm_count * 8) grid = s->sm_count * 8;
    rc = fold_replicas(out, slots, padded_count(count), (int)kSlots, result, count, user_acc, grid, s->st_comp);
    if (rc) return rc;
  }
  CU_TRY(cudaMemcpyAsync(B, result, out_bytes, cudaMemcpyDeviceToHost, s->st_comp));
  CU_TRY(cudaStreamSynchronize(s->st_comp));
  return SKETCH_OK;
}

int apply_host(const sketch_t* cs, const float* A, int32_t n, int64_t lda, void* B, int out, int rounding,
               uint64_t sr_seed, const sketch_opts_t* o) {
  sketch* s = const_cast<sketch*>(cs);
  if (!s || !A || !B) return SKETCH_ERR_NULL;
  if (n <= 0) return SKETCH_ERR_INVALID;
  if (lda < n) return SKETCH_ERR_LDA;
  int64_t rb = o ? o->row_begin : 0, rows = o ? o->rows : 0;
  if (rb < 0 || rows < 0 || rb > s->m) return SKETCH_ERR_INVALID;
  if (rows == 0) rows = s->m - rb;
  if (rb + rows > s->m) return SKETCH_ERR_INVALID;
  int rc = ensure_device(s);
  if (rc) return rc;
  rc = ensure_host_path(s);
  if (rc) return rc;
  rc = apply_host_impl(s, A, n, lda, B, out, rounding, sr_seed, o, rb, rows);
  if (rc) {
    // no copy from the caller's A (or into its B) may still be in flight when the call returns
    cudaStreamSynchronize(s->st_copy);
    cudaStreamSynchronize(s->st_comp);
  }
  return rc;
}

}  // namespace

// =================================================================================================
// Built-in scratch of sketch_apply_f16acc_noalloc (include/sparse_sketch.h).
//
// Some programs that link this library must not allocate device memory once they are running: a solver that has handed
// the whole GPU to its own memory pool at start-up, a real-time or safety-reviewed pipeline whose memory map is frozen
// after initialisation (a cudaMalloc there is both forbidden and a latency spike, since it synchronises the device),
// or a plug-in that is called in a context whose owner forbids allocation.  The ordinary flat scatter keeps its partial
// sketches in a cudaMalloc'ed buffer that grows on demand, which these callers cannot use.  For them the partial
// sketches live in the array below: it is part of the library's device image, so the driver reserves it when the module
// is loaded on a GPU and gives it back when the process exits -- SKETCH_NOALLOC_SCRATCH_BYTES on every GPU that loads
// the library, whether or not the entry point is ever called.
//
// On the host the identifier g_noalloc_scratch is only a handle for the runtime's symbol table -- its host address is
// not a device address and must never reach a kernel.  noalloc_scratch_ptr() asks the runtime for the real address on
// the CURRENT device (cudaGetSymbolAddress), once per device ordinal, and that is the only pointer the launches see.
// =================================================================================================
static __device__ __align__(256) unsigned char g_noalloc_scratch[SKETCH_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
void* g_noalloc_ptr[kNoallocMaxDevices];   // device address of g_noalloc_scratch per device ordinal; nullptr = not asked yet

// Device address of the built-in scratch on the current device.  The first call on a device performs the symbol lookup
// (which may also make the runtime load this library's module on that device); later calls only read the cached pointer.
int noalloc_scratch_ptr(void** out) {
  int dev = -1;
  CU_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoallocMaxDevices) {
    snprintf(g_last_error, sizeof(g_last_error), "sketch_apply_f16acc_noalloc: device ordinal %d outside [0, %d)", dev, kNoallocMaxDevices);
    return SKETCH_ERR_CUDA;
  }
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_ptr[dev]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_noalloc_scratch)");
    if (!p) {
      snprintf(g_last_error, sizeof(g_last_error), "cudaGetSymbolAddress(g_noalloc_scratch) returned a null address on device %d", dev);
      return SKETCH_ERR_CUDA;
    }
    g_noalloc_ptr[dev] = p;
  }
  *out = g_noalloc_ptr[dev];
  return SKETCH_OK;
}

}  // namespace

// =================================================================================================
extern "C" {

int sketch_create(int64_t m, int32_t d, int32_t zeta, uint64_t seed, sketch_t** out) {
  if (!out) return SKETCH_ERR_NULL;
  *out = nullptr;
  if (m <= 0 || d <= 0 || zeta < 1) return SKETCH_ERR_INVALID;
  if (d % zeta != 0) return SKETCH_ERR_DIVISIBILITY;
  if ((uint64_t)m > (1ull << 62) / (uint64_t)zeta) return SKETCH_ERR_INVALID;
  sketch* s = new (std::nothrow) sketch;
  if (!s) return SKETCH_ERR_NOMEM;
  memset(s, 0, sizeof(*s));
  s->m = m;
  s->d = d;
  s->zeta = zeta;
  s->db = (uint32_t)(d / zeta);
  s->seed = seed;
  s->scale = (float)(1.0 / std::sqrt((double)zeta));  // correctly rounded from FP64 (R5)
  *out = s;
  return SKETCH_OK;
}

int sketch_destroy(sketch_t* s) {
  if (!s) return SKETCH_OK;
  if (s->rep) cudaFree(s->rep);
  if (s->sbrep) cudaFree(s->sbrep);
  if (s->packed) cudaFree(s->packed);
  while (s->retired) {
    sketch::Retired* r = s->retired;
    s->retired = r->next;
    cudaFree(r->buf);
    delete r;
  }
  for (int k = 0; k < 2; ++k)
    if (s->stage[k]) cudaFree(s->stage[k]);
  if (s->bdev) cudaFree(s->bdev);
  if (s->ev_scratch) cudaEventDestroy(s->ev_scratch);
  if (s->host_ready) {
    cudaStreamDestroy(s->st_copy);
    cudaStreamDestroy(s->st_comp);
    for (int k = 0; k < 2; ++k) {
      cudaEventDestroy(s->ev_copied[k]);
      cudaEventDestroy(s->ev_done[k]);
    }
  }
  delete s;
  return SKETCH_OK;
}

int sketch_hashes_dump(const sketch_t* cs, int32_t* bucket_dev, uint8_t* signbit_dev, void* stream) {
  sketch* s = const_cast<sketch*>(cs);
  if (!s || !bucket_dev || !signbit_dev) return SKETCH_ERR_NULL;
  int rc = ensure_device(s);
  if (rc) return rc;
  int64_t total = s->m * (int64_t)s->zeta;
  int64_t blocks = (total + 255) / 256;
  int64_t cap = (int64_t)s->sm_count * 16;
  int grid = (int)(blocks < cap ? blocks : cap);
  sk::k_hash_dump<<<grid, 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(s->seed, total, (uint32_t)s->zeta, s->db,
                                                                            bucket_dev, signbit_dev);
  return launch_check("k_hash_dump");
}

int sketch_precompute_hashes(sketch_t* s, void* stream) {
  if (!s) return SKETCH_ERR_NULL;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  bool capturing = false;
  int rc = scratch_acquire(s, st, &capturing);
  if (rc) return rc;
  rc = ensure_packed(s, st, true, capturing);
  if (rc) return rc;
  return scratch_release(s, st, capturing);
}

int sketch_apply_f32acc(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, float* B_dev, void* stream) {
  return apply_device(s, A_dev, n, lda, B_dev, sk::OUT_F32, SKETCH_RN, 0, nullptr, stream);
}

int sketch_apply_f16acc(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev, int rounding,
                        uint64_t sr_seed, void* stream) {
  return apply_device(s, A_dev, n, lda, B_dev, sk::OUT_F16, rounding, sr_seed, nullptr, stream);
}

int sketch_apply_bf16acc(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev, void* stream) {
  return apply_device(s, A_dev, n, lda, B_dev, sk::OUT_BF16, SKETCH_RN, 0, nullptr, stream);
}

int sketch_apply_f32acc_ex(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, float* B_dev,
                           const sketch_opts_t* opts, void* stream) {
  return apply_device(s, A_dev, n, lda, B_dev, sk::OUT_F32, SKETCH_RN, 0, opts, stream);
}

int sketch_apply_f16acc_ex(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev, int rounding,
                           uint64_t sr_seed, const sketch_opts_t* opts, void* stream) {
  return apply_device(s, A_dev, n, lda, B_dev, sk::OUT_F16, rounding, sr_seed, opts, stream);
}

int sketch_apply_bf16acc_ex(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, void* B_dev,
                            const sketch_opts_t* opts, void* stream) {
  return apply_device(s, A_dev, n, lda, B_dev, sk::OUT_BF16, SKETCH_RN, 0, opts, stream);
}

// The flat FP16 scatter with its partial sketches in g_noalloc_scratch instead of the handle's cudaMalloc'ed buffer.
// Same kernels and the same arithmetic as sketch_apply_f16acc_ex with variant FLAT_VEC (GENERIC for shapes the vector REDs
// cannot take) and `replicas` partial sketches; nothing on this path calls cudaMalloc, cudaFree or a library routine that
// allocates (cudaMemsetAsync, the two launches and -- first call on a device only -- cudaGetSymbolAddress are all it uses).
int sketch_apply_f16acc_noalloc(const sketch_t* cs, const float* A_dev, int32_t n, int64_t lda, void* B_dev, int rounding,
                                uint64_t sr_seed, void* stream) {
  sketch* s = const_cast<sketch*>(cs);
  int64_t row_begin = 0, rows = 0;
  int rc = validate_apply(s, A_dev, n, lda, B_dev, true, nullptr, &row_begin, &rows);
  if (rc) return rc;
  if (rounding != SKETCH_RN && rounding != SKETCH_SR && rounding != SKETCH_DITHER) return SKETCH_ERR_INVALID;
  // at least two partial sketches must fit: with one, the scatter would go straight into B and need no scratch at all
  const int64_t count = (int64_t)s->d * n;
  const int64_t pstride = padded_count(count);
  const uint64_t slot_bytes = (uint64_t)pstride * 2;
  const uint64_t fit = (uint64_t)SKETCH_NOALLOC_SCRATCH_BYTES / slot_bytes;
  if (fit < 2) {
    snprintf(g_last_error, sizeof(g_last_error),
             "sketch_apply_f16acc_noalloc: a %d x %d FP16 sketch takes %llu bytes per partial sketch; two of them do not fit the "
             "built-in scratch of %llu bytes (limit: d * n <= %llu)",
             s->d, n, (unsigned long long)slot_bytes, (unsigned long long)SKETCH_NOALLOC_SCRATCH_BYTES,
             (unsigned long long)SKETCH_NOALLOC_SCRATCH_BYTES / 4);
    return SKETCH_ERR_SCRATCH_LIMIT;
  }
  // as many partial sketches as fit, at most 256, and no more than keep zeroing + folding under 1/8 of A's bytes
  // (the rule of the allocating path, make_plan)
  uint64_t P = fit < 256 ? fit : 256;
  const uint64_t by_input = (uint64_t)rows * (uint64_t)n * 4 / 8 / slot_bytes;
  if (P > by_input) P = by_input < 2 ? 2 : by_input;
  sketch_opts_t o;
  memset(&o, 0, sizeof(o));
  o.variant = SKETCH_VARIANT_FLAT_VEC;
  o.replicas = (int32_t)P;
  Plan p;
  rc = make_plan(s, n, lda, A_dev, B_dev, sk::OUT_F16, rounding, &o, rows, &p);   // host only
  if (rc == SKETCH_ERR_UNSUPPORTED) {
    o.variant = SKETCH_VARIANT_GENERIC;
    rc = make_plan(s, n, lda, A_dev, B_dev, sk::OUT_F16, rounding, &o, rows, &p);
  }
  if (rc) return rc;
  void* scratch = nullptr;
  rc = noalloc_scratch_ptr(&scratch);
  if (rc) return rc;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  // the array keeps what the previous call left in it: every partial sketch this call adds into starts at zero
  CU_TRY(cudaMemsetAsync(scratch, 0, (size_t)(slot_bytes * P), st));
  sk::ScatterArgs a = make_args(s, A_dev, n, lda, scratch, row_begin, rows, sr_seed, p.vec);
  a.replicas = (int32_t)P;
  if (p.variant == SKETCH_VARIANT_GENERIC) rc = launched(sk::launch_generic(a, sk::OUT_F16, rounding, p.grid, st), "k_generic (noalloc)");
  else rc = launched(sk::launch_flat_f16(a, s->zeta, p.vec, rounding, 0, p.grid, st), "k_flat<f16> (noalloc)");
  if (rc) return rc;
  int grid = (int)((count + 255) / 256);
  if (grid > s->sm_count * 8) grid = s->sm_count * 8;
  return fold_replicas(sk::OUT_F16, scratch, pstride, (int)P, B_dev, count, 0, grid, st);   // overwrites B: a complete sketch
}

int sketch_apply_f16acc_with_rhs(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, const float* b_dev,
                                 void* B16_dev, float* Sb32_dev, const sketch_opts_t* opts, void* stream) {
  if (!b_dev || !Sb32_dev) return SKETCH_ERR_NULL;
  return apply_device(s, A_dev, n, lda, B16_dev, sk::OUT_F16, SKETCH_RN, 0, opts, stream, b_dev, Sb32_dev);
}

int sketch_apply_f32acc_with_rhs(const sketch_t* s, const float* A_dev, int32_t n, int64_t lda, const float* b_dev,
                                 float* B32_dev, float* Sb32_dev, const sketch_opts_t* opts, void* stream) {
  if (!b_dev || !Sb32_dev) return SKETCH_ERR_NULL;
  return apply_device(s, A_dev, n, lda, B32_dev, sk::OUT_F32, SKETCH_RN, 0, opts, stream, b_dev, Sb32_dev);
}

int sketch_widen(const void* B16_dev, int64_t count, int is_bf16, float* out_dev, void* stream) {
  if (!B16_dev || !out_dev) return SKETCH_ERR_NULL;
  if (count < 0) return SKETCH_ERR_INVALID;
  if (!aligned(B16_dev, 2) || !aligned(out_dev, 4)) return SKETCH_ERR_ALIGNMENT;
  if (count == 0) return SKETCH_OK;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  int64_t blocks = (count + 255) / 256;
  const int cap = grid_cap_current_device();
  int grid = (int)(blocks < cap ? blocks : cap);
  if (is_bf16) sk::k_widen<sk::OUT_BF16><<<grid, 256, 0, st>>>(static_cast<const uint16_t*>(B16_dev), count, out_dev);
  else sk::k_widen<sk::OUT_F16><<<grid, 256, 0, st>>>(static_cast<const uint16_t*>(B16_dev), count, out_dev);
  return launch_check("k_widen");
}

int sketch_apply_f32acc_host(const sketch_t* s, const float* A_host, int32_t n, int64_t lda, float* B_host,
                             const sketch_opts_t* opts) {
  return apply_host(s, A_host, n, lda, B_host, sk::OUT_F32, SKETCH_RN, 0, opts);
}

int sketch_apply_f16acc_host(const sketch_t* s, const float* A_host, int32_t n, int64_t lda, void* B_host, int rounding,
                             uint64_t sr_seed, const sketch_opts_t* opts) {
  if (rounding != SKETCH_RN && rounding != SKETCH_SR && rounding != SKETCH_DITHER) return SKETCH_ERR_INVALID;
  return apply_host(s, A_host, n, lda, B_host, sk::OUT_F16, rounding, sr_seed, opts);
}

int sketch_red_probe(void* sketch_dev, int32_t d, int32_t n, int32_t kind, int32_t replicas, int32_t grid_ctas,
                     int32_t iters, uint64_t* red_ops_out, void* stream) {
  if (!sketch_dev) return SKETCH_ERR_NULL;
  if (d <= 0 || n <= 0 || kind < 0 || kind > 8 || replicas < 1 || grid_ctas < 1 || iters < 0) return SKETCH_ERR_INVALID;
  const int vec[9] = {2, 4, 8, 1, 2, 4, 8, 8, 4};
  if (n % vec[kind] != 0) return SKETCH_ERR_INVALID;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  uint64_t ops = (uint64_t)grid_ctas * sk::kFlatThreads * (uint64_t)iters;
  if (kind >= 7) {
    // one bulk reduction per warp and iteration of min(row, 2 KiB) bytes; counted in 16-byte units so that payload = ops * 16
    const int eb = kind == 8 ? 4 : 2;
    int64_t row = (int64_t)n * eb;
    if (row % 16 != 0) return SKETCH_ERR_INVALID;
    int32_t chunk = (int32_t)(row < 2048 ? row : 2048);
    if (row % chunk != 0) return SKETCH_ERR_INVALID;
    if (kind == 7) sk::k_l2_probe<7><<<grid_ctas, sk::kFlatThreads, 2 * chunk, st>>>(sketch_dev, d, n, replicas, iters, chunk);
    else sk::k_l2_probe<8><<<grid_ctas, sk::kFlatThreads, 2 * chunk, st>>>(sketch_dev, d, n, replicas, iters, chunk);
    ops = (uint64_t)grid_ctas * (sk::kFlatThreads / 32) * (uint64_t)iters * (uint64_t)(chunk / 16);
  } else if (kind == 6) {
    sk::k_l2_probe<6><<<grid_ctas, sk::kFlatThreads, 0, st>>>(sketch_dev, d, n, replicas, iters, 0);
  } else {
    switch (kind) {
      case 0: sk::k_red_probe<0><<<grid_ctas, sk::kFlatThreads, 0, st>>>(sketch_dev, d, n, replicas, iters); break;
      case 1: sk::k_red_probe<1><<<grid_ctas, sk::kFlatThreads, 0, st>>>(sketch_dev, d, n, replicas, iters); break;
      case 2: sk::k_red_probe<2><<<grid_ctas, sk::kFlatThreads, 0, st>>>(sketch_dev, d, n, replicas, iters); break;
      case 3: sk::k_red_probe<3><<<grid_ctas, sk::kFlatThreads, 0, st>>>(sketch_dev, d, n, replicas, iters); break;
      case 4: sk::k_red_probe<4><<<grid_ctas, sk::kFlatThreads, 0, st>>>(sketch_dev, d, n, replicas, iters); break;
      default: sk::k_red_probe<5><<<grid_ctas, sk::kFlatThreads, 0, st>>>(sketch_dev, d, n, replicas, iters); break;
    }
  }
  if (red_ops_out) *red_ops_out = ops;
  return launch_check("k_red_probe");
}

int sketch_stream_probe(const void* src_dev, int64_t bytes, int32_t kind, int32_t grid_ctas, void* sink_dev, void* stream) {
  if (!src_dev) return SKETCH_ERR_NULL;
  if (bytes < 0 || kind < 0 || kind > 1 || grid_ctas < 1) return SKETCH_ERR_INVALID;
  if (!aligned(src_dev, 32)) return SKETCH_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (kind == 0) {
    sk::k_stream_probe<0><<<grid_ctas, 256, 0, st>>>(reinterpret_cast<const float*>(src_dev), bytes, reinterpret_cast<uint64_t*>(sink_dev));
  } else {
    const size_t smem = 4 * 32768 + 64;
    cudaError_t e = sk::allow_max_dynamic_smem<sk::k_stream_probe<1>>();
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(k_stream_probe)");
    sk::k_stream_probe<1><<<grid_ctas, 32, smem, st>>>(reinterpret_cast<const float*>(src_dev), bytes, reinterpret_cast<uint64_t*>(sink_dev));
  }
  return launch_check("k_stream_probe");
}

int sketch_convert_probe(const float* p_dev, const uint32_t* rbits_dev, int64_t count, int32_t kind, uint16_t* out_dev, void* stream) {
  if (!p_dev || !out_dev) return SKETCH_ERR_NULL;
  if (count < 0 || kind < 0 || kind > 7) return SKETCH_ERR_INVALID;
  if ((kind == 1 || kind == 2 || kind >= 4) && !rbits_dev) return SKETCH_ERR_NULL;
  if (count == 0) return SKETCH_OK;
  int64_t blocks = (count + 255) / 256;
  const int cap = grid_cap_current_device();
  int grid = (int)(blocks < cap ? blocks : cap);
  sk::k_convert_probe<<<grid, 256, 0, reinterpret_cast<cudaStream_t>(stream)>>>(p_dev, rbits_dev, count, kind, out_dev);
  return launch_check("k_convert_probe");
}

int sketch_plan(const sketch_t* cs, int32_t n, int64_t lda, int is_f16, int rounding, const sketch_opts_t* opts,
                int32_t* variant_out, int32_t* replicas_out, int32_t* hash_mode_out, int32_t* grid_out) {
  sketch* s = const_cast<sketch*>(cs);
  if (!s) return SKETCH_ERR_NULL;
  if (n <= 0) return SKETCH_ERR_INVALID;
  if (lda < n) return SKETCH_ERR_LDA;
  int64_t rb = opts ? opts->row_begin : 0, rows = opts ? opts->rows : 0;
  if (rows == 0) rows = s->m - rb;
  Plan p;
  // plan for 256-byte aligned buffers (what cudaMalloc returns)
  if (is_f16 < 0 || is_f16 > 2) return SKETCH_ERR_INVALID;
  int rc = make_plan(s, n, lda, reinterpret_cast<const void*>(256), reinterpret_cast<const void*>(256),
                     is_f16 == 2 ? sk::OUT_BF16 : is_f16 == 1 ? sk::OUT_F16 : sk::OUT_F32, rounding, opts, rows, &p);
  if (rc) return rc;
  if (variant_out) *variant_out = p.variant;
  if (replicas_out) *replicas_out = p.replicas;
  if (hash_mode_out) *hash_mode_out = p.hash_mode;
  if (grid_out) *grid_out = p.variant == SKETCH_VARIANT_TMEM ? p.grid * p.tm.CS : p.grid;
  return SKETCH_OK;
}

uint64_t sketch_launch_count(void) { return g_launches.load(); }

const char* sketch_strerror(int code) {
  switch (code) {
    case SKETCH_OK: return "ok";
    case SKETCH_ERR_INVALID: return "invalid argument value";
    case SKETCH_ERR_NULL: return "null pointer";
    case SKETCH_ERR_DIVISIBILITY: return "d is not divisible by zeta";
    case SKETCH_ERR_LDA: return "lda < n";
    case SKETCH_ERR_ALIGNMENT: return "buffer is not sufficiently aligned";
    case SKETCH_ERR_UNSUPPORTED: return "the forced variant does not support this shape";
    case SKETCH_ERR_CUDA: return "CUDA runtime error (see sketch_last_error)";
    case SKETCH_ERR_NOMEM: return "out of memory";
    case SKETCH_ERR_CAPTURE: return "library scratch would have to be allocated inside a stream capture (see sketch_last_error)";
    case SKETCH_ERR_SCRATCH_LIMIT: return "sketch too large for the built-in scratch of sketch_apply_f16acc_noalloc (see sketch_last_error)";
  }
  return "unknown error code";
}

const char* sketch_last_error(void) { return g_last_error; }

const char* sketch_version(void) { return "sparse_sketch 0.1 sm_100a"; }

}  // extern "C"
