// tmem_host.cu -- host side of the tensor-memory-privatised scatter: geometry selection (tmem_shape), the tensor map of
// strided / column-sliced tiles, and the dispatcher over the per-(zeta, mode) instantiation units of launch_tmem.cu.
// No kernel is instantiated here.
#include "kernel_tmem.cuh"
#include "launch.h"

namespace sk {

// Geometry for an n-feature, d-row, zeta-block sketch accumulated in `mode` (TM_*): the fewest column slices CS that fit
// at all, then the (X, S, BQ) with the fewest issued instructions per KiB of A.  Model (from the SASS of the main loop,
// profiles/r01_tmem_shapes.md): a row slice of 256 X bytes costs 1 + 3 X instructions to load and convert (in each of the
// BQ warps that need it) and 5.25 + 2 X per stack block to read-modify-write.  A lane holds X words of FW = 2 (16-bit
// modes) or 1 (FP32) features: a CTA covers 32 FW X S features.
bool tmem_shape(int n, int d, int zeta, int64_t lda, int gm_force, int mode, TmemShape* out) {
  const int fw = tm_fw(mode), unit = 32 * fw;
  if (n <= 0 || d <= 0 || zeta <= 0 || n % unit != 0 || d % zeta != 0) return false;
  const int NW = 4;
  for (int cs = 1; cs <= 16; ++cs) {   // odd slice counts serve the widths that are not 64 * 2^k (192, 320, 384, ...)
    if (n % (unit * cs) != 0) continue;
    const int nc = n / cs;
    if (lda != nc && nc > 256) continue;   // strided tiles come through a tensor-map box of at most 256 elements a side
    double best = 0.0;
    bool found = false;
    for (int x = 4; x >= 1; x >>= 1) {
      if (nc % (unit * x) != 0) continue;
      const int s = nc / (unit * x);
      if (s != 1 && s != 2 && s != 4) continue;
      for (int bq = 1; bq <= 4; bq *= 2) {
        if (s * bq > NW || zeta % bq != 0 || d % bq != 0) continue;
        if (bq > 1 && tm_perj(mode)) continue;   // per-contribution conversion reads the FP32 tile: one bucket group
        const int64_t cols = (int64_t)(d / bq) * x;
        if (cols > kTmemCols / (NW / 4) || cols % 8 != 0) continue;
        const double cost = bq * (4.0 / x + 12.0) + zeta * (21.0 / x + 8.0);
        if (!found || cost < best - 1e-9) {
          found = true;
          best = cost;
          out->X = x; out->S = s; out->BQ = bq; out->CS = cs; out->NW = NW;
          // group mode (kernel_tmem.cuh), from the sweep in profiles/r01_tmem_shapes.md: with four bucket groups
          // (one block per warp, one LDTM per row) the chained groups are latency-bound and deferral with groups of
          // 4 rows wins (c4: 3.57 -> 4.13 TB/s); with two bucket groups the chained kernel is faster (c4-512: 5.37 vs
          // 5.07 TB/s).  Deferral needs few clashes -- ZB * C(4,2) / (d/zeta) <= 0.15 -- and d/zeta >= G (G + 1).
          // Only the FP16-RN path has the deferral kernels.
          const double zb = (double)zeta / bq, dbk = (double)d / zeta;
          out->GM = (mode == TM_F16 && bq == 4 && zb * 6.0 / dbk <= 0.15 && dbk >= 20) ? 1 : 0;
          // sketches a quarter of a warp's tensor-memory region or smaller (one bucket group): replicated rows -- each row of a
          // group adds into its own private copy, no chain (kernel_tmem.cuh GM = 5; c2: 70.7 -> 64.9 us per step)
          // (instantiated for X = 1 and for X = 2 with one feature slice, convert-once modes: d = 2n shapes only fit it at X = S = 1)
          if (bq == 1 && (x == 1 || (x == 2 && s == 1)) && !tm_perj(mode) && (int64_t)(zeta >= 8 ? 2 : 4) * cols <= kTmemCols / (NW / 4)) out->GM = 5;
          // tuning / tests (sketch_opts_t::tmem_group_mode): forced where the mode exists for this geometry
          if (gm_force == 0) out->GM = 0;   // chained groups exist for every geometry and mode
          if (mode == TM_F16 && gm_force >= 0 && bq > 1 && (gm_force == 0 || (gm_force == 1 && dbk >= 20) || (gm_force == 2 && dbk >= 72))) out->GM = gm_force;
        }
      }
    }
    if (found) return true;
  }
  return false;
}

size_t tmem_smem_bytes_for(int zeta, int n_cta, int bq, int gm, int mode) { return tmem_smem_bytes(zeta, n_cta, bq, gm, mode); }
int tmem_rows_per_stage(int n_cta, int bq, int zeta) { return tmem_stage_rows(n_cta, bq, zeta); }
int tmem_features_per_cta(const TmemShape& h, int mode) { return 32 * tm_fw(mode) * h.X * h.S; }

// 2-D tensor map over the row range: {n features, rows} FP32, row pitch lda, box {n_cta features, box_rows rows}.
// Limits (checked by tmem_tensor_map_ok, i.e. by the plan): coordinates are int32, the row pitch is a multiple of 16
// bytes below 2^40, a box side is at most 256 elements.
bool tmem_tensor_map_ok(int64_t lda, int64_t rows, int n_cta) {
  return rows <= 0x7FFFFFFFll && lda % 4 == 0 && lda * 4 < (1ll << 40) && n_cta <= 256;
}

cudaError_t tmem_make_tensor_map(const float* A, int n, int64_t lda, int64_t rows, int n_cta, int box_rows, CUtensorMap* out) {
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_fn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q);
    if (e != cudaSuccess) return e;
    if (q != cudaDriverEntryPointSuccess || !p) return cudaErrorNotSupported;
    fn = reinterpret_cast<encode_fn>(p);
  }
  const cuuint64_t dims[2] = {(cuuint64_t)n, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)lda * 4};
  const cuuint32_t box[2] = {(cuuint32_t)n_cta, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(A), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

#define SK_DECL(z, m) cudaError_t launch_tmem_z##z##_m##m(const TmemArgs&, const TmemShape&, const CUtensorMap&, int, cudaStream_t);
#define SK_DECL_Z(z) SK_DECL(z, 0) SK_DECL(z, 1) SK_DECL(z, 2) SK_DECL(z, 3) SK_DECL(z, 4)
SK_DECL_Z(1) SK_DECL_Z(2) SK_DECL_Z(4) SK_DECL_Z(8)

// tmap: the tensor map of this (A, n, lda, rows, geometry) when the tile is not contiguous (lda != n / CS), else ignored
cudaError_t launch_tmem(const TmemArgs& g, int zeta, int mode, const TmemShape& h, const CUtensorMap* tmap, int grid, cudaStream_t st) {
  if (mode < 0 || mode > 4 || tmem_features_per_cta(h, mode) * h.CS != g.s.n) return kNoKernel;
  static const CUtensorMap kNoMap = {};
  const CUtensorMap& tm = (g.s.lda != g.s.n / h.CS) ? *tmap : kNoMap;
  typedef cudaError_t (*fn_t)(const TmemArgs&, const TmemShape&, const CUtensorMap&, int, cudaStream_t);
#define SK_ROW(z) {launch_tmem_z##z##_m0, launch_tmem_z##z##_m1, launch_tmem_z##z##_m2, launch_tmem_z##z##_m3, launch_tmem_z##z##_m4}
  static const fn_t table[4][5] = {SK_ROW(1), SK_ROW(2), SK_ROW(4), SK_ROW(8)};
  const int zi = zeta == 1 ? 0 : zeta == 2 ? 1 : zeta == 4 ? 2 : zeta == 8 ? 3 : -1;
  if (zi < 0) return kNoKernel;
  return table[zi][mode](g, h, tm, grid, st);
}

}  // namespace sk
