// launch_tmem.cu -- instantiations of the tensor-memory-privatised scatter.  Compiled once per zeta
// (-DSK_TMEM_ZETA=1|2|4|8) so the four families build in parallel; the zeta = 4 unit also holds the
// shape logic and the dispatcher.
#include <cstring>

#include "kernel_tmem.cuh"
#include "launch.h"

#ifndef SK_TMEM_ZETA
#error "compile with -DSK_TMEM_ZETA=<1|2|4|8>"
#endif

namespace sk {
namespace {

template <int X, int S, int BQ, int NW, int GM>
cudaError_t go(const TmemArgs& g, const CUtensorMap& tmap, int grid, int cs, cudaStream_t st) {
  constexpr int Z = SK_TMEM_ZETA, N = 64 * X * S;
  if constexpr (Z % BQ != 0) {
    return kNoKernel;
  } else {
    constexpr auto k = k_tmem<Z, X, S, BQ, NW, GM>;
    const size_t smem = tmem_smem_bytes(Z, N, BQ, GM);
    cudaError_t e = allow_max_dynamic_smem<k>();
    if (e != cudaSuccess) return e;
    k<<<dim3((unsigned)grid, (unsigned)cs), (NW + tmem_producers(N, BQ, GM, Z)) * 32, smem, st>>>(g, tmap);
    return cudaGetLastError();
  }
}

cudaError_t dispatch(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st) {
  if (h.NW == 4) {
    switch (h.X * 100 + h.S * 10 + h.BQ) {
      case 111: return go<1, 1, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 121: return go<1, 2, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 141: return go<1, 4, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 211: return go<2, 1, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 221: return go<2, 2, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 241: return go<2, 4, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 411: return go<4, 1, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 421: return go<4, 2, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 441: return go<4, 4, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 112: return h.GM == 1 ? go<1, 1, 2, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<1, 1, 2, 4, 2>(g, tmap, grid, h.CS, st) : go<1, 1, 2, 4, 0>(g, tmap, grid, h.CS, st);
      case 122: return h.GM == 1 ? go<1, 2, 2, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<1, 2, 2, 4, 2>(g, tmap, grid, h.CS, st) : go<1, 2, 2, 4, 0>(g, tmap, grid, h.CS, st);
      case 212: return h.GM == 1 ? go<2, 1, 2, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<2, 1, 2, 4, 2>(g, tmap, grid, h.CS, st) : go<2, 1, 2, 4, 0>(g, tmap, grid, h.CS, st);
      case 222: return h.GM == 1 ? go<2, 2, 2, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<2, 2, 2, 4, 2>(g, tmap, grid, h.CS, st) : go<2, 2, 2, 4, 0>(g, tmap, grid, h.CS, st);
      case 412: return h.GM == 1 ? go<4, 1, 2, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<4, 1, 2, 4, 2>(g, tmap, grid, h.CS, st) : go<4, 1, 2, 4, 0>(g, tmap, grid, h.CS, st);
      case 422: return h.GM == 1 ? go<4, 2, 2, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<4, 2, 2, 4, 2>(g, tmap, grid, h.CS, st) : go<4, 2, 2, 4, 0>(g, tmap, grid, h.CS, st);
      case 114: return h.GM == 1 ? go<1, 1, 4, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<1, 1, 4, 4, 2>(g, tmap, grid, h.CS, st) : go<1, 1, 4, 4, 0>(g, tmap, grid, h.CS, st);
      case 214: return h.GM == 1 ? go<2, 1, 4, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<2, 1, 4, 4, 2>(g, tmap, grid, h.CS, st) : go<2, 1, 4, 4, 0>(g, tmap, grid, h.CS, st);
      case 414: return h.GM == 1 ? go<4, 1, 4, 4, 1>(g, tmap, grid, h.CS, st) : h.GM == 2 ? go<4, 1, 4, 4, 2>(g, tmap, grid, h.CS, st) : go<4, 1, 4, 4, 0>(g, tmap, grid, h.CS, st);
    }
  }
  return kNoKernel;
}

}  // namespace

#if SK_TMEM_ZETA == 1
cudaError_t launch_tmem_z1(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st) { return dispatch(g, h, tmap, grid, st); }
#elif SK_TMEM_ZETA == 2
cudaError_t launch_tmem_z2(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st) { return dispatch(g, h, tmap, grid, st); }
#elif SK_TMEM_ZETA == 8
cudaError_t launch_tmem_z8(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st) { return dispatch(g, h, tmap, grid, st); }
#elif SK_TMEM_ZETA == 4
cudaError_t launch_tmem_z4(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st) { return dispatch(g, h, tmap, grid, st); }

// Geometry for an n-feature, d-row, zeta-block sketch: the fewest column slices CS that fit at all, then
// the (X, S, BQ) with the fewest issued instructions per KiB of A.  Model (from the SASS of the main loop,
// profiles/r01_tmem_shapes.md): a row slice of 256 X bytes costs 1 + 3 X instructions to load and convert
// (in each of the BQ warps that need it) and 5.25 + 2 X per stack block to read-modify-write.
bool tmem_shape(int n, int d, int zeta, int64_t lda, int gm_force, TmemShape* out) {
  if (n <= 0 || d <= 0 || zeta <= 0 || n % 64 != 0 || d % zeta != 0) return false;
  const int NW = 4;
  for (int cs = 1; cs <= 16; ++cs) {   // odd slice counts serve the widths that are not 64 * 2^k (192, 320, 384, ...)
    if (n % (64 * cs) != 0) continue;
    const int nc = n / cs;
    if (lda != nc && nc > 256) continue;   // strided tiles come through a tensor-map box of at most 256 elements a side
    double best = 0.0;
    bool found = false;
    for (int x = 4; x >= 1; x >>= 1) {
      if (nc % (64 * x) != 0) continue;
      const int s = nc / (64 * x);
      if (s != 1 && s != 2 && s != 4) continue;
      for (int bq = 1; bq <= 4; bq *= 2) {
        if (s * bq > NW || zeta % bq != 0 || d % bq != 0) continue;
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
          const double zb = (double)zeta / bq, dbk = (double)d / zeta;
          out->GM = (bq == 4 && zb * 6.0 / dbk <= 0.15 && dbk >= 20) ? 1 : 0;
          // tuning / tests (sketch_opts_t::tmem_group_mode): forced where the mode exists for this geometry
          if (gm_force >= 0 && bq > 1 && (gm_force == 0 || (gm_force == 1 && dbk >= 20) || (gm_force == 2 && dbk >= 72))) out->GM = gm_force;
        }
      }
    }
    if (found) return true;
  }
  return false;
}

size_t tmem_smem_bytes_for(int zeta, int n_cta, int bq, int gm) { return tmem_smem_bytes(zeta, n_cta, bq, gm); }
int tmem_rows_per_stage(int n_cta, int bq, int zeta) { return tmem_stage_rows(n_cta, bq, zeta); }

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

// tmap: the tensor map of this (A, n, lda, rows, geometry) when the tile is not contiguous (lda != n / CS), else ignored
cudaError_t launch_tmem_f16(const TmemArgs& g, int zeta, const TmemShape& h, const CUtensorMap* tmap, int grid, cudaStream_t st) {
  if (64 * h.X * h.S * h.CS != g.s.n) return kNoKernel;
  static const CUtensorMap kNoMap = {};
  const CUtensorMap& tm = (g.s.lda != g.s.n / h.CS) ? *tmap : kNoMap;
  switch (zeta) {
    case 1: return launch_tmem_z1(g, h, tm, grid, st);
    case 2: return launch_tmem_z2(g, h, tm, grid, st);
    case 4: return launch_tmem_z4(g, h, tm, grid, st);
    case 8: return launch_tmem_z8(g, h, tm, grid, st);
  }
  return kNoKernel;
}
#endif

}  // namespace sk
