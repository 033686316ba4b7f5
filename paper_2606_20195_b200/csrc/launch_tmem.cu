// launch_tmem.cu -- instantiations of the tensor-memory-privatised scatter.  Compiled once per (zeta, mode)
// (-DSK_TMEM_ZETA=1|2|4|8 -DSK_TMEM_MODE=0..4, kernel_tmem.cuh: TM_*) so the twenty families build in parallel; the shape
// logic and the dispatcher over these units live in tmem_host.cu.
#include "kernel_tmem.cuh"
#include "launch.h"

#if !defined(SK_TMEM_ZETA) || !defined(SK_TMEM_MODE)
#error "compile with -DSK_TMEM_ZETA=<1|2|4|8> -DSK_TMEM_MODE=<0..4>"
#endif

namespace sk {
namespace {

constexpr int Z = SK_TMEM_ZETA, MODE = SK_TMEM_MODE;

template <int X, int S, int BQ, int NW, int GM>
cudaError_t go(const TmemArgs& g, const CUtensorMap& tmap, int grid, int cs, cudaStream_t st) {
  constexpr int N = 32 * tm_fw(MODE) * X * S;
  if constexpr (Z % BQ != 0 || ((GM == 1 || GM == 2) && MODE != TM_F16) || (tm_perj(MODE) && (BQ != 1 || GM == 5))) {
    return kNoKernel;
  } else {
    constexpr auto k = k_tmem<Z, X, S, BQ, NW, GM, MODE>;
    const size_t smem = tmem_smem_bytes(Z, N, BQ, GM, MODE);
    cudaError_t e = allow_max_dynamic_smem<k>();
    if (e != cudaSuccess) return e;
    // one more warp when a right-hand side rides along (kernel_tmem.cuh: the right-hand-side warp)
    k<<<dim3((unsigned)grid, (unsigned)cs), (NW + tmem_producers(N, BQ, GM, Z) + (g.rhs != nullptr ? 1 : 0)) * 32, smem, st>>>(g, tmap);
    return cudaGetLastError();
  }
}

template <int X, int S, int BQ>
cudaError_t by_gm(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st) {
  if (h.GM == 1) return go<X, S, BQ, 4, 1>(g, tmap, grid, h.CS, st);
  if (h.GM == 2) return go<X, S, BQ, 4, 2>(g, tmap, grid, h.CS, st);
  return go<X, S, BQ, 4, 0>(g, tmap, grid, h.CS, st);
}

cudaError_t dispatch(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st) {
  if (h.NW == 4) {
    switch (h.X * 100 + h.S * 10 + h.BQ) {
      case 111: return h.GM == 5 ? go<1, 1, 1, 4, 5>(g, tmap, grid, h.CS, st) : go<1, 1, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 121: return h.GM == 5 ? go<1, 2, 1, 4, 5>(g, tmap, grid, h.CS, st) : go<1, 2, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 141: return h.GM == 5 ? go<1, 4, 1, 4, 5>(g, tmap, grid, h.CS, st) : go<1, 4, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 211: return h.GM == 5 ? go<2, 1, 1, 4, 5>(g, tmap, grid, h.CS, st) : go<2, 1, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 221: return go<2, 2, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 241: return go<2, 4, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 411: return go<4, 1, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 421: return go<4, 2, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 441: return go<4, 4, 1, 4, 0>(g, tmap, grid, h.CS, st);
      case 112: return by_gm<1, 1, 2>(g, h, tmap, grid, st);
      case 122: return by_gm<1, 2, 2>(g, h, tmap, grid, st);
      case 212: return by_gm<2, 1, 2>(g, h, tmap, grid, st);
      case 222: return by_gm<2, 2, 2>(g, h, tmap, grid, st);
      case 412: return by_gm<4, 1, 2>(g, h, tmap, grid, st);
      case 422: return by_gm<4, 2, 2>(g, h, tmap, grid, st);
      case 114: return by_gm<1, 1, 4>(g, h, tmap, grid, st);
      case 214: return by_gm<2, 1, 4>(g, h, tmap, grid, st);
      case 414: return by_gm<4, 1, 4>(g, h, tmap, grid, st);
    }
  }
  return kNoKernel;
}

}  // namespace

#define SK_CAT4_(a, b, c, d) a##b##c##d
#define SK_CAT4(a, b, c, d) SK_CAT4_(a, b, c, d)
cudaError_t SK_CAT4(launch_tmem_z, SK_TMEM_ZETA, _m, SK_TMEM_MODE)(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid,
                                                                   cudaStream_t st) {
  return dispatch(g, h, tmap, grid, st);
}

}  // namespace sk
