// launch_flat_f16.cu -- instantiations of the flat FP16 scatter: RN with on-the-fly or packed hashes, SR and dither
// (per-contribution conversion; hashes on the fly only).
#include "kernel_flat.cuh"
#include "launch.h"

namespace sk {
namespace {

template <int ZETA, int VEC, int RND>
cudaError_t go(const ScatterArgs& a, int pw, int grid, cudaStream_t st) {
  if constexpr (RND == RND_RN) {
    if (pw == 2) k_flat<ZETA, VEC, OUT_F16, RND, uint16_t><<<grid, kFlatThreads, 0, st>>>(a);
    else if (pw == 4) k_flat<ZETA, VEC, OUT_F16, RND, uint32_t><<<grid, kFlatThreads, 0, st>>>(a);
    else k_flat<ZETA, VEC, OUT_F16, RND, uint8_t><<<grid, kFlatThreads, 0, st>>>(a);
  } else {
    if (pw != 0) return kNoKernel;
    k_flat<ZETA, VEC, OUT_F16, RND, uint8_t><<<grid, kFlatThreads, 0, st>>>(a);
  }
  return cudaGetLastError();
}

template <int ZETA, int RND>
cudaError_t by_vec(const ScatterArgs& a, int vec, int pw, int grid, cudaStream_t st) {
  switch (vec) {
    case 8: return go<ZETA, 8, RND>(a, pw, grid, st);
    case 4: return go<ZETA, 4, RND>(a, pw, grid, st);
    case 2: return go<ZETA, 2, RND>(a, pw, grid, st);
  }
  return kNoKernel;
}

template <int RND>
cudaError_t by_zeta(const ScatterArgs& a, int zeta, int vec, int pw, int grid, cudaStream_t st) {
  switch (zeta) {
    case 1: return by_vec<1, RND>(a, vec, pw, grid, st);
    case 2: return by_vec<2, RND>(a, vec, pw, grid, st);
    case 4: return by_vec<4, RND>(a, vec, pw, grid, st);
    case 8: return by_vec<8, RND>(a, vec, pw, grid, st);
  }
  return kNoKernel;
}

}  // namespace

cudaError_t launch_flat_f16(const ScatterArgs& a, int zeta, int vec, int rounding, int packed_width, int grid,
                            cudaStream_t st) {
  switch (rounding) {
    case RND_RN: return by_zeta<RND_RN>(a, zeta, vec, packed_width, grid, st);
    case RND_SR: return by_zeta<RND_SR>(a, zeta, vec, packed_width, grid, st);
    case RND_DITHER: return by_zeta<RND_DITHER>(a, zeta, vec, packed_width, grid, st);
  }
  return kNoKernel;
}

}  // namespace sk
