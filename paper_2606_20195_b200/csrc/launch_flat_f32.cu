// launch_flat_f32.cu -- instantiations of the flat FP32 scatter (the in-library baseline) and the generic fallback.
#include "kernel_flat.cuh"
#include "launch.h"

namespace sk {
namespace {

template <int ZETA, int VEC>
cudaError_t go(const ScatterArgs& a, int pw, int grid, cudaStream_t st) {
  if (pw == 2) k_flat<ZETA, VEC, OUT_F32, RND_RN, uint16_t><<<grid, kFlatThreads, 0, st>>>(a);
  else if (pw == 4) k_flat<ZETA, VEC, OUT_F32, RND_RN, uint32_t><<<grid, kFlatThreads, 0, st>>>(a);
  else k_flat<ZETA, VEC, OUT_F32, RND_RN, uint8_t><<<grid, kFlatThreads, 0, st>>>(a);
  return cudaGetLastError();
}

template <int ZETA>
cudaError_t by_vec(const ScatterArgs& a, int vec, int pw, int grid, cudaStream_t st) {
  switch (vec) {
    case 4: return go<ZETA, 4>(a, pw, grid, st);
    case 2: return go<ZETA, 2>(a, pw, grid, st);
    case 1: return go<ZETA, 1>(a, pw, grid, st);
  }
  return kNoKernel;
}

}  // namespace

cudaError_t launch_flat_f32(const ScatterArgs& a, int zeta, int vec, int packed_width, int grid, cudaStream_t st) {
  switch (zeta) {
    case 1: return by_vec<1>(a, vec, packed_width, grid, st);
    case 2: return by_vec<2>(a, vec, packed_width, grid, st);
    case 4: return by_vec<4>(a, vec, packed_width, grid, st);
    case 8: return by_vec<8>(a, vec, packed_width, grid, st);
  }
  return kNoKernel;
}

cudaError_t launch_generic(const ScatterArgs& a, int out, int rounding, int grid, cudaStream_t st) {
  if (out == OUT_F32) k_generic<OUT_F32, RND_RN><<<grid, kFlatThreads, 0, st>>>(a);
  else if (out == OUT_BF16) k_generic<OUT_BF16, RND_RN><<<grid, kFlatThreads, 0, st>>>(a);
  else if (rounding == RND_SR) k_generic<OUT_F16, RND_SR><<<grid, kFlatThreads, 0, st>>>(a);
  else if (rounding == RND_DITHER) k_generic<OUT_F16, RND_DITHER><<<grid, kFlatThreads, 0, st>>>(a);
  else k_generic<OUT_F16, RND_RN><<<grid, kFlatThreads, 0, st>>>(a);
  return cudaGetLastError();
}

}  // namespace sk
