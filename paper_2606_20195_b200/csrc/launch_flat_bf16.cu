// launch_flat_bf16.cu -- instantiations of the flat bfloat16 scatter (the BF16 control of PAPER.md:382, :396): RN
// conversion, red.global.add.noftz.bf16x2 in its 4-, 8- and 16-byte forms, hashes on the fly.
#include "kernel_flat.cuh"
#include "launch.h"

namespace sk {
namespace {

template <int ZETA>
cudaError_t by_vec(const ScatterArgs& a, int vec, int grid, cudaStream_t st) {
  switch (vec) {
    case 8: k_flat<ZETA, 8, OUT_BF16, RND_RN, uint8_t><<<grid, kFlatThreads, 0, st>>>(a); break;
    case 4: k_flat<ZETA, 4, OUT_BF16, RND_RN, uint8_t><<<grid, kFlatThreads, 0, st>>>(a); break;
    case 2: k_flat<ZETA, 2, OUT_BF16, RND_RN, uint8_t><<<grid, kFlatThreads, 0, st>>>(a); break;
    default: return kNoKernel;
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_flat_bf16(const ScatterArgs& a, int zeta, int vec, int grid, cudaStream_t st) {
  switch (zeta) {
    case 1: return by_vec<1>(a, vec, grid, st);
    case 2: return by_vec<2>(a, vec, grid, st);
    case 4: return by_vec<4>(a, vec, grid, st);
    case 8: return by_vec<8>(a, vec, grid, st);
  }
  return kNoKernel;
}

}  // namespace sk
