// launch_smem.cu -- instantiations of the shared-memory-privatised scatter and its hash-pack kernel.
#include "kernel_small.cuh"
#include "kernel_smem.cuh"
#include "launch.h"

namespace sk {
namespace {

template <int ZETA>
cudaError_t go(const SmemArgs& g, int wpc, int grid, size_t smem_bytes, cudaStream_t st) {
  cudaError_t e;
  if (wpc <= 4) {
    constexpr auto k = k_smem<ZETA, smem_batch_steps(ZETA, true), 4>;
    e = allow_max_dynamic_smem<k>();
    if (e != cudaSuccess) return e;
    k<<<grid, wpc * 32, smem_bytes, st>>>(g);
  } else {
    constexpr auto k = k_smem<ZETA, smem_batch_steps(ZETA, false), 16>;
    e = allow_max_dynamic_smem<k>();
    if (e != cudaSuccess) return e;
    k<<<grid, wpc * 32, smem_bytes, st>>>(g);
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t launch_smem_f16(const SmemArgs& g, int zeta, int wpc, int grid, size_t smem_bytes, cudaStream_t st) {
  switch (zeta) {
    case 1: return go<1>(g, wpc, grid, smem_bytes, st);
    case 2: return go<2>(g, wpc, grid, smem_bytes, st);
    case 4: return go<4>(g, wpc, grid, smem_bytes, st);
    case 8: return go<8>(g, wpc, grid, smem_bytes, st);
  }
  return kNoKernel;
}

namespace {
template <int ZETA>
cudaError_t go_small(const SmallArgs& g, int grid, size_t smem_bytes, cudaStream_t st) {
  constexpr auto k = k_small<ZETA>;
  if (smem_bytes > 48 * 1024) {
    cudaError_t e = allow_max_dynamic_smem<k>();
    if (e != cudaSuccess) return e;
  }
  k<<<grid, kSmallWarps * 32, smem_bytes, st>>>(g);
  return cudaGetLastError();
}
}  // namespace

cudaError_t launch_small_f16(const SmallArgs& g, int zeta, int grid, size_t smem_bytes, cudaStream_t st) {
  switch (zeta) {
    case 1: return go_small<1>(g, grid, smem_bytes, st);
    case 2: return go_small<2>(g, grid, smem_bytes, st);
    case 4: return go_small<4>(g, grid, smem_bytes, st);
    case 8: return go_small<8>(g, grid, smem_bytes, st);
  }
  return kNoKernel;
}
int small_warps() { return kSmallWarps; }

int smem_ring_rows(int zeta, int wpc) { return smem_rows_per_step(zeta) * smem_batch_steps(zeta, wpc <= 4); }
int smem_step_rows(int zeta) { return smem_rows_per_step(zeta); }
int smem_max_bucket() { return kSmemMaxBucket; }

cudaError_t launch_hash_pack_rot(uint64_t seed, int zeta, int64_t rows, uint32_t db, uint16_t* out, int grid,
                                 cudaStream_t st) {
  switch (zeta) {
    case 1: k_hash_pack_rot<1><<<grid, 256, 0, st>>>(seed, rows, db, out); break;
    case 2: k_hash_pack_rot<2><<<grid, 256, 0, st>>>(seed, rows, db, out); break;
    case 4: k_hash_pack_rot<4><<<grid, 256, 0, st>>>(seed, rows, db, out); break;
    case 8: k_hash_pack_rot<8><<<grid, 256, 0, st>>>(seed, rows, db, out); break;
    default: return kNoKernel;
  }
  return cudaGetLastError();
}

}  // namespace sk
