// launch.h -- host-side launchers, one translation unit per kernel family so nvcc compiles them in parallel.
// Each returns the launch status (cudaGetLastError), or kNoKernel when no instantiation exists for the combination
// -- the host-side plan rules those out before anything is launched, so seeing it is an internal error.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>

#include "args.h"

namespace sk {

constexpr cudaError_t kNoKernel = cudaErrorInvalidDeviceFunction;

// Raise a kernel's dynamic-shared-memory limit to the device's opt-in maximum, once per (kernel, device): the hot
// call then does no cudaFuncSetAttribute (SURVEY 8b "never allocates per call"; a captured stream sees launches only).
template <auto Kernel>
inline cudaError_t allow_max_dynamic_smem() {
  static std::atomic<uint64_t> done{0};   // bit per device ordinal
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 64 && ((done.load(std::memory_order_acquire) >> dev) & 1ull)) return cudaSuccess;
  int optin = 0;
  e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(Kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, optin);
  if (e == cudaSuccess && dev < 64) done.fetch_or(1ull << dev, std::memory_order_release);
  return e;
}

cudaError_t launch_flat_f16(const ScatterArgs& a, int zeta, int vec, int rounding, int packed_width, int grid,
                            cudaStream_t st);
cudaError_t launch_flat_f32(const ScatterArgs& a, int zeta, int vec, int packed_width, int grid, cudaStream_t st);
cudaError_t launch_flat_bf16(const ScatterArgs& a, int zeta, int vec, int grid, cudaStream_t st);
cudaError_t launch_generic(const ScatterArgs& a, int out /* OUT_* */, int rounding /* RND_* */, int grid, cudaStream_t st);

// shared-memory-privatised FP16-RN scatter; wpc = warps per CTA = n / 64
cudaError_t launch_smem_f16(const SmemArgs& g, int zeta, int wpc, int grid, size_t smem_bytes, cudaStream_t st);
int smem_ring_rows(int zeta, int wpc);  // rows one loop iteration (one load batch) of that instantiation covers
int smem_step_rows(int zeta);           // R: rows per step; row ranges given to the kernel start at a multiple of it
// a1 precomputed: 16-bit entries (bucket | sign<<15), index row*zeta + t for block (row mod R + t) mod zeta
cudaError_t launch_hash_pack_rot(uint64_t seed, int zeta, int64_t rows, uint32_t db, uint16_t* out, int grid,
                                 cudaStream_t st);
int smem_max_bucket();
// per-warp shared-memory partials for small inputs / narrow matrices (kernel_small.cuh); smem = warps * d * n * 2 bytes
cudaError_t launch_small_f16(const SmallArgs& g, int zeta, int grid, size_t smem_bytes, cudaStream_t st);
int small_warps();

// tensor-memory-privatised scatter (kernel_tmem.cuh).  mode = TM_* (FP16-RN, bfloat16, FP16 with SR / dither, FP32
// accumulate).  Geometry: n = 32 FW X S CS with FW = 2 (16-bit modes) or 1 (FP32) features per tensor-memory word; a lane
// holds X words, S feature slices and BQ bucket groups per CTA, CS column slices across CTAs (gridDim.y), NW consumer
// warps.  tmem_shape picks it, returns false when no geometry fits the 512 TMEM columns of a warp's lane quadrant.
struct TmemShape {
  int X, S, BQ, CS, NW, GM;
};
bool tmem_shape(int n, int d, int zeta, int64_t lda, int gm_force /* -1 = auto */, int mode, TmemShape* out);
bool tmem_tensor_map_ok(int64_t lda, int64_t rows, int n_cta);
cudaError_t tmem_make_tensor_map(const float* A, int n, int64_t lda, int64_t rows, int n_cta, int box_rows, CUtensorMap* out);
size_t tmem_smem_bytes_for(int zeta, int n_cta, int bq, int gm, int mode);  // n_cta = n / CS
int tmem_rows_per_stage(int n_cta, int bq, int zeta);
int tmem_features_per_cta(const TmemShape& h, int mode);
cudaError_t launch_tmem(const TmemArgs& g, int zeta, int mode, const TmemShape& h, const CUtensorMap* tmap, int grid, cudaStream_t st);

}  // namespace sk
