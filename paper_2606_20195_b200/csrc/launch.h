// launch.h -- host-side launchers, one translation unit per kernel family so nvcc compiles them in parallel.
// Each returns the launch status (cudaGetLastError) or cudaErrorInvalidValue for an unsupported combination.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include "args.h"

namespace sk {

cudaError_t launch_flat_f16(const ScatterArgs& a, int zeta, int vec, int rounding, int packed_width, int grid,
                            cudaStream_t st);
cudaError_t launch_flat_f32(const ScatterArgs& a, int zeta, int vec, int packed_width, int grid, cudaStream_t st);
cudaError_t launch_generic(const ScatterArgs& a, bool f16, int rounding, int grid, cudaStream_t st);

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

// tensor-memory-privatised FP16-RN scatter (kernel_tmem.cuh).  Geometry: n = 64 * X * S * CS; lane holds X half2
// words, S feature slices and BQ bucket groups per CTA, CS column slices across CTAs (gridDim.y), NW consumer warps.
// tmem_shape picks it, returns false when no geometry fits the 512 TMEM columns of a warp's lane quadrant.
struct TmemShape {
  int X, S, BQ, CS, NW, GM;
};
bool tmem_shape(int n, int d, int zeta, int64_t lda, TmemShape* out);
size_t tmem_smem_bytes_for(int zeta, int n_cta, int bq, int gm);  // n_cta = n / CS
int tmem_rows_per_stage(int n_cta, int bq, int zeta);
cudaError_t launch_tmem_f16(const TmemArgs& g, int zeta, const TmemShape& h, int grid, cudaStream_t st);
cudaError_t launch_tmem_z1(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st);
cudaError_t launch_tmem_z2(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st);
cudaError_t launch_tmem_z4(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st);
cudaError_t launch_tmem_z8(const TmemArgs& g, const TmemShape& h, const CUtensorMap& tmap, int grid, cudaStream_t st);

}  // namespace sk
