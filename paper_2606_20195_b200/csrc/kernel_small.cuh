// kernel_small.cuh -- shared-memory-privatised FP16-RN scatter for SMALL inputs and narrow matrices (any even n).
//
// BASELINE config 1 (m = 4096, n = 16, d = 32) is launch-bound for every kernel, but the flat scatter is worse than
// that: its zeta*m*n/2 half2 updates land in a 1 KiB sketch, i.e. ~1000 REDs queue on each 32-byte L2 sector
// (measured 10 us per sketch, 4 us of it this serialisation; profiles/r01_variant_sweep.md).  Here every warp keeps a
// private partial sketch [d][n/2] of half2 words in shared memory (PAPER.md:114-136 restated per warp):
//   hashes   one lane per (row, block) of a batch of 8 rows (a1), broadcast with a shuffle; two batches per step so
//            that 16 row loads are in flight together;
//   scatter  lane <-> (block jj, column pair): the ZETA blocks of a row own disjoint sketch rows, so
//            the 32 words one instruction touches are pairwise distinct; a lane meets "its" word again only in a later
//            row, in program order -- plain LDS / HFMA2 (q*(+-1)+acc = one RN16 add per half) / STS;
//   flush    the CTA's 8 partials are added word by word (FP16 adds) and sent to B with result-discarding REDs
//            (PAPER.md:175-187); B was zero-initialised by the caller's memset (a0).
#pragma once

#include "args.h"
#include "device_util.cuh"

namespace sk {

constexpr int kSmallWarps = 8;

SK_DEVINL uint32_t small_hfma2(uint32_t q, uint32_t mult, uint32_t acc) {
  uint32_t d;
  asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(q), "r"(mult), "r"(acc));
  return d;
}
SK_DEVINL uint32_t small_hadd2(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("add.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}

template <int ZETA>
__global__ void __launch_bounds__(kSmallWarps * 32) k_small(SmallArgs g) {
  constexpr int RB = ZETA == 8 ? 4 : 8;   // rows per hash batch (RB * ZETA <= 32 hashing lanes)
  constexpr int NB = 2;                   // batches whose loads are in flight together
  constexpr int PP = 32 / ZETA;           // column pairs per pass
  extern __shared__ uint32_t part[];      // [kSmallWarps][d * n/2]
  const ScatterArgs& a = g.s;
  const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint32_t pairs = (uint32_t)a.n / 2, words = (uint32_t)g.d * pairs;
  uint32_t* const mine = part + warp * words;
  for (uint32_t k = lane; k < words; k += 32) mine[k] = 0u;
  __syncwarp();

  const int64_t w0 = ((int64_t)blockIdx.x * kSmallWarps + warp) * g.rows_per_warp;
  const int64_t w1 = min(a.rows, w0 + g.rows_per_warp);
  const uint32_t jj = lane / PP, pl = lane % PP;
  for (int64_t r0 = w0; r0 < w1; r0 += NB * RB) {
    // a1: lane <-> (row r0 + t * RB + lane / ZETA, block lane % ZETA) of batch t
    uint32_t e[NB];
#pragma unroll
    for (int t = 0; t < NB; ++t) {
      const int64_t hr = r0 + t * RB + lane / ZETA;
      e[t] = (lane < RB * ZETA && hr < w1) ? hash_entry(a.seed, (uint64_t)(a.row_begin + hr) * ZETA + lane % ZETA, lane % ZETA, a.db) : 0u;
    }
    for (uint32_t p0 = 0; p0 < pairs; p0 += PP) {
      const uint32_t pair = p0 + pl;
      float2 v[NB * RB];
#pragma unroll
      for (int b = 0; b < NB * RB; ++b) {       // a2: all loads of the step first (latency)
        v[b] = make_float2(0.f, 0.f);
        if (pair < pairs && r0 + b < w1) v[b] = __ldg(reinterpret_cast<const float2*>(a.A + (r0 + b) * a.lda) + pair);
      }
#pragma unroll
      for (int b = 0; b < NB * RB; ++b) {
        const uint32_t eb = __shfl_sync(0xFFFFFFFFu, e[b / RB], (b % RB) * ZETA + jj);
        if (pair < pairs && r0 + b < w1) {
          const uint32_t q = pack_rn(v[b].x * a.scale, v[b].y * a.scale);   // a3, a4
          uint32_t* const w = mine + entry_bucket(eb) * pairs + pair;
          *w = small_hfma2(q, 0x3C003C00u ^ entry_signmask_h2(eb), *w);     // a5
        }
      }
    }
  }
  __syncthreads();
  uint32_t* const B = reinterpret_cast<uint32_t*>(a.B);
  for (uint32_t k = threadIdx.x; k < words; k += kSmallWarps * 32) {
    uint32_t acc = part[k];
#pragma unroll
    for (int w = 1; w < kSmallWarps; ++w) acc = small_hadd2(acc, part[w * words + k]);
    if (acc != 0u) red_h2(B + k, acc);
  }
}

}  // namespace sk
