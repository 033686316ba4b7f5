// kernel_misc.cuh -- small kernels around the scatter (include from exactly one translation unit):
//   k_hash_dump / k_hash_pack32   a1  hash stage (dump for tests; plain 32-bit packed array)
//   k_reduce_replicas<...>        folds the P L2-resident partial sketches of the flat variant
//   k_red_probe<...>              L2 atomic-throughput microbenchmark (roofline term 2)
//   k_convert_probe               a4 in isolation: RN / SR / dither / bfloat16 / the hardware cvt.rs, element by element
#pragma once

#include "args.h"
#include "device_util.cuh"
#include "kernel_tmem.cuh"   // mbarrier / TMA wrappers for the streaming probe

namespace sk {

// ------------------------------------------------------------------------------------------------
// a1: hash stage as stand-alone kernels
// ------------------------------------------------------------------------------------------------
__global__ void k_hash_dump(uint64_t seed, int64_t total, uint32_t zeta, uint32_t db, int32_t* __restrict__ bucket,
                            uint8_t* __restrict__ signbit) {
  int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += stride) {
    uint32_t j = (uint32_t)(idx % zeta);
    uint32_t e = hash_entry(seed, (uint64_t)idx, j, db);
    bucket[idx] = (int32_t)entry_bucket(e);
    signbit[idx] = (uint8_t)(e >> 31);
  }
}

// plain 32-bit packed entries (bucket | sign<<31) for sketches whose d does not fit the ranked 16-bit form
__global__ void k_hash_pack32(uint64_t seed, int64_t total, uint32_t zeta, uint32_t db, uint32_t* __restrict__ packed) {
  int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += stride)
    packed[idx] = hash_entry(seed, (uint64_t)idx, (uint32_t)(idx % zeta), db);
}

// ------------------------------------------------------------------------------------------------
// Fold P partial sketches.  FP16: sequential RN16 adds in replica order (every accumulation of the
// FP16 path stays an FP16 RN add, "All policies subsequently use RN atomic addition");
// FP32: float adds.  accumulate != 0 adds the fold into the existing out.
// ------------------------------------------------------------------------------------------------
template <int OUT>
__global__ void k_reduce_replicas(const void* __restrict__ rep, int64_t replica_stride, int32_t replicas, void* __restrict__ out,
                                  int64_t count, int accumulate) {
  int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < count; k += stride) {
    if constexpr (OUT == OUT_F16) {
      const __half* r = reinterpret_cast<const __half*>(rep);
      __half* o = reinterpret_cast<__half*>(out);
      __half acc = accumulate ? o[k] : __ushort_as_half(0);
      for (int p = 0; p < replicas; ++p) acc = __hadd(acc, r[(int64_t)p * replica_stride + k]);
      o[k] = acc;
    } else if constexpr (OUT == OUT_BF16) {
      const __nv_bfloat16* r = reinterpret_cast<const __nv_bfloat16*>(rep);
      __nv_bfloat16* o = reinterpret_cast<__nv_bfloat16*>(out);
      __nv_bfloat16 acc = accumulate ? o[k] : __ushort_as_bfloat16(0);
      for (int p = 0; p < replicas; ++p) acc = __hadd(acc, r[(int64_t)p * replica_stride + k]);
      o[k] = acc;
    } else {
      const float* r = reinterpret_cast<const float*>(rep);
      float* o = reinterpret_cast<float*>(out);
      float acc = accumulate ? o[k] : 0.f;
      for (int p = 0; p < replicas; ++p) acc = __fadd_rn(acc, r[(int64_t)p * replica_stride + k]);
      o[k] = acc;
    }
  }
}

// exact widening of a 16-bit sketch to FP32 (PAPER.md:356 "widen FP16 SA exactly"; :312 "layout/promotion")
template <int OUT>
__global__ void k_widen(const uint16_t* __restrict__ in, int64_t count, float* __restrict__ out) {
  int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < count; k += stride)
    out[k] = OUT == OUT_BF16 ? __bfloat162float(__ushort_as_bfloat16(in[k])) : __half2float(__ushort_as_half(in[k]));
}

// ------------------------------------------------------------------------------------------------
// L2 atomic-throughput probe: same address pattern as k_flat (a random bucket row per lane group of
// n/VEC lanes, consecutive lanes on consecutive VEC-column chunks), values from registers, no A loads.
// ------------------------------------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(kFlatThreads) k_red_probe(void* sketch, int32_t d, int32_t n, int32_t replicas, int32_t iters) {
  constexpr bool F16 = KIND < 3;
  constexpr int VEC = (KIND == 0) ? 2 : (KIND == 1) ? 4 : (KIND == 2) ? 8 : (KIND == 3) ? 1 : (KIND == 4) ? 2 : 4;
  const uint32_t cpr = (uint32_t)n / VEC;
  const uint64_t gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const uint64_t gthreads = (uint64_t)gridDim.x * blockDim.x;
  char* base = reinterpret_cast<char*>(sketch) + (size_t)(blockIdx.x % replicas) * (size_t)d * n * (F16 ? 2 : 4);
  const uint32_t ch = (uint32_t)(gtid % cpr);
  const uint64_t grp = gtid / cpr;
  const uint64_t ngrp = (gthreads + cpr - 1) / cpr;
  for (int32_t it = 0; it < iters; ++it) {
    uint64_t h = splitmix64(grp + (uint64_t)it * ngrp);
    uint32_t bucket = __umulhi((uint32_t)(h >> 32), (uint32_t)d);
    size_t off = (size_t)bucket * n + (size_t)ch * VEC;
    uint32_t hv = (h & 1) ? 0x3C003C00u : 0xBC00BC00u;  // +-1.0 pairs: sums stay small
    float fv = (h & 1) ? 1.f : -1.f;
    if constexpr (KIND == 0) red_h2(reinterpret_cast<__half*>(base) + off, hv);
    else if constexpr (KIND == 1) red_h4(reinterpret_cast<__half*>(base) + off, hv, hv);
    else if constexpr (KIND == 2) red_h8(reinterpret_cast<__half*>(base) + off, hv, hv, hv, hv);
    else if constexpr (KIND == 3) red_f1(reinterpret_cast<float*>(base) + off, fv);
    else if constexpr (KIND == 4) red_f2(reinterpret_cast<float*>(base) + off, fv, fv);
    else red_f4(reinterpret_cast<float*>(base) + off, fv, fv, fv, fv);
  }
}

// Candidates for sketches beyond tensor memory, same address pattern, no A loads:
//   KIND 6  owner-exclusive plain read-modify-write in L2: ld.global.cg.v4 -> 4 x HADD2 -> st.global.cg.v4 (16 bytes per
//           lane; hazards between lanes ignored -- an upper bound for any non-atomic L2-resident replica design)
//   KIND 7/8  TMA bulk reduction: one elected lane per warp issues cp.reduce.async.bulk.global.shared::cta ... add of a
//           whole converted row slice (`chunk` bytes of FP16 / FP32 words from shared memory) onto a random sketch row;
//           no per-lane RED instructions at all, so whatever limits it is the L2 side alone
template <int KIND>
__global__ void __launch_bounds__(kFlatThreads) k_l2_probe(void* sketch, int32_t d, int32_t n, int32_t replicas, int32_t iters, int32_t chunk) {
  constexpr int EB = KIND == 8 ? 4 : 2;
  char* base = reinterpret_cast<char*>(sketch) + (size_t)(blockIdx.x % replicas) * (size_t)d * n * EB;
  if constexpr (KIND == 6) {
    const uint32_t cpr = (uint32_t)n / 8;
    const uint64_t gtid = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint64_t gthreads = (uint64_t)gridDim.x * blockDim.x;
    const uint32_t ch = (uint32_t)(gtid % cpr);
    const uint64_t grp = gtid / cpr, ngrp = (gthreads + cpr - 1) / cpr;
    for (int32_t it = 0; it < iters; ++it) {
      uint64_t h = splitmix64(grp + (uint64_t)it * ngrp);
      uint32_t bucket = __umulhi((uint32_t)(h >> 32), (uint32_t)d);
      uint4* p = reinterpret_cast<uint4*>(base + ((size_t)bucket * n + (size_t)ch * 8) * 2);
      const uint32_t hv = (h & 1) ? 0x3C003C00u : 0xBC00BC00u;
      uint4 v;
      asm volatile("ld.global.cg.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
      asm("add.rn.f16x2 %0, %0, %1;" : "+r"(v.x) : "r"(hv));
      asm("add.rn.f16x2 %0, %0, %1;" : "+r"(v.y) : "r"(hv));
      asm("add.rn.f16x2 %0, %0, %1;" : "+r"(v.z) : "r"(hv));
      asm("add.rn.f16x2 %0, %0, %1;" : "+r"(v.w) : "r"(hv));
      asm volatile("st.global.cg.v4.b32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
    }
  } else {
    extern __shared__ __align__(128) unsigned char probe_smem[];   // [2][chunk]: a row slice of +1 and one of -1
    const uint32_t words = (uint32_t)chunk / 4;
    for (uint32_t k = threadIdx.x; k < 2 * words; k += blockDim.x)
      reinterpret_cast<uint32_t*>(probe_smem)[k] = KIND == 7 ? (k < words ? 0x3C003C00u : 0xBC00BC00u) : (k < words ? 0x3F800000u : 0xBF800000u);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    const uint32_t src = (uint32_t)__cvta_generic_to_shared(probe_smem);
    const uint32_t per_row = (uint32_t)n * EB / (uint32_t)chunk;          // chunks per sketch row
    const uint64_t gw = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = ((uint64_t)gridDim.x * blockDim.x) >> 5;
    if ((threadIdx.x & 31) == 0) {
      for (int32_t it = 0; it < iters; ++it) {
        uint64_t h = splitmix64(gw + (uint64_t)it * nw);
        uint32_t bucket = __umulhi((uint32_t)(h >> 32), (uint32_t)d);
        char* dst = base + (size_t)bucket * n * EB + (size_t)((uint32_t)(h >> 8) % per_row) * chunk;
        const uint32_t s = src + ((h & 1) ? (uint32_t)chunk : 0u);
        if constexpr (KIND == 7)
          asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.noftz.f16 [%0], [%1], %2;" ::"l"(dst), "r"(s), "r"(chunk) : "memory");
        else
          asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f32 [%0], [%1], %2;" ::"l"(dst), "r"(s), "r"(chunk) : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        if ((it & 7) == 7) asm volatile("cp.async.bulk.wait_group.read 8;" ::: "memory");
      }
      asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Read-only streaming probe: how fast this GPU delivers a buffer that is read once and never written -- the ceiling of
// step a2, next to which MEASURED_PEAKS.json's COPY rate (read + write) is the contract's denominator.
//   KIND 0  256-bit ld.global.nc.L1::no_allocate.L2::evict_first loads, grid-stride (the flat kernels' loads)
//   KIND 1  TMA bulk copies of 32 KiB into a 4-slot shared-memory ring per CTA, one CTA per SM, completion on mbarriers,
//           nobody reads the tiles (k_tmem's producer with the consumers removed)
// `sink` (8 bytes, device) is written only if the XOR of everything read equals a value it cannot have by accident.
// ------------------------------------------------------------------------------------------------
template <int KIND>
__global__ void __launch_bounds__(256) k_stream_probe(const float* __restrict__ src, int64_t bytes, uint64_t* sink) {
  if constexpr (KIND == 0) {
    const int64_t vecs = bytes / 32;
    uint32_t acc = 0;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < vecs; k += (int64_t)gridDim.x * blockDim.x) {
      float v[8];
      ld_stream<8>(src + k * 8, v);
#pragma unroll
      for (int i = 0; i < 8; ++i) acc ^= __float_as_uint(v[i]);
    }
    if (acc == 0x7FC12345u && sink) *sink = acc;
  } else {
    constexpr uint32_t TILE = 32768, NS = 4;
    extern __shared__ __align__(1024) unsigned char probe_ring[];
    const uint32_t ring = smem_u32(probe_ring), bars = ring + NS * TILE;
    if (threadIdx.x == 0) {
      for (uint32_t k = 0; k < NS; ++k) mbar_init(bars + 8 * k, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      asm volatile("fence.proxy.async;" ::: "memory");
      const uint64_t policy = l2_evict_first_policy();
      const int64_t tiles = bytes / TILE;
      uint32_t it = 0;
      for (int64_t t = blockIdx.x; t < tiles; t += gridDim.x, ++it) {
        const uint32_t slot = it % NS;
        if (it >= NS) mbar_wait(bars + 8 * slot, ((it / NS) - 1) & 1);   // the copy that used this slot last has landed
        mbar_expect_tx(bars + 8 * slot, TILE);
        bulk_g2s(ring + slot * TILE, reinterpret_cast<const unsigned char*>(src) + t * TILE, TILE, bars + 8 * slot, policy);
        mbar_arrive(bars + 8 * slot);
      }
      for (uint32_t k = (it > NS ? it - NS : 0); k < it; ++k) mbar_wait(bars + 8 * (k % NS), (k / NS) & 1);
      if (sink && probe_ring[0] == 0xA5 && probe_ring[TILE - 1] == 0x5A && bytes < 0) *sink = 1;
    }
  }
}

// ------------------------------------------------------------------------------------------------
// a4 in isolation (tests; SURVEY 8c row 14 "the hardware cvt.rs.f16x2.f32 may be used only if shown bit-identical"):
// out[k] = the 16-bit conversion of p[k] under `kind` with the random bits r[k].
//   0 RN16   1 SR16 (R13, r24 = r & 0xFFFFFF)   2 dither (R20, same r24)   3 bfloat16 RN
//   4 / 5    hardware cvt.rs.f16x2.f32 d, a, b, rbits with p in BOTH sources: the half converted from b (low, 4) / a (high, 5)
//   6 / 7    the library's SR pair conversion pack_sr_bits(p, p, r24 in both fields): low (6) / high (7) half
// ------------------------------------------------------------------------------------------------
__global__ void k_convert_probe(const float* __restrict__ p, const uint32_t* __restrict__ r, int64_t count, int kind, uint16_t* __restrict__ out) {
  int64_t stride = (int64_t)gridDim.x * blockDim.x;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < count; k += stride) {
    const float x = p[k];
    const uint32_t rb = r ? r[k] : 0u;
    uint32_t v;
    switch (kind) {
      case 0: v = pack_rn(x, x) & 0xFFFFu; break;
      case 1: v = sr16_bits(x, rb & 0xFFFFFFu); break;
      case 2: v = pack_rn(dither_f32(x, rb & 0xFFFFFFu), 0.f) & 0xFFFFu; break;
      case 3: v = pack_bf16_rn(x, x) & 0xFFFFu; break;
      case 6: case 7: {   // the library's pair conversion (fast path on the normal grid, integer rule elsewhere): r24 in both fields of R
        const uint64_t R = ((uint64_t)(rb & 0xFFFFFFu) << 40) | ((uint64_t)(rb & 0xFFFFFFu) << 16);
        const uint32_t d = pack_sr_bits(x, x, R);
        v = kind == 6 ? (d & 0xFFFFu) : (d >> 16);
        break;
      }
      default: {
        uint32_t d;
        asm("cvt.rs.f16x2.f32 %0, %1, %2, %3;" : "=r"(d) : "f"(x), "f"(x), "r"(rb));
        v = kind == 4 ? (d & 0xFFFFu) : (d >> 16);
      }
    }
    out[k] = (uint16_t)v;
  }
}

}  // namespace sk
