// kernel_flat.cuh -- streaming scatter kernels with result-discarding global RED:
//   k_flat<...>     the paper's Listings 1/2 restated for sm_100a: shared hashes + 8/16-byte vector RED
//   k_generic<...>  any-n / any-alignment scalar fallback
#pragma once

#include "args.h"
#include "device_util.cuh"

namespace sk {

// packed entry -> canonical 32-bit entry (bucket | sign<<31).  16-bit entries are the form written by
// k_hash_pack_rot (kernel_smem.cuh): bucket in bits 0..10, sign in bit 15, stored in sub-step order.
template <typename PackT>
SK_DEVINL uint32_t unpack_entry(PackT p) {
  if constexpr (sizeof(PackT) == 2) return ((uint32_t)p & 0x07FFu) | (((uint32_t)p >> 15) << 31);
  else return (uint32_t)p;
}

// ------------------------------------------------------------------------------------------------
// Flat scatter: every contribution is one result-discarding RED into an L2-resident sketch.
//
// One warp owns a "macro step" of HB = 32/ZETA consecutive rows.  Lane l hashes (row l/ZETA, block
// l%ZETA) once -- 32 hashes per warp instead of n/VEC redundant ones per row -- and the HB*n floats
// are then consumed as 32-lane chunks of VEC consecutive columns (coalesced 32*VEC*4-byte requests),
// each lane fetching its row's ZETA entries by shuffle.  The product s*a is rounded to FP16 once per
// element and the block sign applied by XOR, which is bit-identical to RN16((eps*s)*a) because RN is
// odd; SR converts per contribution.
// Replicas: CTA b adds into partial sketch b % P, which cuts same-address serialisation in L2 and the
// depth of every running sum by P; k_reduce_replicas folds them.
// ------------------------------------------------------------------------------------------------
template <int VEC, int OUT, int ROUNDING>
SK_DEVINL void emit_contribution(void* Bbase, int64_t off, const float (&p)[VEC], const uint32_t (&q)[VEC / 2 > 0 ? VEC / 2 : 1],
                                 uint32_t e, uint64_t sr_seed, uint64_t sr_ctr) {
  if constexpr (OUT != OUT_F32) {
    uint16_t* dst = reinterpret_cast<uint16_t*>(Bbase) + off;
    uint32_t w[VEC / 2];
    if constexpr (ROUNDING == RND_RN) {
      uint32_t sm = entry_signmask_h2(e);   // binary16 and bfloat16 keep the sign in bit 15 of each half
#pragma unroll
      for (int k = 0; k < VEC / 2; ++k) w[k] = q[k] ^ sm;
    } else {
      uint32_t sf = entry_signmask_f32(e);  // SR / dither convert the SIGNED product, per contribution
#pragma unroll
      for (int k = 0; k < VEC / 2; ++k)
        w[k] = pack_f16<ROUNDING>(__uint_as_float(__float_as_uint(p[2 * k]) ^ sf), __uint_as_float(__float_as_uint(p[2 * k + 1]) ^ sf),
                                  sr_seed, sr_ctr + k);
    }
    if constexpr (VEC == 8) red_p8<OUT>(dst, w[0], w[1], w[2], w[3]);
    else if constexpr (VEC == 4) red_p4<OUT>(dst, w[0], w[1]);
    else red_p2<OUT>(dst, w[0]);
  } else {
    float* dst = reinterpret_cast<float*>(Bbase) + off;
    uint32_t sf = entry_signmask_f32(e);
    float w[VEC];
#pragma unroll
    for (int k = 0; k < VEC; ++k) w[k] = __uint_as_float(__float_as_uint(p[k]) ^ sf);
    if constexpr (VEC == 8) {
      red_f4(dst, w[0], w[1], w[2], w[3]);
      red_f4(dst + 4, w[4], w[5], w[6], w[7]);
    } else if constexpr (VEC == 4) red_f4(dst, w[0], w[1], w[2], w[3]);
    else if constexpr (VEC == 2) red_f2(dst, w[0], w[1]);
    else red_f1(dst, w[0]);
  }
}

template <int ZETA, int VEC, int OUT, int ROUNDING, typename PackT>
__global__ void __launch_bounds__(kFlatThreads) k_flat(ScatterArgs a) {
  constexpr bool F16 = OUT != OUT_F32;   // a 16-bit sketch (binary16 or bfloat16)
  static_assert(32 % ZETA == 0, "ZETA must divide 32");
  constexpr int HB = 32 / ZETA;            // rows per macro step
  constexpr bool PRE = sizeof(PackT) > 1;  // PackT = uint8_t means "hash on the fly"
  const uint32_t lane = threadIdx.x & 31;
  const int64_t warps = ((int64_t)gridDim.x * kFlatThreads) >> 5;
  const int64_t gwarp = ((int64_t)blockIdx.x * kFlatThreads + threadIdx.x) >> 5;
  const int64_t macros = (a.rows + HB - 1) / HB;
  const uint32_t chunks = (uint32_t)HB * a.cpr;  // chunks per macro step
  char* Bbase = reinterpret_cast<char*>(a.B) +
                (size_t)(blockIdx.x % a.replicas) * (size_t)a.replica_stride * (F16 ? 2 : 4);
  const uint32_t npairs = ((uint32_t)a.n + 1u) >> 1;

  for (int64_t mac = gwarp; mac < macros; mac += warps) {
    const int64_t r0 = mac * HB;  // local row of the macro step
    // ---- hash stage: lane l -> (row r0 + l/ZETA, block l%ZETA)
    uint32_t e;
    {
      uint32_t j = lane % ZETA;
      uint64_t ctr = (uint64_t)(a.row_begin + r0) * ZETA + lane;  // (row)*ZETA + j with row = r0 + lane/ZETA
      if constexpr (PRE) {
        int64_t lr = r0 + lane / ZETA;
        uint64_t idx = ctr;
        if constexpr (sizeof(PackT) == 2) {  // entry of block j sits at sub-step t = (j - row mod R) mod ZETA
          constexpr uint32_t R = ZETA >= 4 ? 4 : ZETA;
          const uint32_t rr = (uint32_t)((uint64_t)(a.row_begin + lr) % R);
          idx = ctr - j + ((j + ZETA - rr) % ZETA);
        }
        e = (lr < a.rows) ? unpack_entry<PackT>(reinterpret_cast<const PackT*>(a.packed)[idx]) : 0u;
      } else {
        e = hash_entry(a.seed, ctr, j, a.db);
      }
    }
    // ---- stream the HB x n floats
    for (uint32_t c = lane; c < ((chunks + 31u) & ~31u); c += 32) {
      // c / cpr: magic 0 <=> cpr == 1; magic ~0 <=> the multiply-high form is not exact for this width (host: make_args)
      uint32_t rr = a.cpr_magic == 0u ? c : (a.cpr_magic == 0xFFFFFFFFu ? c / a.cpr : __umulhi(c, a.cpr_magic));
      uint32_t ch = c - rr * a.cpr;
      bool valid = (c < chunks) && (r0 + rr < a.rows);
      rr = valid ? rr : 0u;
      float p[VEC];
      uint32_t q[VEC / 2 > 0 ? VEC / 2 : 1];
      if (valid) {
        ld_stream<VEC>(a.A + (r0 + rr) * a.lda + (int64_t)ch * VEC, p);
#pragma unroll
        for (int k = 0; k < VEC; ++k) p[k] *= a.scale;
      } else {
#pragma unroll
        for (int k = 0; k < VEC; ++k) p[k] = 0.f;
      }
      if constexpr (F16 && ROUNDING == RND_RN) {
#pragma unroll
        for (int k = 0; k < VEC / 2; ++k) q[k] = OUT == OUT_BF16 ? pack_bf16_rn(p[2 * k], p[2 * k + 1]) : pack_rn(p[2 * k], p[2 * k + 1]);
      }
#pragma unroll
      for (int j = 0; j < ZETA; ++j) {
        uint32_t ej = __shfl_sync(0xFFFFFFFFu, e, rr * ZETA + j);
        if (valid) {
          int64_t off = (int64_t)entry_bucket(ej) * a.n + (int64_t)ch * VEC;
          uint64_t sr_ctr = ((uint64_t)(a.row_begin + r0 + rr) * ZETA + j) * npairs + (uint64_t)ch * (VEC / 2);
          emit_contribution<VEC, OUT, ROUNDING>(Bbase, off, p, q, ej, a.sr_seed, sr_ctr);
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Generic fallback: one lane per (row, column) element, runtime zeta, scalar RED; any n, lda, alignment.
// ------------------------------------------------------------------------------------------------
template <int OUT, int ROUNDING>
__global__ void __launch_bounds__(kFlatThreads) k_generic(ScatterArgs a) {
  constexpr bool F16 = OUT != OUT_F32;
  const int64_t total = a.rows * (int64_t)a.n;
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  const uint32_t npairs = ((uint32_t)a.n + 1u) >> 1;
  char* Bbase = reinterpret_cast<char*>(a.B) +
                (size_t)(blockIdx.x % a.replicas) * (size_t)a.replica_stride * (F16 ? 2 : 4);
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += stride) {
    int64_t r = idx / a.n;
    int32_t c = (int32_t)(idx - r * a.n);
    float p = a.A[r * a.lda + c] * a.scale;
    for (int32_t j = 0; j < a.zeta; ++j) {
      uint64_t ctr = (uint64_t)(a.row_begin + r) * (uint64_t)a.zeta + (uint64_t)j;
      uint32_t e = hash_entry(a.seed, ctr, (uint32_t)j, a.db);
      int64_t off = (int64_t)entry_bucket(e) * a.n + c;
      float ps = __uint_as_float(__float_as_uint(p) ^ entry_signmask_f32(e));
      if constexpr (F16) {
        uint16_t v;
        if constexpr (OUT == OUT_BF16) {
          v = __bfloat16_as_ushort(__float2bfloat16_rn(ps));
        } else if constexpr (ROUNDING == RND_RN) {
          v = __half_as_ushort(__float2half_rn(ps));
        } else {
          const uint64_t pc = ctr * npairs + (uint64_t)(c >> 1);
          uint64_t R = ROUNDING == RND_SR ? splitmix64(a.sr_seed ^ pc) : dither_bits(a.sr_seed, pc);
          uint32_t r24 = (c & 1) ? ((uint32_t)(R >> 16) & 0xFFFFFFu) : (uint32_t)(R >> 40);
          v = ROUNDING == RND_SR ? (uint16_t)sr16_bits(ps, r24) : __half_as_ushort(__float2half_rn(dither_f32(ps, r24)));
        }
        uint16_t* dst = reinterpret_cast<uint16_t*>(Bbase) + off;
        if (off == a.odd_tail) red_h1_cas<OUT>(dst, v);   // last element of an odd-sized B
        else red_h1<OUT>(dst, v);
      } else {
        red_f1(reinterpret_cast<float*>(Bbase) + off, ps);
      }
    }
  }
}

}  // namespace sk
