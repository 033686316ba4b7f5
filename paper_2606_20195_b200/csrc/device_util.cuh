// device_util.cuh -- device-side building blocks of the sm_100a sparse-sketch kernels:
// the counter hash, FP32->FP16 conversion RN / SR (a4) and the
// result-discarding reductions (a5, a6).
#pragma once

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>

#include "args.h"

#define SK_DEVINL __device__ __forceinline__

namespace sk {

// ------------------------------------------------------------------------------------------------
// Hash: h = splitmix64(seed ^ ctr), ctr = i*zeta + j (BASELINE.json:north_star; R1-R4).
// Packed entry: bucket | signbit << 31.
// ------------------------------------------------------------------------------------------------
SK_DEVINL uint64_t splitmix64(uint64_t x) {
  uint64_t z = x + 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

SK_DEVINL uint32_t hash_entry(uint64_t seed, uint64_t ctr, uint32_t j, uint32_t db) {
  uint64_t h = splitmix64(seed ^ ctr);
  uint32_t bucket = j * db + __umulhi((uint32_t)(h >> 32), db);  // ((h>>32)*db)>>32, db < 2^31
  return bucket | ((uint32_t)h << 31);
}

SK_DEVINL uint32_t entry_bucket(uint32_t e) { return e & 0x7FFFFFFFu; }
// 0x80008000 when the sign bit is set, else 0: XOR mask for a packed half2 (RN is odd)
SK_DEVINL uint32_t entry_signmask_h2(uint32_t e) { return (uint32_t)((int32_t)e >> 31) & 0x80008000u; }
SK_DEVINL uint32_t entry_signmask_f32(uint32_t e) { return e & 0x80000000u; }

// ------------------------------------------------------------------------------------------------
// Conversion FP32 -> packed half2 {lo = x0, hi = x1}.
// RN: cvt.rn.f16x2.f32 (SASS F2FP.F16.F32.PACK_AB), round-to-nearest-even, subnormals kept,
//     |x| >= 65520 -> inf; the __float2half of PAPER.md:127-129.
// ------------------------------------------------------------------------------------------------
SK_DEVINL uint32_t pack_rn(float x0, float x1) {
  __half2 h = __floats2half2_rn(x0, x1);
  return *reinterpret_cast<uint32_t*>(&h);
}

// bfloat16 control: cvt.rn.bf16x2.f32, round-to-nearest-even, subnormals kept, overflow -> inf
SK_DEVINL uint32_t pack_bf16_rn(float x0, float x1) {
  uint32_t d;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(d) : "f"(x1), "f"(x0));   // first source -> upper half
  return d;
}

// SR (R13): magnitude rounded toward zero to l, moved one grid step away
// from zero iff u < t with t = (|p|-|l|)/w and u = (r24 + 1/2) 2^-24.  All-integer evaluation:
// with s discarded bits and rem their value, u < t  <=>  (2 r24 + 1) 2^s < rem 2^25.
SK_DEVINL uint32_t sr16_bits(float p, uint32_t r24) {
  uint32_t fb = __float_as_uint(p);
  uint32_t sign = (fb >> 16) & 0x8000u;
  uint32_t mag = fb & 0x7FFFFFFFu;
  if (mag > 0x7F800000u) return sign | 0x7E00u;   // NaN
  if (mag >= 0x47800000u) return sign | 0x7C00u;  // |p| >= 65536 -> inf
  if (mag >= 0x38800000u) {                       // |p| >= 2^-14: FP16 normal grid, 13 discarded bits
    uint32_t trunc = (mag >> 13) - 0x1C000u;      // rebias 127 -> 15
    uint32_t rem = mag & 0x1FFFu;
    uint32_t up = ((r24 >> 11) < rem) ? 1u : 0u;  // (2 r24+1) < rem<<12  <=>  r24>>11 < rem
    return sign | (trunc + up);                   // carry walks into the exponent; 0x7BFF+1 = inf
  }
  // FP16 subnormal grid, spacing 2^-24
  uint32_t ef = mag >> 23;                                       // biased FP32 exponent, 0 = FP32 subnormal
  uint32_t M = (mag & 0x7FFFFFu) | (ef ? 0x800000u : 0u);        // |p| = M * 2^(e-23)
  int e = ef ? (int)ef - 127 : -126;
  int s = -1 - e;                                                // 14 .. 125
  uint32_t l = (s < 24) ? (M >> s) : 0u;
  uint32_t rem = (s < 24) ? (M & ((1u << s) - 1u)) : M;
  uint64_t lhs = 2ull * r24 + 1ull;
  bool up;
  if (s <= 25) up = lhs < ((uint64_t)rem << (25 - s));
  else if (s < 49) up = (lhs << (s - 25)) < (uint64_t)rem;
  else up = false;
  return sign | (l + (up ? 1u : 0u));
}

// one 64-bit draw per column pair (R14): bits 63..40 -> even column, bits 39..16 -> odd column.
// Fast path (R22): when both magnitudes lie on the FP16 NORMAL grid [2^-14, 65504) -- 13 discarded bits -- the
// hardware cvt.rs.f16x2.f32 IS rule R13 with the 13-bit random field of each half = the complement of r24's top 13 bits
// (it adds the field to the discarded bits and carries; R13 rounds up iff r24 >> 11 < rem).  Shown bit-identical there on
// 6.8e8 samples (tests/test_gpu_modes.py); below 2^-14 and from 65504 up it is not (or not shown), so those pairs take the
// integer rule.  One instruction instead of ~35 for the pair.
SK_DEVINL uint32_t pack_sr_bits(float x0, float x1, uint64_t R) {
  const uint32_t m0 = __float_as_uint(x0) & 0x7FFFFFFFu, m1 = __float_as_uint(x1) & 0x7FFFFFFFu;
  constexpr uint32_t LO = 0x38800000u, SPAN = 0x477FE000u - 0x38800000u;   // 2^-14 .. 65504
  if (((m0 - LO) < SPAN) && ((m1 - LO) < SPAN)) {
    const uint32_t f0 = ~(uint32_t)(R >> 51) & 0x1FFFu;          // r24(even) >> 11, complemented
    const uint32_t f1 = ~(uint32_t)(R >> 27) & 0x1FFFu;          // r24(odd) >> 11, complemented
    uint32_t d;
    asm("cvt.rs.f16x2.f32 %0, %1, %2, %3;" : "=r"(d) : "f"(x1), "f"(x0), "r"(f0 | (f1 << 16)));   // first source -> upper half
    return d;
  }
  const uint32_t lo = sr16_bits(x0, (uint32_t)(R >> 40));
  const uint32_t hi = sr16_bits(x1, (uint32_t)(R >> 16) & 0xFFFFFFu);
  return lo | (hi << 16);
}
SK_DEVINL uint32_t pack_sr(float x0, float x1, uint64_t sr_seed, uint64_t ctr) {
  return pack_sr_bits(x0, x1, splitmix64(sr_seed ^ ctr));
}

// Dither, Eq. (6) (R20): RN16(q + (u0 - 1/2) c q), every operation one FP32 operation
// rounded to nearest in the written order (no contraction into an FMA).  u0 - 1/2 = (r24 - 2^23) 2^-24 exactly, and
// fl(((r24 - 2^23) 2^-24) c) = fl((r24 - 2^23) c) 2^-24: a power-of-two factor commutes with the rounding (no underflow:
// the product is 0 or at least 2^-34), so the two roundings of t and w collapse into one multiply by c 2^-24.
SK_DEVINL float dither_f32(float q, uint32_t r24) {
  const float ti = (float)((int32_t)r24 - (1 << 23));               // exact: |.| <= 2^23
  const float w = __fmul_rn(ti, 0.00097656f * 5.9604644775390625e-08f);   // c 2^-24: the literal's bits, exponent - 24
  const float e = __fmul_rn(w, q);
  return __fadd_rn(q, e);
}
// one xorshift64 step (13, 7, 17) on the counter hash (state 0 replaced), R21; bit layout as R14
SK_DEVINL uint64_t dither_bits(uint64_t sr_seed, uint64_t ctr) {
  uint64_t x = splitmix64(sr_seed ^ ctr);
  x = x ? x : 0x9E3779B97F4A7C15ull;
  x ^= x << 13;
  x ^= x >> 7;
  x ^= x << 17;
  return x;
}
SK_DEVINL uint32_t pack_dither(float x0, float x1, uint64_t sr_seed, uint64_t ctr) {
  const uint64_t R = dither_bits(sr_seed, ctr);
  return pack_rn(dither_f32(x0, (uint32_t)(R >> 40)), dither_f32(x1, (uint32_t)(R >> 16) & 0xFFFFFFu));
}
// conversion of one signed column pair under rule RND (FP16 path)
template <int RND>
SK_DEVINL uint32_t pack_f16(float x0, float x1, uint64_t sr_seed, uint64_t ctr) {
  if constexpr (RND == RND_SR) return pack_sr(x0, x1, sr_seed, ctr);
  else if constexpr (RND == RND_DITHER) return pack_dither(x0, x1, sr_seed, ctr);
  else return pack_rn(x0, x1);
}

// ------------------------------------------------------------------------------------------------
// Result-discarding reductions to global memory (L2).  PAPER.md:177-183: atom.global.add with the
// result unused -> SASS REDG (no return path).  sm_90+/sm_100a also take 8- and 16-byte vector forms
// (REDG.E.ADD.F16x4 / F16x8 / F32x2 / F32x4): one instruction, one L2 transaction, 2-4 column pairs.
// .noftz keeps FP16 subnormals; every half / float component is added independently.
// ------------------------------------------------------------------------------------------------
SK_DEVINL void red_h2(void* p, uint32_t a) {
  asm volatile("red.global.add.noftz.f16x2 [%0], %1;" ::"l"(p), "r"(a) : "memory");
}
SK_DEVINL void red_h4(void* p, uint32_t a, uint32_t b) {
  asm volatile("red.global.add.noftz.v2.f16x2 [%0], {%1,%2};" ::"l"(p), "r"(a), "r"(b) : "memory");
}
SK_DEVINL void red_h8(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("red.global.add.noftz.v4.f16x2 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d)
               : "memory");
}
SK_DEVINL void red_b2(void* p, uint32_t a) {
  asm volatile("red.global.add.noftz.bf16x2 [%0], %1;" ::"l"(p), "r"(a) : "memory");
}
SK_DEVINL void red_b4(void* p, uint32_t a, uint32_t b) {
  asm volatile("red.global.add.noftz.v2.bf16x2 [%0], {%1,%2};" ::"l"(p), "r"(a), "r"(b) : "memory");
}
SK_DEVINL void red_b8(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("red.global.add.noftz.v4.bf16x2 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d)
               : "memory");
}
// packed 16-bit REDs by element type
template <int OUT> SK_DEVINL void red_p2(void* p, uint32_t a) { if constexpr (OUT == OUT_BF16) red_b2(p, a); else red_h2(p, a); }
template <int OUT> SK_DEVINL void red_p4(void* p, uint32_t a, uint32_t b) { if constexpr (OUT == OUT_BF16) red_b4(p, a, b); else red_h4(p, a, b); }
template <int OUT> SK_DEVINL void red_p8(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  if constexpr (OUT == OUT_BF16) red_b8(p, a, b, c, d); else red_h8(p, a, b, c, d);
}
SK_DEVINL void red_f1(void* p, float a) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(p), "f"(a) : "memory");
}
SK_DEVINL void red_f2(void* p, float a, float b) {
  asm volatile("red.global.add.v2.f32 [%0], {%1,%2};" ::"l"(p), "f"(a), "f"(b) : "memory");
}
SK_DEVINL void red_f4(void* p, float a, float b, float c, float d) {
  asm volatile("red.global.add.v4.f32 [%0], {%1,%2,%3,%4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d)
               : "memory");
}

// scalar FP16 add for odd n: there is no native scalar f16 RED on sm_100a (red.global.add.noftz.f16
// assembles to a CAS loop), so add {v, +0} or {+0, v} with the packed RED on the enclosing aligned
// 4-byte word: x + (+0) = x for every x except -0 -> +0, which the path never produces (R10).
template <int OUT = OUT_F16>
SK_DEVINL void red_h1(void* p, uint16_t v) {
  uintptr_t a = reinterpret_cast<uintptr_t>(p);
  uint32_t word = (a & 2) ? ((uint32_t)v << 16) : (uint32_t)v;
  red_p2<OUT>(reinterpret_cast<void*>(a & ~(uintptr_t)3), word);
}

// The last element of a sketch with an odd number of elements has no partner inside B: its enclosing word would
// reach two bytes past the buffer.  That one element is added with a 16-bit compare-and-swap loop instead.
template <int OUT = OUT_F16>
SK_DEVINL void red_h1_cas(void* p, uint16_t v) {
  unsigned short* q = reinterpret_cast<unsigned short*>(p);
  unsigned short old = *reinterpret_cast<volatile unsigned short*>(q), assumed;
  do {
    assumed = old;
    unsigned short sum;
    if constexpr (OUT == OUT_BF16) sum = __bfloat16_as_ushort(__hadd(__ushort_as_bfloat16(assumed), __ushort_as_bfloat16(v)));
    else sum = __half_as_ushort(__hadd(__ushort_as_half(assumed), __ushort_as_half(v)));
    old = atomicCAS(q, assumed, sum);
  } while (old != assumed);
}

// ------------------------------------------------------------------------------------------------
// Streaming loads of A: read once, never reused -> bypass L1 allocation; the 256-bit form also takes
// L2::evict_first (ptxas accepts that modifier only on .v8.b32/.v4.b64 loads).
// ------------------------------------------------------------------------------------------------
template <int VEC>
SK_DEVINL void ld_stream(const float* p, float (&v)[VEC]) {
  if constexpr (VEC == 8) {
    asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3]), "=f"(v[4]), "=f"(v[5]), "=f"(v[6]), "=f"(v[7])
                 : "l"(p));
  } else if constexpr (VEC == 4) {
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v[0]), "=f"(v[1]), "=f"(v[2]), "=f"(v[3])
                 : "l"(p));
  } else if constexpr (VEC == 2) {
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0,%1}, [%2];"
                 : "=f"(v[0]), "=f"(v[1])
                 : "l"(p));
  } else {
    asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(v[0]) : "l"(p));
  }
}

}  // namespace sk
