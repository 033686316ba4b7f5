// kernel_smem.cuh -- shared-memory-privatised FP16-RN scatter for sm_100a.
//
// Each CTA keeps one private d x n FP16 partial sketch in shared memory and streams a contiguous range
// of rows; at the end it flushes the partial sketch into B with 16-byte result-discarding REDs.
// sm_100a has no native shared-memory FP16 add (atomicAdd on shared assembles to a CAS loop), so every
// sketch word has exactly one owner at any time and is updated with plain LDS.128 / HFMA2 / STS.128:
//   - warp w of the CTA owns the 64-column slice [64w, 64w+64): no two warps touch the same word;
//   - inside a warp the lanes are R = 4 rows x 8 column chunks of 8 columns.  One "row group" (4
//     consecutive rows, aligned to 4 in the global row index) is scattered per step: for every stack
//     block j the 4 rows read-modify-write their 4 buckets of block j at once.  Two rows of a group
//     collide in block j with probability ~6/(d/zeta); the hash stage ranks such rows (rank = number
//     of earlier rows of the group with the same bucket in that block) and a group with a non-zero
//     rank takes a slow path that applies rank 0, then rank 1, ...  In the common path the ZETA
//     read-modify-writes of a group are independent (blocks are disjoint row ranges of the sketch,
//     PAPER.md:59-63), so the ZETA LDS.128 are in flight together.
// The product s*a is rounded to FP16 once per element; the block sign enters as the +-1 multiplier of
// HFMA2 (q * (+-1) + acc: the product is exact, one rounding = RN16(acc +- q)).
// A goes straight from HBM into registers with 256-bit streaming loads through an NQ-deep register
// ring (NQ row groups = NQ KiB in flight per warp): staging A through shared memory would add
// 8 B/float to a shared-memory pipe that the 2*2*ZETA B/float of read-modify-write traffic already
// loads, and the register file is otherwise idle (2-6 warps per SM).
// Hash stage (a1) in its precomputed form: k_hash_pack_ranked writes one 16-bit entry per (row, block)
//   bucket | rank<<11 | group_max_rank<<13 | sign<<15
// and every lane loads its row's ZETA entries (2*ZETA bytes, +ZETA/(2n) of A's traffic) through the
// same register ring.  (The on-the-fly form of this kernel cost ~25 of 135 instructions per row group,
// profiles/r01_smem_hash_on_the_fly.md; the flat kernels keep both forms.)
#pragma once

#include "args.h"
#include "device_util.cuh"

namespace sk {

constexpr int kSmemVec = 8;                            // columns per lane
constexpr int kSmemLpr = 8;                            // lanes per row
constexpr int kSmemR = 4;                              // rows per group
constexpr int kSmemColsPerWarp = kSmemVec * kSmemLpr;  // 64
constexpr int kSmemMaxBucket = 2048;                   // 11-bit bucket field of the ranked 16-bit entry
constexpr int kSmemPadRows = 128;                      // rows the packed array extends beyond m (ring look-ahead)

// ranked 16-bit entry
constexpr uint32_t kE16Bucket = 0x07FFu;
constexpr uint32_t kE16RankShift = 11;  // 2 bits
constexpr uint32_t kE16GmaxShift = 13;  // 2 bits: largest rank in the row group (same in all its entries)

// ring depth (row groups in flight per warp) per instantiation; the host sizes rows_per_cta from it
constexpr int smem_ring_depth(int zeta, bool small_cta) { return small_cta ? (zeta == 8 ? 8 : 12) : 4; }

// ------------------------------------------------------------------------------------------------
// a1 (precomputed form): ranked entries for every (row, block), rows padded beyond m.
// One warp hashes 32/ZETA rows; ranks come from shuffles inside the aligned 4-row group.
// ------------------------------------------------------------------------------------------------
template <int ZETA>
__global__ void k_hash_pack_ranked(uint64_t seed, int64_t rows_padded, uint32_t db, uint16_t* __restrict__ packed) {
  constexpr int HB = 32 / ZETA;
  constexpr int GL = kSmemR * ZETA;  // lanes per row group
  static_assert(GL <= 32, "ZETA <= 8");
  const uint32_t lane = threadIdx.x & 31;
  const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int64_t batches = rows_padded / HB;
  for (int64_t b = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; b < batches; b += warps) {
    const uint64_t ctr = (uint64_t)b * 32 + lane;  // (row)*ZETA + j with row = b*HB + lane/ZETA
    const uint32_t e = hash_entry(seed, ctr, lane % ZETA, db);
    const uint32_t bucket = entry_bucket(e);
    const uint32_t row_in_group = (lane / ZETA) % kSmemR;
    uint32_t rank = 0;
#pragma unroll
    for (int k = 1; k < kSmemR; ++k) {
      const uint32_t other = __shfl_up_sync(0xFFFFFFFFu, bucket, k * ZETA);
      rank += (row_in_group >= (uint32_t)k && other == bucket) ? 1u : 0u;
    }
    uint32_t gmax = rank;
#pragma unroll
    for (int off = 1; off < GL; off <<= 1) gmax = max(gmax, __shfl_xor_sync(0xFFFFFFFFu, gmax, off));
    packed[ctr] = (uint16_t)(bucket | (rank << kE16RankShift) | (gmax << kE16GmaxShift) | ((e >> 31) << 15));
  }
}

template <int ZETA> struct EntRow;  // a row's ZETA 16-bit entries as one load
template <> struct EntRow<1> { using type = uint16_t; };
template <> struct EntRow<2> { using type = uint32_t; };
template <> struct EntRow<4> { using type = uint2; };
template <> struct EntRow<8> { using type = uint4; };

template <int ZETA>
SK_DEVINL uint32_t entrow_word(const typename EntRow<ZETA>::type& e, int w) {
  if constexpr (ZETA == 1) return (uint32_t)e;
  else if constexpr (ZETA == 2) return e;
  else if constexpr (ZETA == 4) return w == 0 ? e.x : e.y;
  else return w == 0 ? e.x : w == 1 ? e.y : w == 2 ? e.z : e.w;
}

// acc (4 half2 words) += mult * q  (mult = +-1 in both halves)
SK_DEVINL void rmw_add(uint4& acc, const uint32_t (&q)[4], uint32_t mult) {
  const __half2 m = *reinterpret_cast<const __half2*>(&mult);
  __half2 x0 = __hfma2(*reinterpret_cast<const __half2*>(&q[0]), m, *reinterpret_cast<__half2*>(&acc.x));
  __half2 x1 = __hfma2(*reinterpret_cast<const __half2*>(&q[1]), m, *reinterpret_cast<__half2*>(&acc.y));
  __half2 x2 = __hfma2(*reinterpret_cast<const __half2*>(&q[2]), m, *reinterpret_cast<__half2*>(&acc.z));
  __half2 x3 = __hfma2(*reinterpret_cast<const __half2*>(&q[3]), m, *reinterpret_cast<__half2*>(&acc.w));
  acc.x = *reinterpret_cast<uint32_t*>(&x0);
  acc.y = *reinterpret_cast<uint32_t*>(&x1);
  acc.z = *reinterpret_cast<uint32_t*>(&x2);
  acc.w = *reinterpret_cast<uint32_t*>(&x3);
}

template <int ZETA, int NQ, int MAXW>
__global__ void __launch_bounds__(MAXW * 32) k_smem(SmemArgs g) {
  constexpr int VEC = kSmemVec, LPR = kSmemLpr, R = kSmemR;
  static_assert(ZETA == 1 || ZETA == 2 || ZETA == 4 || ZETA == 8, "ZETA in {1,2,4,8}");
  static_assert(2 * NQ * R <= kSmemPadRows, "packed-array padding covers the look-ahead");
  constexpr int RING_ROWS = NQ * R;
  constexpr int JC = ZETA < 4 ? ZETA : 4;  // blocks handled together (bounds the accumulator registers)
  using ent_t = typename EntRow<ZETA>::type;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const ScatterArgs& a = g.s;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t r = lane / LPR, pcol = lane % LPR;
  const uint32_t row_pitch = (uint32_t)a.n * 2u;  // bytes per sketch row in shared memory

  // ---- a0 (private part): zero the partial sketch
  {
    uint4* z = reinterpret_cast<uint4*>(smem_raw);
    const uint32_t n16 = (uint32_t)g.d * row_pitch / 16u;
    for (uint32_t k = tid; k < n16; k += blockDim.x) z[k] = make_uint4(0, 0, 0, 0);
  }
  __syncthreads();

  const int64_t cta_r0 = (int64_t)blockIdx.x * g.rows_per_cta;
  const int64_t cta_r1 = min(a.rows, cta_r0 + g.rows_per_cta);  // a.rows is a multiple of RING_ROWS here
  const uint32_t col0 = warp * kSmemColsPerWarp + pcol * VEC;  // first column of this lane
  unsigned char* const my_col = smem_raw + col0 * 2u;
  unsigned char* const my_dummy = smem_raw + (uint32_t)g.d * row_pitch + tid * 16u;  // 16 private bytes behind the sketch

  // The host gives every CTA a whole number of ring iterations (rows_per_cta and the range handed to this
  // kernel are multiples of NQ*R rows; the ragged remainder of a range goes to the flat kernel), so the
  // loop below needs no row checks and exists in a single copy.
  if (cta_r0 < cta_r1) {
    const int64_t iters = (cta_r1 - cta_r0) / RING_ROWS;
    const int64_t group_stride = (int64_t)R * a.lda;
    const float* const first_ptr = a.A + (cta_r0 + r) * a.lda + col0;        // this lane's (iteration 0, group 0)
    const ent_t* ent_ptr = reinterpret_cast<const ent_t*>(a.packed) + (a.row_begin + cta_r0 + r);

    float buf[NQ][VEC];
    ent_t ent[NQ];
    const float* ld_ptr = first_ptr;  // walks one group per load
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      ld_stream<VEC>(ld_ptr, buf[q]);
      ld_ptr += group_stride;
      ent[q] = __ldg(ent_ptr + q * R);
    }

    for (int64_t it = 0; it < iters; ++it) {
      // the last iteration has nothing left to prefetch: it re-reads iteration 0 (valid addresses, data unused)
      if (it + 1 == iters) {
        ld_ptr = first_ptr;
        ent_ptr -= it * RING_ROWS + RING_ROWS;
      }
#pragma unroll
      for (int q = 0; q < NQ; ++q) {
        float p[VEC];
#pragma unroll
        for (int k = 0; k < VEC; ++k) p[k] = buf[q][k] * a.scale;
        const ent_t my_ent = ent[q];
        // refill this ring slot with the same group of the next iteration
        ld_stream<VEC>(ld_ptr, buf[q]);
        ld_ptr += group_stride;
        ent[q] = __ldg(ent_ptr + RING_ROWS + q * R);

        uint32_t qv[VEC / 2];
#pragma unroll
        for (int k = 0; k < VEC / 2; ++k) qv[k] = pack_rn(p[2 * k], p[2 * k + 1]);
#pragma unroll
        for (int jc = 0; jc < ZETA; jc += JC) {
          unsigned char* addr[JC];
          uint32_t mult[JC], e16[JC];
#pragma unroll
          for (int j = 0; j < JC; ++j) {
            const uint32_t w = entrow_word<ZETA>(my_ent, (jc + j) >> 1);
            e16[j] = ((jc + j) & 1) ? (w >> 16) : (w & 0xFFFFu);
            addr[j] = my_col + (e16[j] & kE16Bucket) * row_pitch;
            // sign bit of the entry replicated into both halves, XOR +1.0: +-1.0 in both halves
            mult[j] = (__byte_perm(w, 0, ((jc + j) & 1) ? 0x3232 : 0x1010) & 0x80008000u) ^ 0x3C003C00u;
          }
          // pass 0: every (row, block) of rank 0.  No two of them share a word, so the JC read-modify-writes
          // are independent: all loads first.  Ranked-later rows aim at the lane's private dummy word instead
          // (no branch, no predicate on the memory operations).
          {
            uint4 acc[JC];
#pragma unroll
            for (int j = 0; j < JC; ++j) {
              unsigned char* const a0 = (e16[j] & (3u << kE16RankShift)) ? my_dummy : addr[j];
              acc[j] = *reinterpret_cast<uint4*>(a0);
            }
#pragma unroll
            for (int j = 0; j < JC; ++j) rmw_add(acc[j], qv, mult[j]);
#pragma unroll
            for (int j = 0; j < JC; ++j) {
              unsigned char* const a0 = (e16[j] & (3u << kE16RankShift)) ? my_dummy : addr[j];
              *reinterpret_cast<uint4*>(a0) = acc[j];
            }
          }
          __syncwarp();
          // rows that share a bucket with an earlier row of the group (~6/(d/zeta) of the groups per block):
          // one more pass per rank; gmax is the same in every lane (the warp is one row group)
          const uint32_t gmax = (e16[0] >> kE16GmaxShift) & 3u;
          for (uint32_t k = 1; k <= gmax; ++k) {
#pragma unroll
            for (int j = 0; j < JC; ++j) {
              if (((e16[j] >> kE16RankShift) & 3u) == k) {
                uint4 acc = *reinterpret_cast<uint4*>(addr[j]);
                rmw_add(acc, qv, mult[j]);
                *reinterpret_cast<uint4*>(addr[j]) = acc;
              }
            }
            __syncwarp();
          }
        }
      }
      ent_ptr += RING_ROWS;
    }
  }
  __syncthreads();

  // ---- flush: partial sketch -> B with 16-byte result-discarding REDs (layouts coincide: [d][n])
  {
    const uint4* z = reinterpret_cast<const uint4*>(smem_raw);
    const uint32_t n16 = (uint32_t)g.d * row_pitch / 16u;
    __half* B = reinterpret_cast<__half*>(a.B);
    // stagger the start so the CTAs do not all hit the same L2 lines at once
    const uint32_t shift = (uint32_t)((blockIdx.x * 2654435761u) % n16);
    for (uint32_t k0 = tid; k0 < n16; k0 += blockDim.x) {
      uint32_t k = k0 + shift;
      k = (k >= n16) ? k - n16 : k;
      uint4 v = z[k];
      if ((v.x | v.y | v.z | v.w) != 0u) red_h8(B + (size_t)k * 8, v.x, v.y, v.z, v.w);
    }
  }
}

}  // namespace sk
