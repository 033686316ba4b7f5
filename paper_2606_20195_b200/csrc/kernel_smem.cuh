// kernel_smem.cuh -- shared-memory-privatised FP16 scatter for sm_100a.
//
// Each CTA keeps one private d x n FP16 partial sketch in shared memory and streams a contiguous range
// of rows; at the end it flushes the partial sketch into B with 16-byte result-discarding REDs.
// sm_100a has no native shared-memory FP16 add (atomicAdd on shared assembles to a CAS loop), so every
// sketch word has exactly one owner at any time and is updated with plain LDS.128 / HFMA2 / STS.128:
//   - warp w of the CTA owns the 64-column slice [64w, 64w+64): no two warps touch the same word;
//   - inside a warp the lanes are R = 4 rows x 8 column chunks of 8 columns.  One "row group" (4 rows)
//     is scattered per step: for every stack block j the 4 rows read-modify-write their 4 buckets of
//     block j at once.  Two rows of a group collide in block j with probability ~6/(d/zeta); the hash
//     stage ranks such rows (rank = number of earlier rows of the group with the same bucket in that
//     block), and a group with any non-zero rank takes a slow path that applies the ranks one after
//     the other.  In the common path the ZETA read-modify-writes of a group are independent, so the
//     ZETA LDS.128 are in flight together (blocks are disjoint row ranges of the sketch).
// The product s*a is rounded to FP16 once per element; the block sign enters as the +-1 multiplier of
// HFMA2 (q * (+-1) + acc: the product is exact, one rounding = RN16(acc +- q)).
// A goes straight from HBM into registers with 256-bit streaming loads through an 8-deep register
// ring (8 row groups = 8 KiB in flight per warp): staging A through shared memory would add 8 B/float
// to a shared-memory pipe that the 2*2*ZETA B/float of read-modify-write traffic already loads.
#pragma once

#include "kernels.cuh"

namespace sk {

struct SmemArgs {
  ScatterArgs s;
  int64_t rows_per_cta;  // multiple of kSmemRingRows
  int32_t d;
};

constexpr int kSmemVec = 8;                 // columns per lane
constexpr int kSmemLpr = 8;                 // lanes per row
constexpr int kSmemR = 4;                   // rows per group
constexpr int kSmemNq = 8;                  // ring depth in row groups
constexpr int kSmemRingRows = kSmemNq * kSmemR;  // 32
constexpr int kSmemColsPerWarp = kSmemVec * kSmemLpr;  // 64
constexpr uint32_t kRankShift = 28;         // entry bits 28..30: rank inside the row group
constexpr uint32_t kRankMask = 7u << kRankShift;
constexpr uint32_t kBucketMask = (1u << kRankShift) - 1u;

// acc (4 half2 words) += sign * q
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

template <int ZETA, int ROUNDING, int MAXW>
__global__ void __launch_bounds__(MAXW * 32) k_smem(SmemArgs g) {
  constexpr int VEC = kSmemVec, LPR = kSmemLpr, R = kSmemR, NQ = kSmemNq;
  static_assert(32 % ZETA == 0, "ZETA must divide 32");
  constexpr int HB = 32 / ZETA;                 // rows per hash batch (lane l -> row l/ZETA, block l%ZETA)
  constexpr int GPB = (HB >= R) ? HB / R : 1;   // row groups per hash batch
  constexpr int BPG = (HB >= R) ? 1 : R / HB;   // hash batches per row group (ZETA = 16, 32)
  static_assert(BPG == 1, "ZETA <= 8 supported");
  constexpr int JC = ZETA < 4 ? ZETA : 4;       // blocks handled together (bounds the accumulator registers)
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
  const int64_t cta_r1 = min(a.rows, cta_r0 + g.rows_per_cta);
  const uint32_t col0 = warp * kSmemColsPerWarp + pcol * VEC;  // first column of this lane
  unsigned char* const my_col = smem_raw + col0 * 2u;
  const uint32_t npairs = ((uint32_t)a.n + 1u) >> 1;

  if (cta_r0 < cta_r1) {
    const int64_t nrows = cta_r1 - cta_r0;
    const int64_t iters = (nrows + kSmemRingRows - 1) / kSmemRingRows;
    const int64_t full_iters = nrows / kSmemRingRows;  // iterations whose 32 rows all exist
    // lane's load pointer for (iteration 0, group 0); a group is R rows further, an iteration 32 rows
    const float* ld_ptr = a.A + (cta_r0 + r) * a.lda + col0;
    const int64_t group_stride = (int64_t)R * a.lda;

    float buf[NQ][VEC];
    // prologue: iteration 0's groups
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
      if ((int64_t)q * R + r < nrows) ld_stream<VEC>(ld_ptr + q * group_stride, buf[q]);
      else {
#pragma unroll
        for (int k = 0; k < VEC; ++k) buf[q][k] = 0.f;
      }
    }

    for (int64_t it = 0; it < iters; ++it) {
      const int64_t it_row0 = cta_r0 + it * kSmemRingRows;  // local row of this iteration's first row
      // how the next iteration's loads must be issued: 0 = none, 1 = unchecked, 2 = row-checked
      const int next_mode = (it + 1 < full_iters) ? 1 : (it + 1 < iters) ? 2 : 0;
      const float* next_ptr = ld_ptr + (it + 1) * (int64_t)NQ * group_stride;
      const int64_t next_rows_left = nrows - (it + 1) * kSmemRingRows;  // rows that exist in the next iteration

#pragma unroll
      for (int hb = 0; hb < NQ / GPB; ++hb) {
        // ---- hash stage for HB rows: lane l -> (row l/ZETA, block l%ZETA), plus the rank inside its group
        uint32_t e;
        {
          const int64_t b0 = it_row0 + (int64_t)hb * HB;
          const uint64_t ctr = (uint64_t)(a.row_begin + b0) * ZETA + lane;
          e = hash_entry(a.seed, ctr, lane % ZETA, a.db);
          const uint32_t bucket = entry_bucket(e);
          const uint32_t row_in_group = (lane / ZETA) % R;
          uint32_t rank = 0;
#pragma unroll
          for (int k = 1; k < R; ++k) {
            const uint32_t other = __shfl_up_sync(0xFFFFFFFFu, bucket, k * ZETA);
            rank += (row_in_group >= (uint32_t)k && other == bucket) ? 1u : 0u;
          }
          e |= rank << kRankShift;
        }
#pragma unroll
        for (int gq = 0; gq < GPB; ++gq) {
          const int q = hb * GPB + gq;
          float p[VEC];
#pragma unroll
          for (int k = 0; k < VEC; ++k) p[k] = buf[q][k] * a.scale;
          // refill this ring slot with the same group of the next iteration
          if (next_mode == 1) {
            ld_stream<VEC>(next_ptr + q * group_stride, buf[q]);
          } else if (next_mode == 2) {
            if ((int64_t)q * R + r < next_rows_left) ld_stream<VEC>(next_ptr + q * group_stride, buf[q]);
            else {
#pragma unroll
              for (int k = 0; k < VEC; ++k) buf[q][k] = 0.f;
            }
          }
          uint32_t qv[VEC / 2];
          if constexpr (ROUNDING == 0) {
#pragma unroll
            for (int k = 0; k < VEC / 2; ++k) qv[k] = pack_rn(p[2 * k], p[2 * k + 1]);
          }
          const uint32_t rib = (uint32_t)gq * R + r;  // row in hash batch
#pragma unroll
          for (int jc = 0; jc < ZETA; jc += JC) {
            uint32_t ej[JC];
            unsigned char* addr[JC];
            uint32_t mult[JC];
            uint32_t anyrank = 0;
#pragma unroll
            for (int j = 0; j < JC; ++j) {
              ej[j] = __shfl_sync(0xFFFFFFFFu, e, rib * ZETA + jc + j);
              addr[j] = my_col + (ej[j] & kBucketMask) * row_pitch;
              mult[j] = (entry_signmask_h2(ej[j])) ^ 0x3C003C00u;  // +-1.0 in both halves
              anyrank |= ej[j];
            }
            uint32_t w[JC][VEC / 2];
#pragma unroll
            for (int j = 0; j < JC; ++j) {
              if constexpr (ROUNDING == 0) {
#pragma unroll
                for (int k = 0; k < VEC / 2; ++k) w[j][k] = qv[k];
              } else {
                // SR converts every contribution separately (the draw depends on (row, block, pair))
                const uint32_t sf = entry_signmask_f32(ej[j]);
                const int64_t grow = a.row_begin + it_row0 + (int64_t)hb * HB + rib;
                const uint64_t sr_ctr = ((uint64_t)grow * ZETA + (jc + j)) * npairs + (uint64_t)(col0 >> 1);
#pragma unroll
                for (int k = 0; k < VEC / 2; ++k)
                  w[j][k] = pack_sr(__uint_as_float(__float_as_uint(p[2 * k]) ^ sf),
                                    __uint_as_float(__float_as_uint(p[2 * k + 1]) ^ sf), a.sr_seed, sr_ctr + k);
                mult[j] = 0x3C003C00u;  // sign already applied before the conversion
              }
            }
            if (!__any_sync(0xFFFFFFFFu, (anyrank & kRankMask) != 0u)) {
              // common path: the JC read-modify-writes are independent -> all loads first
              uint4 acc[JC];
#pragma unroll
              for (int j = 0; j < JC; ++j) acc[j] = *reinterpret_cast<uint4*>(addr[j]);
#pragma unroll
              for (int j = 0; j < JC; ++j) rmw_add(acc[j], w[j], mult[j]);
#pragma unroll
              for (int j = 0; j < JC; ++j) *reinterpret_cast<uint4*>(addr[j]) = acc[j];
            } else {
              // some rows of the group share a bucket: apply rank 0, then rank 1, ...
              for (uint32_t k = 0; k < (uint32_t)R; ++k) {
                bool more = false;
#pragma unroll
                for (int j = 0; j < JC; ++j) {
                  const uint32_t rk = (ej[j] & kRankMask) >> kRankShift;
                  if (rk == k) {
                    uint4 acc = *reinterpret_cast<uint4*>(addr[j]);
                    rmw_add(acc, w[j], mult[j]);
                    *reinterpret_cast<uint4*>(addr[j]) = acc;
                  }
                  more |= rk > k;
                }
                __syncwarp();
                if (!__any_sync(0xFFFFFFFFu, more)) break;
              }
            }
            __syncwarp();
          }
        }
      }
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
