// kernel_tmem.cuh -- tensor-memory-privatised FP16-RN scatter for sm_100a.
//
// The partial sketch of a warp lives in TENSOR MEMORY (TMEM: 128 lanes x 512 columns x 32 bit per SM, the
// tcgen05 accumulator store), not in shared memory.  What makes that possible: every feature of one input
// row goes to the SAME sketch row (bucket(i, j) does not depend on the column), so with
//     TMEM lane   <->  feature-column group (lane l of the warp holds X half2 words = 2X adjacent features)
//     TMEM column <->  sketch row:  bucket b occupies columns [b*X, b*X + X)
// the address of a read-modify-write is warp-uniform, which is exactly what tcgen05.ld / tcgen05.st
// (shape 32x32b.xX: each lane reads/writes X consecutive columns of its own TMEM lane) require.  One
// contribution of a whole row slice is then  LDTM.xX -> X x HFMA2 -> STTM.xX  (q * (+-1) + acc = one RN16 add
// per FP16 half), and the SM's L1/shared data pipe -- 81 % busy in the shared-memory kernel
// (profiles/r01_smem_c5.md) -- only carries A itself.
//
// CTA = NW consumer warps + 1 producer warp, one CTA per SM (it allocates all 512 TMEM columns).
//   producer  : per stage of T rows: cp.async.bulk (TMA, L2 evict-first) of the A tile into a ring of NS
//               shared-memory slots, completion on an mbarrier; meanwhile its 32 lanes compute the stage's
//               hashes ON THE FLY (a1: splitmix64 counter hash, one lane per row) and store per (row, block)
//               an 8-byte entry {TMEM column offset = bucket*X, HFMA2 multiplier = +-1.0 in both halves}.
//               No separate hash pass, no packed hash array in HBM.
//   consumers : warp w owns TMEM lanes [32*(w%4), +32) (the hardware's lane quadrant of that warp) and
//               columns [(w/4)*d*X, +d*X): a private d x 64X partial sketch.  n = 64*X*S: a row is cut in S
//               column slices; warp w takes slice w%S of the rows of row-set w/S of every stage.
//               Rows are processed in groups of G: all LDTMs of a group are issued, then one
//               tcgen05.wait::ld, then the HFMA2s and STTMs.  Two rows of a group that hit the same
//               bucket are chained in registers (the later row adds onto the earlier row's result and both
//               store the chain's final value) -- the bucket is warp-uniform, so this is a select, not
//               divergence.  tcgen05.wait::st orders a group's LDTMs behind the previous group's STTMs.
//   flush     : LDTM.x8 -> result-discarding vector REDs into B.
//
// Sketches larger than one warp's 512 TMEM columns (d * X > 512) are split two ways:
//   BQ bucket groups : the zeta stack blocks are cut into BQ groups of ZB = zeta / BQ consecutive blocks
//               (disjoint sketch-row ranges); a warp of group b holds only the d / BQ sketch
//               rows of its blocks and adds only those contributions.  Every row is then converted by BQ
//               warps, which costs shared-memory reads and F2FPs but no tensor-memory capacity.
//   CS column slices : gridDim.y CTAs share a row range, CTA y takes the features [y * N, (y + 1) * N) of every
//               row (N = 64 * X * S); its A tile is fetched row by row (N * 4 bytes each), the hashes are
//               recomputed per slice.  d = 1024, n = 256: X = 2, BQ = 4, CS = 2;  d = 2048: X = 1, BQ = 4, CS = 4.
// Accumulation is FP16 RN throughout; the hierarchy is (warp-private partial) -> RED into B.
#pragma once

#include <cuda.h>  // CUtensorMap (type only; the encoder is fetched with cudaGetDriverEntryPoint)

#include "args.h"
#include "device_util.cuh"

namespace sk {

constexpr int kTmemCols = 512;

// ---------------------------------------------------------------------------------------- PTX wrappers
SK_DEVINL uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

SK_DEVINL void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
SK_DEVINL void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
SK_DEVINL void mbar_arrive(uint32_t bar) {
  asm volatile("{ .reg .b64 st; mbarrier.arrive.shared::cta.b64 st, [%0]; }" ::"r"(bar) : "memory");
}
SK_DEVINL void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}" ::"r"(bar), "r"(parity) : "memory");
}
SK_DEVINL uint64_t l2_evict_first_policy() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// TMA bulk copy global -> shared, completion (bytes) on an mbarrier; 16-byte aligned, size % 16 == 0
SK_DEVINL void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t policy) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}

// TMA tiled copy of a {N features x T rows} box at (column c0, row c1) of the 2-D tensor map; rows and
// columns outside the tensor are zero-filled and still counted in the transaction bytes
SK_DEVINL void tensor_g2s(uint32_t dst, const CUtensorMap* tmap, int32_t c0, int32_t c1, uint32_t bar, uint64_t policy) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
               ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tmap)), "r"(c0), "r"(c1), "r"(bar), "l"(policy) : "memory");
}

template <int X> SK_DEVINL void tmem_ld(uint32_t taddr, uint32_t (&v)[X]) {
  static_assert(X == 1 || X == 2 || X == 4, "X");
  if constexpr (X == 1) asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v[0]) : "r"(taddr));
  else if constexpr (X == 2) asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=r"(v[0]), "=r"(v[1]) : "r"(taddr));
  else asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(taddr));
}
SK_DEVINL void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(taddr));
}
// store executed only when `on` is non-zero (warp-uniform by construction: the instruction is .sync.aligned)
template <int X> SK_DEVINL void tmem_st_if(uint32_t on, uint32_t taddr, const uint32_t (&v)[X]) {
  if constexpr (X == 1)
    asm volatile("{ .reg .pred p; setp.ne.u32 p, %2, 0; @p tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1}; }" ::"r"(taddr), "r"(v[0]), "r"(on));
  else if constexpr (X == 2)
    asm volatile("{ .reg .pred p; setp.ne.u32 p, %3, 0; @p tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2}; }" ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(on));
  else
    asm volatile("{ .reg .pred p; setp.ne.u32 p, %5, 0; @p tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4}; }" ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(on));
}
template <int X> SK_DEVINL void tmem_st(uint32_t taddr, const uint32_t (&v)[X]) {
  if constexpr (X == 1) asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "r"(v[0]));
  else if constexpr (X == 2) asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" ::"r"(taddr), "r"(v[0]), "r"(v[1]));
  else asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]));
}
SK_DEVINL void tmem_st8_zero(uint32_t taddr) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(taddr), "r"(0u));
}
SK_DEVINL void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
SK_DEVINL void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// tcgen05.ld writes its registers asynchronously: every use must be ordered behind tcgen05.wait::ld.  An
// empty volatile asm that "modifies" the register gives the compiler that dependency at no cost.
SK_DEVINL void tmem_tie(uint32_t& v) { asm volatile("" : "+r"(v)); }

SK_DEVINL uint32_t hfma2_u32(uint32_t q, uint32_t mult, uint32_t acc) {
  uint32_t d;
  asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(q), "r"(mult), "r"(acc));
  return d;
}

// ---------------------------------------------------------------------------------------- geometry
template <int ZETA, int X, int S, int BQ, int NW, int T>
struct TmemGeom {
  static_assert(NW % 4 == 0 && NW % (S * BQ) == 0, "consumer warps: whole lane quadrants, whole slice x bucket-group sets");
  static_assert(ZETA % BQ == 0, "bucket groups are whole stack blocks");
  static constexpr int ZB = ZETA / BQ;         // stack blocks one warp accumulates
  static constexpr int RS = NW / (S * BQ);     // row-sets per stage
  static constexpr int TR = T / RS;            // rows of a stage one warp processes
  #ifndef SK_TMEM_G_SMALL
#define SK_TMEM_G_SMALL 4
#endif
  static constexpr int G = (ZB >= 4 || (BQ > 1 && ZB >= 2)) ? 2 : SK_TMEM_G_SMALL;  // rows per group (LDTMs in flight = G * ZB)
  static_assert(TR % G == 0, "whole groups");
  static constexpr int N = 64 * X * S;         // features of the CTA's column slice
  static constexpr int WC = kTmemCols / (NW / 4);  // tensor-memory columns of one warp's private region
  static constexpr int A_BYTES = T * N * 4;
  static constexpr int E_BYTES = T * ZETA * 8;
  static constexpr int STAGE_BYTES = A_BYTES + E_BYTES;
};

// rows per stage: 32 KiB of A per stage (16 KiB at n = 64), at least 16 rows
__host__ __device__ constexpr int tmem_stage_rows(int n) { return n <= 128 ? 64 : n == 256 ? 32 : 16; }
__host__ __device__ constexpr int tmem_stages(int n) { return n <= 512 ? 4 : 3; }
constexpr size_t tmem_smem_bytes(int zeta, int n) {
  return (size_t)tmem_stages(n) * ((size_t)tmem_stage_rows(n) * n * 4 + (size_t)tmem_stage_rows(n) * zeta * 8) + 16 * 8 + 16;
}

// ---------------------------------------------------------------------------------------- the kernel
template <int ZETA, int X, int S, int BQ, int NW>
__global__ void __launch_bounds__((NW + 1) * 32, 1) k_tmem(TmemArgs g, const __grid_constant__ CUtensorMap tmap) {
  constexpr int T = tmem_stage_rows(64 * X * S), NS = tmem_stages(64 * X * S);
  using Geo = TmemGeom<ZETA, X, S, BQ, NW, T>;
  constexpr int TR = Geo::TR, G = Geo::G, N = Geo::N, ZB = Geo::ZB;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const ScatterArgs& a = g.s;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // shared-memory carve-up: [NS][A tile | entries] then the barriers
  const uint32_t smem0 = smem_u32(smem_raw);
  const uint32_t bars = smem0 + NS * Geo::STAGE_BYTES;     // full[NS], empty[NS], 8 B each
  uint32_t* const tbase_p = reinterpret_cast<uint32_t*>(smem_raw + NS * Geo::STAGE_BYTES + 16 * NS);

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tbase_p)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 32) {
    for (int k = 0; k < NS; ++k) {
      mbar_init(bars + 8 * k, 1);              // full: the producer's arrive (+ the TMA transaction bytes)
      mbar_init(bars + 8 * (NS + k), NW);      // empty: one arrive per consumer warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tbase = *tbase_p;

  const int64_t nstages = (a.rows + T - 1) / T;
  const int64_t col0 = (int64_t)blockIdx.y * N;   // first feature of this CTA's column slice
  const uint32_t dloc = (uint32_t)g.d / BQ;        // sketch rows one warp holds

  if (warp == NW) {
    // ================================================================ producer: TMA + hash stage (a1, a2)
    const uint64_t policy = l2_evict_first_policy();
    const bool contiguous = (a.lda == N);          // implies a single column slice
    uint32_t it = 0;
    for (int64_t st = blockIdx.x; st < nstages; st += gridDim.x, ++it) {
      const uint32_t slot = it % NS, ph = (it / NS) & 1;
      const uint32_t sA = smem0 + slot * Geo::STAGE_BYTES, sE = sA + Geo::A_BYTES;
      const uint32_t full = bars + 8 * slot, empty = bars + 8 * (NS + slot);
      mbar_wait(empty, ph ^ 1);                // passes at once the first time round the ring
      const int64_t row0 = st * T;
      const int32_t nrows = (int32_t)min((int64_t)T, a.rows - row0);
      if (contiguous) {
        if (lane == 0) {
          mbar_expect_tx(full, (uint32_t)nrows * N * 4);
          bulk_g2s(sA, a.A + row0 * a.lda, (uint32_t)nrows * N * 4, full, policy);
        }
      } else if (lane == 0) {                  // strided rows / column slice: one tiled TMA copy per stage
        mbar_expect_tx(full, (uint32_t)T * N * 4);
        tensor_g2s(sA, &tmap, (int32_t)col0, (int32_t)row0, full, policy);
      }
      if (contiguous && nrows < T) {           // last stage of the matrix: rows past the end contribute +0
        const uint32_t z0 = sA + nrows * N * 4, z1 = sA + Geo::A_BYTES;
        for (uint32_t p = z0 + lane * 16; p < z1; p += 32 * 16) asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(p), "r"(0u) : "memory");
      }
      // a1: entries of rows lane, lane + 32, ...: {(bucket - first sketch row of the block's group) * X, +-1.0 | +-1.0}
#pragma unroll
      for (int rr = 0; rr < (T + 31) / 32; ++rr) {
        const int32_t r = rr * 32 + (int32_t)lane;
        if (T % 32 != 0 && r >= T) break;      // stages of 16 rows (n >= 512): half a warp hashes
        const uint64_t ctr0 = (uint64_t)(a.row_begin + row0 + r) * ZETA;
        uint32_t w[2 * ZETA];
#pragma unroll
        for (int j = 0; j < ZETA; ++j) {
          const uint32_t e = hash_entry(a.seed, ctr0 + j, j, a.db);
          w[2 * j] = (entry_bucket(e) - (uint32_t)(j / ZB) * dloc) * X;
          w[2 * j + 1] = 0x3C003C00u ^ entry_signmask_h2(e);
        }
        const uint32_t p = sE + r * (ZETA * 8);
        if constexpr (ZETA == 1) asm volatile("st.shared.v2.b32 [%0], {%1,%2};" ::"r"(p), "r"(w[0]), "r"(w[1]) : "memory");
        else {
#pragma unroll
          for (int k = 0; k < ZETA / 2; ++k)
            asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(p + 16 * k), "r"(w[4 * k]), "r"(w[4 * k + 1]), "r"(w[4 * k + 2]), "r"(w[4 * k + 3]) : "memory");
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(full);
    }
  } else {
    // ================================================================ consumers: a3, a4, a5 in tensor memory
    const uint32_t slice = warp % S, bgrp = (warp / S) % BQ, rowset = warp / (S * BQ);
    const uint32_t region = tbase + (((warp & 3u) * 32u) << 16) + (warp >> 2) * (uint32_t)Geo::WC;
    const uint32_t ncols = dloc * X;  // multiple of 8, <= WC (host check)
    for (uint32_t c = 0; c < ncols; c += 8) tmem_st8_zero(region + c);   // a0 (private part)
    tmem_wait_st();

    const float scale = a.scale;
    const uint32_t a_off = (rowset * TR) * (N * 4) + (slice * 64 * X + lane * 2 * X) * 4;
    const uint32_t e_off = (rowset * TR) * (ZETA * 8) + bgrp * (ZB * 8);
    uint32_t it = 0;
    for (int64_t st = blockIdx.x; st < nstages; st += gridDim.x, ++it) {
      const uint32_t slot = it % NS, ph = (it / NS) & 1;
      const unsigned char* const sA = smem_raw + slot * Geo::STAGE_BYTES + a_off;
      const unsigned char* const sE = smem_raw + slot * Geo::STAGE_BYTES + Geo::A_BYTES + e_off;
      mbar_wait(bars + 8 * slot, ph);
#pragma unroll
      for (int g0 = 0; g0 < TR; g0 += G) {
        uint32_t q[G][X], col[G][ZB], mul[G][ZB];
#pragma unroll
        for (int r = 0; r < G; ++r) {
          // a2 (from the staged tile), a3, a4: q = RN16(s * a), two features per word
          float v[2 * X];
          const unsigned char* pa = sA + (g0 + r) * (N * 4);
          if constexpr (X == 1) { const float2 t = *reinterpret_cast<const float2*>(pa); v[0] = t.x; v[1] = t.y; }
          else {
#pragma unroll
            for (int k = 0; k < X / 2; ++k) {
              const float4 t = *reinterpret_cast<const float4*>(pa + 16 * k);
              v[4 * k] = t.x; v[4 * k + 1] = t.y; v[4 * k + 2] = t.z; v[4 * k + 3] = t.w;
            }
          }
#pragma unroll
          for (int k = 0; k < X; ++k) q[r][k] = pack_rn(v[2 * k] * scale, v[2 * k + 1] * scale);
          const unsigned char* pe = sE + (g0 + r) * (ZETA * 8);
          if constexpr (ZB == 1) { const uint2 t = *reinterpret_cast<const uint2*>(pe); col[r][0] = t.x; mul[r][0] = t.y; }
          else {
#pragma unroll
            for (int k = 0; k < ZB / 2; ++k) {
              const uint4 t = *reinterpret_cast<const uint4*>(pe + 16 * k);
              col[r][2 * k] = t.x; mul[r][2 * k] = t.y; col[r][2 * k + 1] = t.z; mul[r][2 * k + 1] = t.w;
            }
          }
        }
        // a5: read-modify-write of G x ZB sketch rows in tensor memory
        uint32_t acc[G][ZB][X];
        tmem_wait_st();                        // the previous group's stores are in TMEM
#pragma unroll
        for (int r = 0; r < G; ++r)
#pragma unroll
          for (int j = 0; j < ZB; ++j) tmem_ld<X>(region + col[r][j], acc[r][j]);
        tmem_wait_ld();
#pragma unroll
        for (int r = 0; r < G; ++r)
#pragma unroll
          for (int j = 0; j < ZB; ++j)
#pragma unroll
            for (int k = 0; k < X; ++k) tmem_tie(acc[r][j][k]);
#pragma unroll
        for (int j = 0; j < ZB; ++j) {
#pragma unroll
          for (int r = 0; r < G; ++r) {
            // chain onto the latest earlier row of the group that hit the same sketch row
#pragma unroll
            for (int p = 0; p < r; ++p) {
              const bool same = col[p][j] == col[r][j];
#pragma unroll
              for (int k = 0; k < X; ++k) acc[r][j][k] = same ? acc[p][j][k] : acc[r][j][k];
            }
#pragma unroll
            for (int k = 0; k < X; ++k) acc[r][j][k] = hfma2_u32(q[r][k], mul[r][j], acc[r][j][k]);
          }
          // rows of the group that share a sketch row all store the chain's final value: the stores need
          // no predicate and their order does not matter
#pragma unroll
          for (int r = G - 2; r >= 0; --r) {
#pragma unroll
            for (int p = G - 1; p > r; --p) {
              const bool same = col[p][j] == col[r][j];
#pragma unroll
              for (int k = 0; k < X; ++k) acc[r][j][k] = same ? acc[p][j][k] : acc[r][j][k];
            }
          }
#pragma unroll
          for (int r = 0; r < G; ++r) tmem_st<X>(region + col[r][j], acc[r][j]);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bars + 8 * (NS + slot));
    }

    // ---- flush: private partial sketch -> B with result-discarding vector REDs (a5's last level)
    tmem_wait_st();
    __half* const Bw = reinterpret_cast<__half*>(a.B) + (size_t)(bgrp * dloc) * a.n + col0 + slice * 64 * X + lane * 2 * X;
    for (uint32_t c = 0; c < ncols; c += 8) {
      uint32_t v[8];
      tmem_ld8(region + c, v);
      tmem_wait_ld();
#pragma unroll
      for (int k = 0; k < 8; ++k) tmem_tie(v[k]);
#pragma unroll
      for (int b = 0; b < 8 / X; ++b) {
        __half* dst = Bw + (size_t)(c / X + b) * a.n;
        if constexpr (X == 1) { if (v[b] != 0u) red_h2(dst, v[b]); }
        else if constexpr (X == 2) { if ((v[2 * b] | v[2 * b + 1]) != 0u) red_h4(dst, v[2 * b], v[2 * b + 1]); }
        else { if ((v[4 * b] | v[4 * b + 1] | v[4 * b + 2] | v[4 * b + 3]) != 0u) red_h8(dst, v[4 * b], v[4 * b + 1], v[4 * b + 2], v[4 * b + 3]); }
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tbase) : "memory");
}

}  // namespace sk
