// kernel_smem.cuh -- shared-memory-privatised FP16-RN scatter for sm_100a.
//
// Each CTA keeps one private d x n FP16 partial sketch in shared memory and streams a contiguous range
// of rows; at the end it flushes the partial sketch into B with 16-byte result-discarding REDs.
// sm_100a has no native shared-memory FP16 add (atomicAdd on shared assembles to a CAS loop), so every
// sketch word is updated with plain LDS / HFMA2 / STS and the schedule guarantees that no two lanes
// touch one word in the same instruction:
//   - warp w of the CTA owns the 64-column slice [64w, 64w+64): no two warps ever touch the same word;
//   - inside a warp the lanes are R rows x LPR column chunks of VEC columns (R = min(zeta, 4); zeta >= 4:
//     4 rows x 8 lanes x 8 columns).  One "step" scatters R consecutive rows (aligned to R in the global
//     row index) in zeta "sub-steps": in sub-step t the lanes of row r update stack block (r + t) mod zeta.
//     The R rows of a step therefore hit R DIFFERENT blocks in every instruction, and blocks are disjoint
//     row ranges of the sketch: a Latin-square schedule with no same-instruction
//     conflicts, whatever the hash says.  Two rows that share a bucket meet in different sub-steps, and the
//     sub-steps of a warp are ordered (LDS/STS issue in order, __syncwarp between them).  To overlap the
//     shared-memory latency with the previous sub-step's HFMA2/STS, the LDS of a sub-step is issued D = 1
//     sub-steps early; the hash stage marks the (row, sub-step) entries whose sketch row is written inside
//     that window (probability ~D/(d/zeta)) and only those lanes repeat the LDS after the store.
//     No ranks, no branches, no divergence.
// The product s*a is rounded to FP16 once per element; the block sign enters as the +-1 multiplier of
// HFMA2 (q * (+-1) + acc: the product is exact, one rounding = RN16(acc +- q)).
// A goes straight from HBM into registers with 256-bit streaming loads (staging A through shared memory
// would add 8 B/float to the L1/shared data pipe that the 4*zeta B/float of read-modify-write traffic
// already loads to ~3/4 of its 128 B/clk).  ptxas tracks all of a warp's global loads with ONE scoreboard,
// so a wait for any load waits for every load in flight: loads are therefore issued in batches of K
// steps.  A batch is converted (a3, a4) into a work set as soon as it has arrived, the next batch is issued
// into the freed registers and is in flight for the whole time the work set is being scattered
// (a rolling ring stalled 26 % of all cycles on the v4 kernel).
// Hash stage (a1) in its precomputed form: k_hash_pack_rot writes one 16-bit entry per (row, sub-step)
//   bucket | sign<<15      for block (row mod R + t) mod zeta
// and every lane loads its row's zeta entries (2*zeta bytes per row, +zeta/(2n) of A's traffic).
#pragma once

#include "args.h"
#include "device_util.cuh"

namespace sk {

constexpr int kSmemColsPerWarp = 64;
constexpr int kSmemMaxBucket = 2047;   // 11-bit bucket field; index d is the CTA's dummy row
constexpr int kSmemDepth = 1;          // D: sub-steps whose LDS is issued ahead of the running read-modify-write
                                       // (measured on B200, c5: D = 0 3.62 ms, D = 1 3.47, D = 2 3.54, D = 3 3.53, D = 4 3.58)
constexpr int kSmemFlagDepth = 1;      // the reload flags cover this many earlier sub-steps (>= D)
constexpr int kSmemHaloRows = 4;       // rows a hash-pack warp recomputes in front of its 28 output rows
// 16-bit entry: bucket | reload<<14 | sign<<15
constexpr uint32_t kE16Bucket = 0x07FFu;
constexpr uint32_t kE16Reload = 0x4000u;

template <int ZETA>
struct SmemGeom {
  static constexpr int R = ZETA >= 4 ? 4 : ZETA;  // rows per step
  static constexpr int LPR = 32 / R;              // lanes per row
  static constexpr int VEC = kSmemColsPerWarp / LPR;  // columns per lane: 8 / 4 / 2
  static constexpr int H2 = VEC / 2;              // half2 words per lane
};

constexpr int smem_rows_per_step(int zeta) { return zeta >= 4 ? 4 : zeta; }
// K: steps per load batch; the host sizes rows_per_cta from it
constexpr int smem_batch_steps(int zeta, bool small_cta) { return small_cta ? 8 : 2; }

// ------------------------------------------------------------------------------------------------
// a1 (precomputed form).  Entry (row, t) describes block j = (row mod R + t) mod ZETA of that row:
//   bucket | reload<<14 | sign<<15.
// Sub-steps are numbered u = (row / R) * ZETA + t.  `reload` is set when one of the D sub-steps before u
// updates the same sketch row: sub-step u-k touches block j through row-slot (row mod R + k) mod ZETA (if
// that is < R) of step floor((u-k)/ZETA).  The scatter kernel issues the LDS of sub-step u before the
// stores of sub-steps u-D .. u-1 and repeats it after them only where `reload` is set.
// One lane per row (ZETA hashes each); a warp covers 32 consecutive rows of which the first 4 are a halo
// (recomputed, not written) so that every partner entry is one shuffle away.
// ------------------------------------------------------------------------------------------------
template <int ZETA>
__global__ void k_hash_pack_rot(uint64_t seed, int64_t rows, uint32_t db, uint16_t* __restrict__ packed) {
  constexpr int R = SmemGeom<ZETA>::R, D = kSmemFlagDepth, H = kSmemHaloRows, OUT = 32 - H;
  static_assert(H % R == 0 && H >= R * ((D + ZETA - 1) / ZETA), "halo covers D sub-steps");
  const uint32_t lane = threadIdx.x & 31;
  const int64_t warps = ((int64_t)gridDim.x * blockDim.x) >> 5;
  const int64_t chunks = (rows + OUT - 1) / OUT;
  for (int64_t c = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; c < chunks; c += warps) {
    const int64_t row = c * OUT - H + lane;  // OUT and H are multiples of R: row mod R == lane mod R
    const uint32_t r = lane % R;
    uint32_t b[ZETA];  // canonical entries of this row, by block
#pragma unroll
    for (int j = 0; j < ZETA; ++j) b[j] = row >= 0 ? hash_entry(seed, (uint64_t)row * ZETA + j, j, db) : 0x7FFFFFFFu;
    uint32_t e[ZETA];  // by sub-step: e[t] = b[(r + t) mod ZETA]
#pragma unroll
    for (int t = 0; t < ZETA; ++t) {
      e[t] = b[t];
#pragma unroll
      for (int rr = 1; rr < R; ++rr) e[t] = (r == (uint32_t)rr) ? b[(rr + t) % ZETA] : e[t];
    }
    uint32_t out[ZETA];
#pragma unroll
    for (int t = 0; t < ZETA; ++t) {
      bool reload = false;
#pragma unroll
      for (int k = 1; k <= D; ++k) {
        const int ds = (t - k >= 0) ? 0 : -((k - t + ZETA - 1) / ZETA);  // step of sub-step u-k relative to this one
        const int tk = ((t - k) % ZETA + ZETA) % ZETA;
        const uint32_t rk = (r + k) % ZETA;                                // its row slot for this block
        const int src = (int)lane + ds * R + (int)rk - (int)r;
        const uint32_t pe = __shfl_sync(0xFFFFFFFFu, e[tk], src & 31);
        reload |= (rk < (uint32_t)R) && (src >= 0) && (entry_bucket(pe) == entry_bucket(e[t]));
      }
      out[t] = entry_bucket(e[t]) | (reload ? kE16Reload : 0u) | ((e[t] >> 31) << 15);
    }
    if (lane >= (uint32_t)H && row < rows) {
      uint16_t* dst = packed + row * ZETA;
      if constexpr (ZETA == 1) dst[0] = (uint16_t)out[0];
      else if constexpr (ZETA == 2) *reinterpret_cast<uint32_t*>(dst) = out[0] | (out[1] << 16);
      else if constexpr (ZETA == 4) *reinterpret_cast<uint2*>(dst) = make_uint2(out[0] | (out[1] << 16), out[2] | (out[3] << 16));
      else *reinterpret_cast<uint4*>(dst) = make_uint4(out[0] | (out[1] << 16), out[2] | (out[3] << 16), out[4] | (out[5] << 16), out[6] | (out[7] << 16));
    }
  }
}

template <int ZETA> struct EntRow;  // a row's ZETA 16-bit entries as one load
template <> struct EntRow<1> { using type = uint16_t; static constexpr int W = 1; };
template <> struct EntRow<2> { using type = uint32_t; static constexpr int W = 1; };
template <> struct EntRow<4> { using type = uint2; static constexpr int W = 2; };
template <> struct EntRow<8> { using type = uint4; static constexpr int W = 4; };

template <int ZETA>
SK_DEVINL void entrow_load(const void* p, uint32_t (&w)[EntRow<ZETA>::W]) {
  if constexpr (ZETA == 1) w[0] = __ldg(reinterpret_cast<const uint16_t*>(p));
  else if constexpr (ZETA == 2) w[0] = __ldg(reinterpret_cast<const uint32_t*>(p));
  else if constexpr (ZETA == 4) {
    const uint2 v = __ldg(reinterpret_cast<const uint2*>(p));
    w[0] = v.x; w[1] = v.y;
  } else {
    const uint4 v = __ldg(reinterpret_cast<const uint4*>(p));
    w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
  }
}

// shared-memory accesses by 32-bit shared-window address (no generic-address arithmetic in the loop)
template <int H2>
SK_DEVINL void lds_h2(uint32_t addr, uint32_t (&v)[H2]) {
  if constexpr (H2 == 4) asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(addr) : "memory");
  else if constexpr (H2 == 2) asm volatile("ld.shared.v2.b32 {%0,%1}, [%2];" : "=r"(v[0]), "=r"(v[1]) : "r"(addr) : "memory");
  else asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v[0]) : "r"(addr) : "memory");
}
template <int H2>
SK_DEVINL void sts_h2(uint32_t addr, const uint32_t (&v)[H2]) {
  if constexpr (H2 == 4) asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
  else if constexpr (H2 == 2) asm volatile("st.shared.v2.b32 [%0], {%1,%2};" ::"r"(addr), "r"(v[0]), "r"(v[1]) : "memory");
  else asm volatile("st.shared.b32 [%0], %1;" ::"r"(addr), "r"(v[0]) : "memory");
}
// the same load again, executed only by lanes whose `flag` is non-zero (registers keep their value elsewhere)
template <int H2>
SK_DEVINL void lds_h2_if(uint32_t flag, uint32_t addr, uint32_t (&v)[H2]) {
  if constexpr (H2 == 4)
    asm volatile("{ .reg .pred p; setp.ne.b32 p, %5, 0; @p ld.shared.v4.b32 {%0,%1,%2,%3}, [%4]; }"
                 : "+r"(v[0]), "+r"(v[1]), "+r"(v[2]), "+r"(v[3]) : "r"(addr), "r"(flag) : "memory");
  else if constexpr (H2 == 2)
    asm volatile("{ .reg .pred p; setp.ne.b32 p, %3, 0; @p ld.shared.v2.b32 {%0,%1}, [%2]; }"
                 : "+r"(v[0]), "+r"(v[1]) : "r"(addr), "r"(flag) : "memory");
  else
    asm volatile("{ .reg .pred p; setp.ne.b32 p, %2, 0; @p ld.shared.b32 %0, [%1]; }" : "+r"(v[0]) : "r"(addr), "r"(flag) : "memory");
}
// acc = q * mult + acc per FP16 half, one rounding, subnormals kept
SK_DEVINL uint32_t hfma2_bits(uint32_t q, uint32_t mult, uint32_t acc) {
  uint32_t d;
  asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(q), "r"(mult), "r"(acc));
  return d;
}

template <int ZETA, int K>
struct SmemLoadSet {  // destination of the K steps of loads in flight
  float a[K][SmemGeom<ZETA>::VEC];
  uint32_t e[K][EntRow<ZETA>::W];
};
template <int ZETA, int K>
struct SmemWorkSet {  // the K steps being scattered: RN16(s*a) pairs and masked entries
  uint32_t q[K][SmemGeom<ZETA>::H2];
  uint32_t e[K][EntRow<ZETA>::W];
};

template <int ZETA, int K, int MAXW, int DEPTH = kSmemDepth>
__global__ void __launch_bounds__(MAXW * 32) k_smem(SmemArgs g) {
  using G = SmemGeom<ZETA>;
  constexpr int R = G::R, LPR = G::LPR, VEC = G::VEC, H2 = G::H2, EW = EntRow<ZETA>::W;
  static_assert(ZETA == 1 || ZETA == 2 || ZETA == 4 || ZETA == 8, "ZETA in {1,2,4,8}");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const ScatterArgs& a = g.s;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t r = lane / LPR, pcol = lane % LPR;
  const uint32_t pitch = (uint32_t)a.n * 2u;  // bytes per sketch row in shared memory

  // ---- a0 (private part): zero the partial sketch (+ the dummy row d that absorbs out-of-range steps)
  {
    uint4* z = reinterpret_cast<uint4*>(smem_raw);
    const uint32_t n16 = ((uint32_t)g.d + 1u) * pitch / 16u;
    for (uint32_t k = tid; k < n16; k += blockDim.x) z[k] = make_uint4(0, 0, 0, 0);
  }
  __syncthreads();

  const int64_t cta_r0 = (int64_t)blockIdx.x * g.rows_per_cta;          // multiple of R
  const int64_t cta_r1 = min(a.rows, cta_r0 + g.rows_per_cta);
  const uint32_t col0 = warp * kSmemColsPerWarp + pcol * VEC;            // first column of this lane
  const uint32_t lane_base = (uint32_t)__cvta_generic_to_shared(smem_raw) + col0 * 2u;
  const uint32_t dummy_word = (uint32_t)g.d | ((uint32_t)g.d << 16);     // every entry -> row d, sign +

  if (cta_r0 < cta_r1) {
    const int64_t last_row = cta_r1 - 1;
    const float* const Acol = a.A + col0;
    const unsigned char* const ent_base = reinterpret_cast<const unsigned char*>(a.packed) + (size_t)a.row_begin * (ZETA * 2);
    const int32_t nsteps = (int32_t)((cta_r1 - cta_r0 + R - 1) / R);

    SmemLoadSet<ZETA, K> L;
    SmemWorkSet<ZETA, K> W;

    // issue the loads of the batch that starts at step s0; rows past the CTA's range re-read its last row
    auto load_batch = [&](int32_t s0) {
#pragma unroll
      for (int s = 0; s < K; ++s) {
        const int64_t row = min(cta_r0 + (int64_t)(s0 + s) * R + r, last_row);
        ld_stream<VEC>(Acol + row * a.lda, L.a[s]);
        entrow_load<ZETA>(ent_base + row * (ZETA * 2), L.e[s]);
      }
    };
    // a3 + a4: first use of every loaded register (waits for the whole batch): q = RN16(s * a), entries of
    // steps past the range -> dummy row.  Afterwards L is free for the next batch of loads.
    auto cook_batch = [&](int32_t s0, uint32_t token) {
      // `token` is 0 at run time but opaque to ptxas: it ties the conversion (and, through the registers of L,
      // the next batch of loads) behind the last read-modify-write of the batch that has just been scattered,
      // so the loads stay one whole scatter phase ahead of their first use instead of being interleaved
      const float scale = __uint_as_float(__float_as_uint(a.scale) | token);
#pragma unroll
      for (int s = 0; s < K; ++s) {
        const bool valid = cta_r0 + (int64_t)(s0 + s) * R + r <= last_row;
#pragma unroll
        for (int k = 0; k < H2; ++k) W.q[s][k] = pack_rn(L.a[s][2 * k] * scale, L.a[s][2 * k + 1] * scale);
#pragma unroll
        for (int w = 0; w < EW; ++w) W.e[s][w] = valid ? L.e[s][w] : dummy_word;
      }
    };
    // a5: the batch is U = K * zeta sub-steps; sub-step u = (step s, t) of row-slot r updates block (r + t) mod zeta.
    // Software pipeline of depth D: the LDS of sub-step u is issued before the HFMA2/STS of sub-steps u-D .. u-1
    // and repeated after them by the lanes whose entry says one of those wrote the same sketch row.
    auto scatter_batch = [&]() -> uint32_t {
      constexpr int U = K * ZETA, D = DEPTH;
      static_assert(D <= kSmemFlagDepth, "reload flags must cover the pipeline depth");
      uint32_t acc[D + 1][H2];
      uint32_t last = 0;
      auto entry = [&](int u) -> uint32_t {  // 16-bit entry of sub-step u in the low half
        const uint32_t w = W.e[u / ZETA][(u % ZETA) >> 1];
        return ((u % ZETA) & 1) ? (w >> 16) : (w & 0xFFFFu);
      };
#pragma unroll
      for (int u = 0; u < U + D; ++u) {
        if (u < U) lds_h2<H2>((entry(u) & kE16Bucket) * pitch + lane_base, acc[u % (D + 1)]);
        const int v = u - D;
        if (v >= 0) {
          const uint32_t ev = entry(v);
          const uint32_t addr = (ev & kE16Bucket) * pitch + lane_base;
          // sign bit of the entry replicated into both halves, XOR +1.0: +-1.0 in both halves
          const uint32_t mult = (((ev & 0x8000u) * 0x10001u)) ^ 0x3C003C00u;
          lds_h2_if<H2>(ev & kE16Reload, addr, acc[v % (D + 1)]);
#pragma unroll
          for (int k = 0; k < H2; ++k) acc[v % (D + 1)][k] = hfma2_bits(W.q[v / ZETA][k], mult, acc[v % (D + 1)][k]);
          sts_h2<H2>(addr, acc[v % (D + 1)]);
          __syncwarp();  // a later sub-step of another lane may read this word
          last = acc[v % (D + 1)][0];
        }
      }
      return last & g.zero;
    };

    load_batch(0);
    cook_batch(0, 0u);
    load_batch(K);
    for (int32_t s0 = 0; s0 < nsteps; s0 += K) {
      const uint32_t token = scatter_batch();  // the loads issued one iteration ago are in flight meanwhile
      cook_batch(s0 + K, token);               // first touch of L: everything in flight is a scatter phase old
      load_batch(s0 + 2 * K);                  // L is free again; consumed across the back-edge
    }
  }
  __syncthreads();

  // ---- flush: partial sketch -> B with 16-byte result-discarding REDs (layouts coincide: [d][n])
  {
    const uint4* z = reinterpret_cast<const uint4*>(smem_raw);
    const uint32_t n16 = (uint32_t)g.d * pitch / 16u;
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
