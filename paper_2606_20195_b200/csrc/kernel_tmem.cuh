// kernel_tmem.cuh -- tensor-memory-privatised scatter (FP16 RN / SR / dither, bfloat16, FP32 accumulate) for sm_100a.
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
// CTA = NW = 4 consumer warps + up to 4 producer warps, one per SM sub-partition (+ 1 right-hand-side warp when a fused b
// rides along), one CTA per SM (it allocates all 512 TMEM columns), persistent over stages of T rows (32 KiB of A, a ring
// of NS shared-memory slots).
//   producers : one TMA copy per stage -- cp.async.bulk for a contiguous tile, a 2-D tensor-map box
//               {N features x T rows} (cp.async.bulk.tensor.2d; rows past the end zero-filled) for strided rows and
//               column slices -- L2 evict-first, completion on an mbarrier; meanwhile their lanes compute the stage's
//               hashes ON THE FLY (a1: splitmix64 counter hash, one lane per row) and store per (row, block) an entry
//               {TMEM address or column offset of the sketch row, HFMA2 multiplier = +-1.0 in both halves}.
//               No separate hash pass, no packed hash array in HBM.
//   consumers : warp w owns TMEM lanes [32*(w%4), +32) (the hardware's lane quadrant of that warp): a private
//               (d/BQ) x 64X partial sketch.  The CTA's N = 64*X*S features are cut in S slices; warp w takes slice
//               w % S and bucket group (w / S) % BQ of the rows of row-set w / (S*BQ) of every stage.
//               Rows are processed in groups of G: all LDTMs of a group are issued, then one tcgen05.wait::ld, then
//               the HFMA2s and STTMs; tcgen05.wait::st orders a group's LDTMs behind the previous group's STTMs.
//               Two rows of a group that hit the same sketch row are chained in registers, kept apart by the producers
//               (deferral), or -- small sketches -- sent to private copies of the partial sketch (replicated rows);
//               see TmemGeom.
//   flush     : LDTM.x8 -> result-discarding vector REDs into B.
//
// Sketches larger than one warp's 512 TMEM columns (d * X > 512) are split two ways:
//   BQ bucket groups : the zeta stack blocks are cut into BQ groups of ZB = zeta / BQ consecutive blocks
//               (disjoint sketch-row ranges); a warp of group b holds only the d / BQ sketch
//               rows of its blocks and adds only those contributions.  Every row is then needed by BQ warps, so
//               the consumers first convert the stage ONCE into a shared FP16 tile (a3, a4) and scatter from that.
//   CS column slices : gridDim.y CTAs (1..16) share a row range, CTA y takes the features [y * N, (y + 1) * N) of
//               every row; the hashes are recomputed per slice.  n = 256: d = 1024 -> X = 2, BQ = 4, CS = 2;
//               d = 2048 -> X = 1, BQ = 4, CS = 4; the paper's n = 1024, d = 2048 -> X = 1, BQ = 4, CS = 16.
// Accumulation is in the MODE's own arithmetic throughout (FP16 RN on the hot path); the hierarchy is
// (warp-private partial [x G copies]) -> RED into B.
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
// no "memory" clobber: these order tensor-memory traffic only (volatile asms keep their mutual order), so the
// compiler may hoist the next group's shared-memory loads above them
SK_DEVINL void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;"); }
SK_DEVINL void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;"); }
// tcgen05.ld writes its registers asynchronously: every use must be ordered behind tcgen05.wait::ld.  An
// empty volatile asm that "modifies" the register gives the compiler that dependency at no cost.
SK_DEVINL void tmem_tie(uint32_t& v) { asm volatile("" : "+r"(v)); }

// acc + q * (+-1): one correctly rounded add per component, subnormals kept
template <int MODE> SK_DEVINL uint32_t tm_fma(uint32_t q, uint32_t mult, uint32_t acc) {
  uint32_t d;
  if constexpr (MODE == TM_F32) asm("fma.rn.f32 %0, %1, %2, %3;" : "=r"(d) : "r"(q), "r"(mult), "r"(acc));
  else if constexpr (MODE == TM_BF16) asm("fma.rn.bf16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(q), "r"(mult), "r"(acc));
  else asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(d) : "r"(q), "r"(mult), "r"(acc));
  return d;
}
// a3, a4 for an RN mode: two adjacent features -> one 16-bit pair
template <int MODE> SK_DEVINL uint32_t tm_pack(float x0, float x1) {
  if constexpr (MODE == TM_BF16) return pack_bf16_rn(x0, x1);
  else return pack_rn(x0, x1);
}

// ---------------------------------------------------------------------------------------- geometry
// rows per stage: 32 KiB of A per stage, at least 16 rows (4 stages x 32 KiB x 148 SMs = 19 MB in flight; with 16 KiB
// stages at n = 64 the consumers waited for data 36 % of their time, profiles/r01_tmem_shapes.md)
// (bucket-group kernels with more than one block per warp keep 64 rows at n = 64: their records, side lists and FP16
// tiles would not fit beside four 32 KiB tiles)
__host__ __device__ constexpr int tmem_stage_rows(int n, int bq, int zeta) {
  return n <= 64 ? ((bq == 1 || zeta == bq) ? 128 : 64) : n <= 128 ? 64 : n == 256 ? 32 : 16;
}
__host__ __device__ constexpr int tmem_stages(int n) { return n <= 512 ? 4 : 3; }
// bytes of one (row, bucket group) side-list item of the deferral modes: {row | slot << 16, 0, then (col, mul) x ZB}
__host__ __device__ constexpr int tmem_rec_bytes(int zb) { return zb == 1 ? 16 : 16 + 8 * zb; }

// GM = group mode: how two rows of one group that hit the same sketch row are kept from losing an update.
//   0      groups of G = 2 (4 for short block lists) rows; same-bucket rows are chained in registers.  Works for any
//          d, costs O(G^2) compares and selects per block, so G stays small and few LDTMs are in flight.
//   1, 2   DEFERRAL, groups of 4 / 8 rows, bucket-group kernels only (BQ > 1).  The producers find every row that
//          shares a sketch row -- in any stack block -- with a LATER row of its group (rare when d / zeta >> G^2).  Such a
//          row is deferred as a whole: its converted FP16 words are moved to a side buffer (the upper half of the stage's
//          FP32 tile, free once the stage is converted in place) and its tile row is zeroed, its main-loop records point,
//          in the clashing blocks, at a substitute sketch row that no row of the group touches (adding +0 there changes
//          nothing), and it is appended to per-stage side lists that the consumers apply one row at a time after the main
//          loop.  The main loop then has pairwise distinct TMEM addresses within a group by construction -- no compares, no
//          selects, 8 read-modify-writes in flight -- reads every row's FP16 words at a compile-time offset, and its records
//          are bare {address, multiplier} pairs (two rows per 16-byte load with one block per warp).
//   5      REPLICATED rows, for sketches a quarter the size of a warp's tensor-memory region or smaller (G (d / BQ) X <= 512
//          columns; c2: d = 128, X = 1): row r of a group adds into private copy r % G of the partial sketch, so the G
//          read-modify-writes of a block never share an address -- no compares, no selects, G = 4 in flight -- and the
//          copies are added in registers at the flush.  Classic privatisation one level further down; chained groups
//          spend about half of the consumer's instructions on the O(G^2) chain (c2: 161 instructions per KiB of A).
template <int ZETA, int X, int S, int BQ, int NW, int GM, int T, int MODE = TM_F16>
struct TmemGeom {
  static constexpr int FW = tm_fw(MODE);
  static_assert(!(GM == 1 || GM == 2) || MODE == TM_F16, "deferral modes exist for the FP16-RN path only");
  static_assert(!tm_perj(MODE) || BQ == 1, "per-contribution conversion: one bucket group");
  static_assert(NW % 4 == 0 && NW % (S * BQ) == 0, "consumer warps: whole lane quadrants, whole slice x bucket-group sets");
  static_assert(ZETA % BQ == 0, "bucket groups are whole stack blocks");
  static_assert(!(GM == 1 || GM == 2) || BQ > 1, "deferral needs the shared FP16 tile of the bucket-group kernels");
  static constexpr int ZB = ZETA / BQ;         // stack blocks one warp accumulates
  static constexpr int RS = NW / (S * BQ);     // row-sets per stage
  static constexpr int TR = T / RS;            // rows of a stage one warp processes
  static constexpr bool DEF = GM == 1 || GM == 2;
  static constexpr bool REPL = GM == 5;
  static constexpr bool ABS = S == 1;             // entries hold absolute tensor-memory addresses (see the producer)
  static constexpr int G = GM == 1 ? 4 : GM == 2 ? 8 : REPL ? (ZB >= 8 ? 2 : 4) : (ZB >= 4 || (BQ > 1 && ZB >= 2)) ? 2 : 4;  // rows per group (LDTMs in flight = G * ZB)
  static_assert(TR % G == 0 && 32 % G == 0, "whole groups");
  static constexpr int N = 32 * FW * X * S;    // features of the CTA's column slice
  static constexpr int WC = kTmemCols / (NW / 4);  // tensor-memory columns of one warp's private region
  static constexpr int A_BYTES = T * N * 4;
  // chained modes: entries [row][zeta] {col, mul}.  Deferral: records [BQ][row] of RB bytes (a warp's 32 rows of one
  // bucket group are stored side by side: no bank conflicts), then per (chunk phase,
  // bucket group) a side list of up to T items of RB bytes, then the NPC * BQ item counts.
  static constexpr int RB = tmem_rec_bytes(ZB);      // side-list item
  static constexpr int REC = 8 * ZB;                 // main-loop record {col, mul} x ZB
  static constexpr int E_BYTES = DEF ? T * BQ * REC : T * ZETA * 8;
  // producer warps: up to four, one per SM sub-partition.  A producer warp shares its sub-partition's issue slots with one
  // consumer warp and a stage is released when the SLOWEST consumer is done, so the hash stage is spread evenly: the
  // stage's 32-row chunks go to NPC warps and the stack blocks (deferral: the bucket groups) of a chunk to NPB warps
  static constexpr int CH = (T + 31) / 32;
  static constexpr int NPC = DEF ? (CH >= 2 ? 2 : 1) : (CH >= 4 ? 4 : CH >= 2 ? 2 : 1);
  static constexpr int NPB = DEF ? (BQ < 4 / NPC ? BQ : 4 / NPC) : (ZETA < 4 / NPC ? ZETA : 4 / NPC);
  static constexpr int NP = NPC * NPB;
  static constexpr int LCAP = T / NPC;         // rows one chunk phase hashes = the most it can defer
  static constexpr int L_BYTES = DEF ? NPC * BQ * LCAP * RB + 128 : 0;
  static constexpr int STAGE_BYTES = A_BYTES + E_BYTES + L_BYTES;
  static_assert(STAGE_BYTES % 128 == 0, "TMA destination alignment");
  // bucket groups: every row is needed by BQ warps, so the consumer warps first convert the stage ONCE into a
  // shared FP16 tile (a3, a4), meet at a named barrier, and then each scatters its own blocks from that tile.
  // Two tiles (stage parity); the deferral modes append one all-zero row to each.
  static constexpr bool SHQ = BQ > 1 && (MODE == TM_F16 || MODE == TM_BF16);   // FP32 words are read from the A tile itself
  // deferral modes: the PRODUCER warps convert the stage, in place (the FP16 tile takes the first half of the FP32
  // tile's bytes), once its TMA copy has landed; the consumers only scatter.  TMA runs NS - 1 stages ahead.
  static constexpr bool PCONV = DEF;
  static constexpr int Q_ROW = N * 2;
  static constexpr int Q_BYTES = T * Q_ROW + (DEF ? Q_ROW : 0);
  static_assert((T * N / 4) % (NW * 32) == 0, "whole conversion passes");
};

__host__ __device__ constexpr int tmem_producers(int n, int bq, int gm, int zeta) {
  const int ch = (tmem_stage_rows(n, bq, zeta) + 31) / 32;
  const bool def = gm == 1 || gm == 2;
  const int npc = !def ? (ch >= 4 ? 4 : ch >= 2 ? 2 : 1) : (ch >= 2 ? 2 : 1);
  const int split = !def ? zeta : bq;
  return npc * (split < 4 / npc ? split : 4 / npc);
}
// ring of stages | barriers + TMEM base (256 B) | chained bucket-group kernels: two converted (FP16) tiles | deferral:
// one all-zero FP16 row + 2 KiB of producer scratch (the sketch rows of a 32-row chunk, a 128-byte line per warp and block)
constexpr size_t tmem_smem_bytes(int zeta, int n, int bq, int gm_, int mode = TM_F16) {
  const int gm = (gm_ == 1 || gm_ == 2) ? gm_ : 0;   // only the deferral modes change the layout
  const size_t t = (size_t)tmem_stage_rows(n, bq, zeta);
  const size_t rb = (size_t)tmem_rec_bytes(zeta / bq);
  const size_t e = gm ? t * bq * (8 * (size_t)(zeta / bq)) + t * bq * rb + 128 : t * zeta * 8;   // records + side lists (T rows in all) + counts
  const bool shq = bq > 1 && (mode == TM_F16 || mode == TM_BF16);
  return (size_t)tmem_stages(n) * (t * n * 4 + e) + 256 + (gm ? 256 + 2048 : shq ? 2 * t * n * 2 : 0);
}

// a5 for R rows x ZB stack blocks of one warp: LDTM, one RN16 add per half (fma.rn.f16x2 by +-1), STTM.
// CHAIN: two rows of the call that hit the same sketch row are chained in registers (the later row adds onto
// the earlier row's result and both store the chain's final value; the bucket is warp-uniform, so this is a
// select, not divergence).  Without CHAIN the caller guarantees distinct sketch rows within a block.
template <int R, int ZB, int X, bool CHAIN, int MODE = TM_F16>
SK_DEVINL void tmem_rmw(uint32_t region, const uint32_t (*q)[tm_perj(MODE) ? ZB : 1][X], const uint32_t (*col)[ZB], const uint32_t (*mul)[ZB]) {
  constexpr bool PERJ = tm_perj(MODE);         // q differs per stack block (the sign went in before the conversion)
  uint32_t acc[R][ZB][X];
  tmem_wait_st();                              // the previous stores are in TMEM
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int j = 0; j < ZB; ++j) tmem_ld<X>(region + col[r][j], acc[r][j]);
  tmem_wait_ld();
#pragma unroll
  for (int r = 0; r < R; ++r)
#pragma unroll
    for (int j = 0; j < ZB; ++j)
#pragma unroll
      for (int k = 0; k < X; ++k) tmem_tie(acc[r][j][k]);
#pragma unroll
  for (int j = 0; j < ZB; ++j) {
#pragma unroll
    for (int r = 0; r < R; ++r) {
      if constexpr (CHAIN) {
#pragma unroll
        for (int p = 0; p < r; ++p) {
          const bool same = col[p][j] == col[r][j];
#pragma unroll
          for (int k = 0; k < X; ++k) acc[r][j][k] = same ? acc[p][j][k] : acc[r][j][k];
        }
      }
#pragma unroll
      for (int k = 0; k < X; ++k) acc[r][j][k] = tm_fma<MODE>(q[r][PERJ ? j : 0][k], PERJ ? tm_one(MODE) : mul[r][j], acc[r][j][k]);
    }
    if constexpr (CHAIN) {
#pragma unroll
      for (int r = R - 2; r >= 0; --r) {
#pragma unroll
        for (int p = R - 1; p > r; --p) {
          const bool same = col[p][j] == col[r][j];
#pragma unroll
          for (int k = 0; k < X; ++k) acc[r][j][k] = same ? acc[p][j][k] : acc[r][j][k];
        }
      }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) tmem_st<X>(region + col[r][j], acc[r][j]);
  }
}

// FP16 words of one lane (X half2) from the shared converted tile
template <int X> SK_DEVINL void lds_q(const unsigned char* p, uint32_t (&q)[X]) {
  if constexpr (X == 1) q[0] = *reinterpret_cast<const uint32_t*>(p);
  else if constexpr (X == 2) { const uint2 t = *reinterpret_cast<const uint2*>(p); q[0] = t.x; q[1] = t.y; }
  else { const uint4 t = *reinterpret_cast<const uint4*>(p); q[0] = t.x; q[1] = t.y; q[2] = t.z; q[3] = t.w; }
}
// record / side-list item of the deferral modes -> head word (q offset or row), (col, mul) x ZB
template <int ZB> SK_DEVINL void lds_rec(const unsigned char* p, uint32_t& head, uint32_t (&col)[ZB], uint32_t (&mul)[ZB]) {
  const uint4 t = *reinterpret_cast<const uint4*>(p);
  head = t.x;
  if constexpr (ZB == 1) { col[0] = t.z; mul[0] = t.w; }
  else {
#pragma unroll
    for (int k = 0; k < ZB / 2; ++k) {
      const uint4 u = *reinterpret_cast<const uint4*>(p + 16 + 16 * k);
      col[2 * k] = u.x; mul[2 * k] = u.y; col[2 * k + 1] = u.z; mul[2 * k + 1] = u.w;
    }
  }
}
template <int ZB> SK_DEVINL void sts_rec(uint32_t p, uint32_t head, const uint32_t (&col)[ZB], const uint32_t (&mul)[ZB]) {
  if constexpr (ZB == 1) {
    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(p), "r"(head), "r"(0u), "r"(col[0]), "r"(mul[0]) : "memory");
  } else {
    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%2,%2};" ::"r"(p), "r"(head), "r"(0u) : "memory");
#pragma unroll
    for (int k = 0; k < ZB / 2; ++k)
      asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(p + 16 + 16 * k), "r"(col[2 * k]), "r"(mul[2 * k]), "r"(col[2 * k + 1]), "r"(mul[2 * k + 1]) : "memory");
  }
}

// ---------------------------------------------------------------------------------------- the kernel
template <int ZETA, int X, int S, int BQ, int NW, int GM, int MODE>
__global__ void __launch_bounds__((NW + tmem_producers(32 * tm_fw(MODE) * X * S, BQ, GM, ZETA) + 1) * 32, 1) k_tmem(TmemArgs g, const __grid_constant__ CUtensorMap tmap) {
  constexpr int FW = tm_fw(MODE);
  constexpr int T = tmem_stage_rows(32 * FW * X * S, BQ, ZETA), NS = tmem_stages(32 * FW * X * S);
  using Geo = TmemGeom<ZETA, X, S, BQ, NW, GM, T, MODE>;
  constexpr int TR = Geo::TR, G = Geo::G, N = Geo::N, ZB = Geo::ZB, RB = Geo::RB, NP = Geo::NP, NPC = Geo::NPC, NPB = Geo::NPB;
  static_assert(NP == tmem_producers(N, BQ, GM, ZETA), "producer warps");
  constexpr int JB = ZETA / NPB;                     // stack blocks one producer warp hashes
  constexpr uint32_t Q0 = NS * Geo::STAGE_BYTES + 256;   // first converted tile (chained modes) / producer scratch (deferral)
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const ScatterArgs& a = g.s;
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

  // shared-memory carve-up: [NS][A tile | entries or records | side lists] then the barriers, then the FP16 tiles
  const uint32_t smem0 = smem_u32(smem_raw);
  const uint32_t bars = smem0 + NS * Geo::STAGE_BYTES;     // full[NS], empty[NS], 8 B each
  uint32_t* const tbase_p = reinterpret_cast<uint32_t*>(smem_raw + NS * Geo::STAGE_BYTES + 24 * NS);   // after full, empty, tma

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tbase_p)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 32) {
    for (int k = 0; k < NS; ++k) {
      mbar_init(bars + 8 * k, NP);             // full: one arrive per producer warp (+ the TMA transaction bytes)
      mbar_init(bars + 8 * (NS + k), NW);      // empty: one arrive per consumer warp
      mbar_init(bars + 8 * (2 * NS + k), 1);   // tma (producer-side conversion only): the issuing lane's arrive + the transaction bytes
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

  if (warp >= NW + NP) {
    // ================================================================ right-hand-side warp (launched only with a fused b)
    // PAPER.md:356 "b in FP32 with the same map": Sb[bucket(i, j)] += +-s b_i, one result-discarding FP32 RED per (row,
    // block), over the rows of this CTA's stages.  The warp shares nothing with the pipeline (it reads b from global memory
    // and recomputes the zeta hashes of its rows), so the kernels without a right-hand side carry none of it.
    if (g.rhs != nullptr) {
      float* const sb = g.Sb + (size_t)((blockIdx.x * gridDim.y + blockIdx.y) % (uint32_t)g.sb_replicas) * (size_t)g.sb_stride;
      // the CS column slices of a row range share its right-hand side: slice y takes every CS-th stage, starting at the y-th
      // (one warp on all of a range's rows would be latency-bound behind the pipeline: e1 3.2 ms against 2.65 ms without b).
      // The loads of a stage's (and of the next stage's) entries are issued before any of them is used.
      const int64_t step = (int64_t)gridDim.x * gridDim.y;
      constexpr int RI = (T + 31) / 32;
      float cur[RI], nxt[RI];
      auto fetch = [&](int64_t st, float (&v)[RI]) {
#pragma unroll
        for (int k = 0; k < RI; ++k) {
          const int64_t row = st * T + k * 32 + lane;
          v[k] = (st < nstages && k * 32 + (int)lane < T && row < a.rows) ? g.rhs[row] : 0.f;
        }
      };
      const int64_t st0 = blockIdx.x + (int64_t)blockIdx.y * gridDim.x;
      fetch(st0, cur);
      for (int64_t st = st0; st < nstages; st += step) {
        fetch(st + step, nxt);
#pragma unroll
        for (int k = 0; k < RI; ++k) {
          const int64_t row = st * T + k * 32 + lane;
          if (k * 32 + (int)lane < T && row < a.rows) {
            const float bv = __fmul_rn(a.scale, cur[k]);
            const uint64_t ctr0 = (uint64_t)(a.row_begin + row) * ZETA;
#pragma unroll
            for (int j = 0; j < ZETA; ++j) {
              const uint32_t e = hash_entry(a.seed, ctr0 + j, j, a.db);
              red_f1(sb + entry_bucket(e), __uint_as_float(__float_as_uint(bv) ^ entry_signmask_f32(e)));
            }
          }
        }
#pragma unroll
        for (int k = 0; k < RI; ++k) cur[k] = nxt[k];
      }
    }
  } else if (warp >= NW) {
    // ================================================================ producers: TMA + hash stage (a1, a2)
    const uint32_t pw = warp - NW;                 // producer warp pw: 32-row chunks cp, cp + NPC, ...; stack blocks [j0, j0 + JB)
    const uint32_t cp = pw % NPC, j0 = (pw / NPC) * JB, b0 = j0 / ZB;
    unsigned char* const scr = smem_raw + Q0 + 256 + pw * (JB * 128);   // deferral: [JB][32] sketch rows
    uint32_t* const xch = reinterpret_cast<uint32_t*>(smem_raw + Q0);  // deferral: [NPC][2][NPB] row masks exchanged by the warps of a chunk phase
    static_assert(!Geo::DEF || (NP * JB * 128 <= 2048 && NP * 2 * 4 <= 256), "producer scratch");
    const uint64_t policy = l2_evict_first_policy();
    const bool contiguous = (a.lda == N);          // implies a single column slice
    // a2: TMA copy of this CTA's k-th stage (producer warp 0).  Waits until the consumers have released the slot;
    // completion (bytes) on `full` (consumer-side conversion) or on `tma` (producer-side conversion)
    auto issue = [&](uint32_t k) {
      const int64_t st = blockIdx.x + (int64_t)k * gridDim.x;
      if (st >= nstages) return;
      const uint32_t slot = k % NS, ph = (k / NS) & 1;
      const uint32_t sA = smem0 + slot * Geo::STAGE_BYTES;
      const uint32_t bar = bars + 8 * ((Geo::PCONV ? 2 * NS : 0) + slot);
      mbar_wait(bars + 8 * (NS + slot), ph ^ 1);   // passes at once the first time round the ring
      if constexpr (Geo::PCONV) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the slot held generic-proxy writes (FP16 tile)
      const int64_t row0 = st * T;
      const int32_t nrows = (int32_t)min((int64_t)T, a.rows - row0);
      if (contiguous) {
        if (lane == 0) {
          mbar_expect_tx(bar, (uint32_t)nrows * N * 4);
          bulk_g2s(sA, a.A + row0 * a.lda, (uint32_t)nrows * N * 4, bar, policy);
        }
        if (nrows < T) {                         // last stage of the matrix: rows past the end contribute +0
          const uint32_t z0 = sA + nrows * N * 4, z1 = sA + Geo::A_BYTES;
          for (uint32_t p = z0 + lane * 16; p < z1; p += 32 * 16) asm volatile("st.shared.v4.b32 [%0], {%1,%1,%1,%1};" ::"r"(p), "r"(0u) : "memory");
        }
      } else if (lane == 0) {                    // strided rows / column slice: one tiled TMA copy per stage
        mbar_expect_tx(bar, (uint32_t)T * N * 4);
        tensor_g2s(sA, &tmap, (int32_t)col0, (int32_t)row0, bar, policy);
      }
      if constexpr (Geo::PCONV) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar);
      }
    };
    constexpr uint32_t AHEAD = NS - 1;
    if constexpr (Geo::PCONV) {
      if (pw == 0)
        for (uint32_t k = 0; k < AHEAD; ++k) issue(k);
    }
    uint32_t it = 0;
    for (int64_t st = blockIdx.x; st < nstages; st += gridDim.x, ++it) {
      const uint32_t slot = it % NS, ph = (it / NS) & 1;
      const uint32_t sA = smem0 + slot * Geo::STAGE_BYTES, sE = sA + Geo::A_BYTES, sL = sE + Geo::E_BYTES;
      const uint32_t full = bars + 8 * slot, empty = bars + 8 * (NS + slot);
      const int64_t row0 = st * T;
      if constexpr (Geo::PCONV) {
        if (pw != 0) mbar_wait(empty, ph ^ 1);   // warp 0 waited before it issued this stage's copy
      } else {
        if (pw == 0) issue(it);
        else mbar_wait(empty, ph ^ 1);
      }
      // a1: rows lane, lane + 32, ... of the stage
      uint32_t cnt = 0;                        // deferral: rows deferred so far in this chunk phase (warp-uniform)
#pragma unroll
      for (int rr = (int)cp; rr < (T + 31) / 32; rr += NPC) {
        const int32_t r = rr * 32 + (int32_t)lane;
        const bool live = (T % 32 == 0) || r < T;   // stages of 16 rows (n >= 512): half a warp's rows exist
        const uint64_t ctr0 = (uint64_t)(a.row_begin + row0 + r) * ZETA;
        uint32_t bk[JB], mulw[JB];             // sketch row, +-1.0 | +-1.0 of blocks j0 + j
#pragma unroll
        for (int j = 0; j < JB; ++j) {
          const uint32_t e = hash_entry(a.seed, ctr0 + j0 + j, j0 + j, a.db);
          bk[j] = entry_bucket(e);
          mulw[j] = tm_one(MODE) ^ (MODE == TM_F32 ? entry_signmask_f32(e) : entry_signmask_h2(e));
        }
        // region of the consumer warp that owns (this row, bucket group b) when there is one feature slice
        auto abase = [&](uint32_t b) -> uint32_t {
          if constexpr (!Geo::ABS) return 0u;
          const uint32_t w = b + (uint32_t)BQ * ((uint32_t)r / TR);
          return tbase + (((w & 3u) * 32u) << 16) + (w >> 2) * (uint32_t)Geo::WC;
        };
        if constexpr (!Geo::DEF) {
          // entries {(bucket - first sketch row of the block's group) * X, multiplier}.  With one feature slice the
          // entry of (row, bucket group) is read by exactly one consumer warp, so it carries that warp's complete
          // tensor-memory address (abase) and the consumer saves an add per (row, block)
          if (live) {
            const uint32_t p = sE + r * (ZETA * 8) + j0 * 8;
            // replicated rows: row r of a group adds into private copy r % G of the warp's partial sketch
            const uint32_t copy = Geo::REPL ? ((uint32_t)r % (uint32_t)G) * (dloc * X) : 0u;
            auto ent = [&](int j) -> uint32_t { const uint32_t bg = (j0 + (uint32_t)j) / ZB; return abase(bg) + (bk[j] - bg * dloc) * X + copy; };
            if constexpr (JB == 1) asm volatile("st.shared.v2.b32 [%0], {%1,%2};" ::"r"(p), "r"(ent(0)), "r"(mulw[0]) : "memory");
            else {
#pragma unroll
              for (int k = 0; k < JB / 2; ++k)
                asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(p + 16 * k), "r"(ent(2 * k)), "r"(mulw[2 * k]), "r"(ent(2 * k + 1)), "r"(mulw[2 * k + 1]) : "memory");
            }
          }
        } else {
          // deferral (see TmemGeom): ls bit j = a later row of my group of G rows has my sketch row in block j
          // the group's sketch rows go through shared memory (one store, G/4 broadcast loads per block; a MATCH.ANY
          // over 32 distinct keys costs ~200 cycles, G - 1 shuffles about as many instructions)
          const uint32_t pg = lane % G;
          uint32_t ls = 0, og[JB][G];
          __syncwarp();
#pragma unroll
          for (int j = 0; j < JB; ++j) reinterpret_cast<uint32_t*>(scr + j * 128)[lane] = bk[j];
          __syncwarp();
#pragma unroll
          for (int j = 0; j < JB; ++j) {
#pragma unroll
            for (int k = 0; k < G / 4; ++k) {
              const uint4 t = *reinterpret_cast<const uint4*>(scr + j * 128 + (lane - pg) * 4 + 16 * k);
              og[j][4 * k] = t.x; og[j][4 * k + 1] = t.y; og[j][4 * k + 2] = t.z; og[j][4 * k + 3] = t.w;
            }
            uint32_t eq = 0;                     // bit i: row i of my group has my sketch row
#pragma unroll
            for (int i = 0; i < G; ++i) eq |= (og[j][i] == bk[j] ? 1u : 0u) << i;
            if ((eq >> (pg + 1)) != 0u) ls |= 1u << j;
          }
          if (!live) ls = 0;
          // the row is deferred as a whole when any block clashes: OR over the NPB warps that share this chunk (they walk
          // the chunks in lockstep; masks through shared memory, one named barrier per chunk phase)
          uint32_t dmask = __ballot_sync(0xFFFFFFFFu, ls != 0u);
          if constexpr (NPB > 1) {
            const uint32_t par = ((uint32_t)rr / NPC) & 1u;          // double-buffered: the next chunk's store cannot overtake a partner's read
            if (lane == 0) xch[(cp * 2 + par) * NPB + pw / NPC] = dmask;
            asm volatile("bar.sync %0, %1;" ::"r"(3 + cp), "n"(NPB * 32) : "memory");
#pragma unroll
            for (int k = 0; k < NPB; ++k) dmask |= xch[(cp * 2 + par) * NPB + k];
          }
          const bool def = (dmask >> lane) & 1u;
          uint32_t fb[JB];                     // sketch row the main loop touches
#pragma unroll
          for (int j = 0; j < JB; ++j) fb[j] = bk[j];
          // substitute sketch row in a clashing block: first of j*db + pg, + G, + 2G, ... that no row of the group
          // hashed to.  Different rows of a group draw from different residue classes mod G, so two substitutes never
          // coincide; at most G candidates are taken, hence the host requires d / zeta >= G * (G + 1).
#pragma unroll
          for (int j = 0; j < JB; ++j) {
            if (__any_sync(0xFFFFFFFFu, (ls >> j) & 1u)) {
              const uint32_t base = (j0 + (uint32_t)j) * a.db + pg;
              uint32_t taken = 0;              // bit t: candidate base + t*G is some row's sketch row
#pragma unroll
              for (int k = 0; k < G; ++k) {
                const uint32_t diff = og[j][k] - base;   // wraps to a huge value when that row lies below base
                if ((diff % G) == 0u && diff / G <= (uint32_t)G) taken |= 1u << (diff / G);
              }
              if ((ls >> j) & 1u) fb[j] = base + (uint32_t)(__ffs((int)~taken) - 1) * G;
            }
          }
#pragma unroll
          // side-buffer slot of a deferred row = its position among the deferred rows of this chunk phase (the same in
          // every bucket group's list)
          const uint32_t pos = cnt + __popc(dmask & ((1u << lane) - 1u));
#pragma unroll
          for (int bb = 0; bb < BQ / NPB; ++bb) {  // my bucket groups b0 + bb
            const uint32_t b = b0 + bb;
            uint32_t cm[ZB], co[ZB], mm[ZB];
#pragma unroll
            for (int jj = 0; jj < ZB; ++jj) {
              cm[jj] = abase(b) + (fb[bb * ZB + jj] - b * dloc) * X;
              co[jj] = abase(b) + (bk[bb * ZB + jj] - b * dloc) * X;
              mm[jj] = mulw[bb * ZB + jj];
            }
            if (live) {
              const uint32_t pr = sE + (b * (uint32_t)T + (uint32_t)r) * Geo::REC;
              if constexpr (ZB == 1) asm volatile("st.shared.v2.b32 [%0], {%1,%2};" ::"r"(pr), "r"(cm[0]), "r"(mm[0]) : "memory");
              else {
#pragma unroll
                for (int k = 0; k < ZB / 2; ++k)
                  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(pr + 16 * k), "r"(cm[2 * k]), "r"(mm[2 * k]), "r"(cm[2 * k + 1]), "r"(mm[2 * k + 1]) : "memory");
              }
            }
            if (def) sts_rec<ZB>(sL + ((cp * BQ + b) * Geo::LCAP + pos) * RB, (uint32_t)r | ((cp * (uint32_t)Geo::LCAP + pos) << 16), co, mm);
          }
          cnt += __popc(dmask);
        }
      }
      if constexpr (Geo::DEF) {
        if (lane < BQ / NPB) asm volatile("st.shared.b32 [%0], %1;" ::"r"(sL + NPC * BQ * Geo::LCAP * RB + (cp * BQ + b0 + lane) * 4), "r"(cnt) : "memory");
      }
      if constexpr (Geo::PCONV) {
        // a3, a4 once per element, in place: FP16 word pair k of the tile lands on bytes [8k, 8k + 8), i.e. on FP32 data
        // that an earlier pass (or, in the first pass, this pass before the barrier) has already read
        mbar_wait(bars + 8 * (2 * NS + slot), ph);
        constexpr uint32_t P = NP * 32;
        constexpr int CI = (T * N / 4) / P, CB = CI < 16 ? CI : 16;
        static_assert((T * N / 4) % P == 0 && CI % CB == 0, "whole conversion passes");
        const uint32_t ptid = pw * 32 + lane;
        const float4* const tile = reinterpret_cast<const float4*>(smem_raw + slot * Geo::STAGE_BYTES);
        uint2* const qt = reinterpret_cast<uint2*>(smem_raw + slot * Geo::STAGE_BYTES);
        const float scale = a.scale;
#pragma unroll 1
        for (int i0 = 0; i0 < CI; i0 += CB) {
          float4 t[CB];
#pragma unroll
          for (int i = 0; i < CB; ++i) t[i] = tile[(uint32_t)(i0 + i) * P + ptid];
          if constexpr (NP > 1) asm volatile("bar.sync 2, %0;" ::"n"(P) : "memory");
          else __syncwarp();
#pragma unroll
          for (int i = 0; i < CB; ++i)
            qt[(uint32_t)(i0 + i) * P + ptid] = make_uint2(pack_rn(t[i].x * scale, t[i].y * scale), pack_rn(t[i].z * scale, t[i].w * scale));
        }
        // deferred rows (a few per thousand): FP16 words -> side buffer (upper half of the tile), tile row <- 0.  The warps
        // that hold the first bucket groups of a chunk phase move the rows of that phase, once every warp's stores are in.
        if constexpr (NP > 1) asm volatile("bar.sync 2, %0;" ::"n"(P) : "memory");
        else __syncwarp();
        if (pw < NPC && cnt != 0u) {
          unsigned char* const q0 = smem_raw + slot * Geo::STAGE_BYTES;
          unsigned char* const sq = q0 + T * Geo::Q_ROW;
          const unsigned char* const items = smem_raw + slot * Geo::STAGE_BYTES + Geo::A_BYTES + Geo::E_BYTES + (cp * BQ + b0) * Geo::LCAP * RB;
          for (uint32_t i = 0; i < cnt; ++i) {
            const uint32_t head = *reinterpret_cast<const uint32_t*>(items + i * RB);
            const uint32_t row = head & 0xFFFFu, sl = head >> 16;
            for (uint32_t o = lane * 4; o < (uint32_t)Geo::Q_ROW; o += 128) {
              *reinterpret_cast<uint32_t*>(sq + sl * Geo::Q_ROW + o) = *reinterpret_cast<const uint32_t*>(q0 + row * Geo::Q_ROW + o);
              *reinterpret_cast<uint32_t*>(q0 + row * Geo::Q_ROW + o) = 0u;
            }
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(full);
      if constexpr (Geo::PCONV) {
        if (pw == 0) issue(it + AHEAD);
      }
    }
  } else {
    // ================================================================ consumers: a3, a4, a5 in tensor memory
    const uint32_t slice = warp % S, bgrp = (warp / S) % BQ, rowset = warp / (S * BQ);
    const uint32_t region = tbase + (((warp & 3u) * 32u) << 16) + (warp >> 2) * (uint32_t)Geo::WC;
    const uint32_t ncols = dloc * X;  // multiple of 8, <= WC (host check); replicated rows: G copies, G * ncols <= WC
    for (uint32_t c = 0; c < ncols * (Geo::REPL ? G : 1); c += 8) tmem_st8_zero(region + c);   // a0 (private part)
    tmem_wait_st();

    const float scale = a.scale;
    const uint32_t a_off = (rowset * TR) * (N * 4) + (slice * 32 * FW * X + lane * FW * X) * 4;
    // per-contribution conversion (SR / dither): counter of this lane's first column pair (R14: (row zeta + j) ceil(n/2) + pair)
    [[maybe_unused]] const uint64_t npairs = ((uint64_t)a.n + 1u) >> 1;
    [[maybe_unused]] const uint64_t pair0 = ((uint64_t)col0 + slice * 64 * X + lane * 2 * X) >> 1;
    const uint32_t e_off = Geo::DEF ? (bgrp * T + rowset * TR) * Geo::REC : (rowset * TR) * (ZETA * 8) + bgrp * (ZB * 8);
    uint32_t it = 0;
    for (int64_t st = blockIdx.x; st < nstages; st += gridDim.x, ++it) {
      const uint32_t slot = it % NS, ph = (it / NS) & 1;
      const unsigned char* const sA = smem_raw + slot * Geo::STAGE_BYTES + a_off;
      const unsigned char* const sE = smem_raw + slot * Geo::STAGE_BYTES + Geo::A_BYTES + e_off;
      mbar_wait(bars + 8 * slot, ph);
      const unsigned char* qlane = nullptr;    // this lane's words of row 0 of the converted tile
      if constexpr (Geo::PCONV) {
        qlane = smem_raw + slot * Geo::STAGE_BYTES + (slice * 64 * X + lane * 2 * X) * 2;   // converted in place by the producers
      } else if constexpr (Geo::SHQ) {
        // a3, a4 once per element: the whole stage -> FP16 tile `it & 1` (row pitch N * 2 bytes)
        const float4* const tile = reinterpret_cast<const float4*>(smem_raw + slot * Geo::STAGE_BYTES);
        unsigned char* const qb = smem_raw + Q0 + (it & 1u) * Geo::Q_BYTES;
        constexpr int CI = (T * N / 4) / (NW * 32), CB = (BQ >= 4 && CI >= 16) ? 16 : (CI < 8 ? CI : 8);   // loads in batches of CB (the stores may alias for all the compiler knows; 16 measured +1-2 % with four bucket groups, -5 % with two)
#pragma unroll
        for (int i0 = 0; i0 < CI; i0 += CB) {
          float4 t[CB];
#pragma unroll
          for (int i = 0; i < CB; ++i) t[i] = tile[(uint32_t)(i0 + i) * (NW * 32) + tid];
#pragma unroll
          for (int i = 0; i < CB; ++i)
            reinterpret_cast<uint2*>(qb)[(uint32_t)(i0 + i) * (NW * 32) + tid] =
                make_uint2(tm_pack<MODE>(t[i].x * scale, t[i].y * scale), tm_pack<MODE>(t[i].z * scale, t[i].w * scale));
        }
        // all consumer warps: tile `it & 1` is complete, and every warp is done scattering tile `(it - 1) & 1`
        asm volatile("bar.sync 1, %0;" ::"n"(NW * 32) : "memory");
        qlane = qb + (slice * 64 * X + lane * 2 * X) * 2;
      }
      if constexpr (Geo::DEF) {
        // software pipeline over the groups of the stage: records two groups ahead, FP16 words one group ahead of the
        // read-modify-write that uses them (their shared-memory latency hides under the tensor-memory round trip)
        constexpr int NG = TR / G;
        uint32_t col[3][G][ZB], mul[3][G][ZB], q[2][G][1][X];
        // records of a group of G rows: {col, mul} x ZB per row, rows side by side (ZB = 1: two rows per 16-byte load)
        auto lds_group = [&](int gi, uint32_t (&c)[G][ZB], uint32_t (&m)[G][ZB]) {
          const unsigned char* pg = sE + gi * G * Geo::REC;
          if constexpr (ZB == 1) {
#pragma unroll
            for (int r = 0; r < G; r += 2) {
              const uint4 t = *reinterpret_cast<const uint4*>(pg + r * 8);
              c[r][0] = t.x; m[r][0] = t.y; c[r + 1][0] = t.z; m[r + 1][0] = t.w;
            }
          } else {
#pragma unroll
            for (int r = 0; r < G; ++r)
#pragma unroll
              for (int k = 0; k < ZB / 2; ++k) {
                const uint4 t = *reinterpret_cast<const uint4*>(pg + r * Geo::REC + 16 * k);
                c[r][2 * k] = t.x; m[r][2 * k] = t.y; c[r][2 * k + 1] = t.z; m[r][2 * k + 1] = t.w;
              }
          }
        };
        const unsigned char* const qrow = qlane + (rowset * TR) * Geo::Q_ROW;
        lds_group(0, col[0], mul[0]);
        if constexpr (NG > 1) lds_group(1, col[1], mul[1]);
#pragma unroll
        for (int r = 0; r < G; ++r) lds_q<X>(qrow + r * Geo::Q_ROW, q[0][r][0]);
#pragma unroll
        for (int gi = 0; gi < NG; ++gi) {
          if (gi + 1 < NG) {
#pragma unroll
            for (int r = 0; r < G; ++r) lds_q<X>(qrow + ((gi + 1) * G + r) * Geo::Q_ROW, q[(gi + 1) & 1][r][0]);
          }
          if (gi + 2 < NG) lds_group(gi + 2, col[(gi + 2) % 3], mul[(gi + 2) % 3]);
          // a5: read-modify-write of G x ZB sketch rows in tensor memory, pairwise distinct by construction
          tmem_rmw<G, ZB, X, false>(Geo::ABS ? 0u : region, q[gi & 1], col[gi % 3], mul[gi % 3]);
        }
      } else {
#pragma unroll
      for (int g0 = 0; g0 < TR; g0 += G) {
        constexpr bool PERJ = tm_perj(MODE);
        uint32_t q[G][PERJ ? ZB : 1][X], col[G][ZB], mul[G][ZB];
        [[maybe_unused]] float v[G][FW * X];     // PERJ: the scaled products, converted per stack block below
#pragma unroll
        for (int r = 0; r < G; ++r) {
          {
            if constexpr (Geo::SHQ) {
              lds_q<X>(qlane + (rowset * TR + g0 + r) * Geo::Q_ROW, q[r][0]);
            } else {
              // a2 (from the staged tile), a3: p = s * a for this lane's FW * X features
              const unsigned char* pa = sA + (g0 + r) * (N * 4);
              if constexpr (FW * X == 1) { v[r][0] = *reinterpret_cast<const float*>(pa); }
              else if constexpr (FW * X == 2) { const float2 t = *reinterpret_cast<const float2*>(pa); v[r][0] = t.x; v[r][1] = t.y; }
              else {
#pragma unroll
                for (int k = 0; k < FW * X / 4; ++k) {
                  const float4 t = *reinterpret_cast<const float4*>(pa + 16 * k);
                  v[r][4 * k] = t.x; v[r][4 * k + 1] = t.y; v[r][4 * k + 2] = t.z; v[r][4 * k + 3] = t.w;
                }
              }
#pragma unroll
              for (int k = 0; k < FW * X; ++k) v[r][k] *= scale;
              // a4 for the convert-once modes: RN16 / RN-bf16 of two features per word, or the FP32 product itself
              if constexpr (MODE == TM_F32) {
#pragma unroll
                for (int k = 0; k < X; ++k) q[r][0][k] = __float_as_uint(v[r][k]);
              } else if constexpr (!PERJ) {
#pragma unroll
                for (int k = 0; k < X; ++k) q[r][0][k] = tm_pack<MODE>(v[r][2 * k], v[r][2 * k + 1]);
              }
            }
            const unsigned char* pe = sE + (g0 + r) * (ZETA * 8);
            if constexpr (ZB == 1) { const uint2 t = *reinterpret_cast<const uint2*>(pe); col[r][0] = t.x; mul[r][0] = t.y; }
            else {
#pragma unroll
              for (int k = 0; k < ZB / 2; ++k) {
                const uint4 t = *reinterpret_cast<const uint4*>(pe + 16 * k);
                col[r][2 * k] = t.x; mul[r][2 * k] = t.y; col[r][2 * k + 1] = t.z; mul[r][2 * k + 1] = t.w;
              }
            }
            if constexpr (PERJ) {
              // a4 per contribution: convert the SIGNED product of (row, block j) with that contribution's own random bits
              const uint64_t grow = (uint64_t)(a.row_begin + st * T + rowset * TR + g0 + r);
#pragma unroll
              for (int j = 0; j < ZB; ++j) {
                const uint32_t sf = (mul[r][j] & 0x8000u) << 16;
                const uint64_t ctr = (grow * ZETA + (bgrp * ZB + j)) * npairs + pair0;
#pragma unroll
                for (int k = 0; k < X; ++k)
                  q[r][j][k] = pack_f16<MODE == TM_F16_SR ? RND_SR : RND_DITHER>(__uint_as_float(__float_as_uint(v[r][2 * k]) ^ sf),
                                                                                 __uint_as_float(__float_as_uint(v[r][2 * k + 1]) ^ sf), a.sr_seed, ctr + k);
              }
            }
          }
        }
        // a5: read-modify-write of G x ZB sketch rows in tensor memory; same-bucket rows chained in registers
        tmem_rmw<G, ZB, X, !Geo::REPL, MODE>(Geo::ABS ? 0u : region, q, col, mul);
      }
      }
      if constexpr (Geo::DEF) {
        // the deferred rows of this stage (TmemGeom): original sketch rows, one row at a time
        const unsigned char* const sL = smem_raw + slot * Geo::STAGE_BYTES + Geo::A_BYTES + Geo::E_BYTES;
#pragma unroll 1
        for (uint32_t pl = 0; pl < (uint32_t)NPC; ++pl) {
          const uint32_t cnt = *reinterpret_cast<const uint32_t*>(sL + NPC * BQ * Geo::LCAP * RB + (pl * BQ + bgrp) * 4);
#pragma unroll 1
          for (uint32_t i = 0; i < cnt; ++i) {
            uint32_t head, q1[1][1][X], c1[1][ZB], m1[1][ZB];
            lds_rec<ZB>(sL + ((pl * BQ + bgrp) * Geo::LCAP + i) * RB, head, c1[0], m1[0]);
            if ((head & 0xFFFFu) / TR != rowset) continue;
            lds_q<X>(qlane + (T + (head >> 16)) * Geo::Q_ROW, q1[0][0]);   // the row's FP16 words, from the side buffer
            tmem_rmw<1, ZB, X, false>(Geo::ABS ? 0u : region, q1, c1, m1);
          }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bars + 8 * (NS + slot));
    }

    // ---- flush: private partial sketch -> B with result-discarding vector REDs (a5's last level)
    tmem_wait_st();
    constexpr int OUT = tm_out(MODE);
    const size_t b_off = (size_t)(bgrp * dloc) * a.n + col0 + slice * 32 * FW * X + lane * FW * X;   // elements
    for (uint32_t c = 0; c < ncols; c += 8) {
      uint32_t v[8];
      tmem_ld8(region + c, v);
      if constexpr (Geo::REPL) {
        // the G private copies of these sketch rows, added in the mode's own arithmetic (one more level of the hierarchy)
        uint32_t w[G - 1][8];
#pragma unroll
        for (int cp = 1; cp < G; ++cp) tmem_ld8(region + cp * ncols + c, w[cp - 1]);
        tmem_wait_ld();
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          tmem_tie(v[k]);
#pragma unroll
          for (int cp = 1; cp < G; ++cp) { tmem_tie(w[cp - 1][k]); v[k] = tm_fma<MODE>(w[cp - 1][k], tm_one(MODE), v[k]); }
        }
      } else {
        tmem_wait_ld();
#pragma unroll
        for (int k = 0; k < 8; ++k) tmem_tie(v[k]);
      }
#pragma unroll
      for (int b = 0; b < 8 / X; ++b) {
        const size_t e_off = b_off + (size_t)(c / X + b) * a.n;
        if constexpr (MODE == TM_F32) {
          float* dst = reinterpret_cast<float*>(a.B) + e_off;
          if constexpr (X == 1) { if (v[b] != 0u) red_f1(dst, __uint_as_float(v[b])); }
          else if constexpr (X == 2) { if ((v[2 * b] | v[2 * b + 1]) != 0u) red_f2(dst, __uint_as_float(v[2 * b]), __uint_as_float(v[2 * b + 1])); }
          else { if ((v[4 * b] | v[4 * b + 1] | v[4 * b + 2] | v[4 * b + 3]) != 0u) red_f4(dst, __uint_as_float(v[4 * b]), __uint_as_float(v[4 * b + 1]), __uint_as_float(v[4 * b + 2]), __uint_as_float(v[4 * b + 3])); }
        } else {
          uint16_t* dst = reinterpret_cast<uint16_t*>(a.B) + e_off;
          if constexpr (X == 1) { if (v[b] != 0u) red_p2<OUT>(dst, v[b]); }
          else if constexpr (X == 2) { if ((v[2 * b] | v[2 * b + 1]) != 0u) red_p4<OUT>(dst, v[2 * b], v[2 * b + 1]); }
          else { if ((v[4 * b] | v[4 * b + 1] | v[4 * b + 2] | v[4 * b + 3]) != 0u) red_p8<OUT>(dst, v[4 * b], v[4 * b + 1], v[4 * b + 2], v[4 * b + 3]); }
        }
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tbase) : "memory");
}

}  // namespace sk
