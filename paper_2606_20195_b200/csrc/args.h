// args.h -- plain argument structs passed by value to the scatter kernels (host + device); CUDA translation units only.
#pragma once
#include <stdint.h>

namespace sk {

// element type of the sketch (what the scatter accumulates in) and conversion rule of the 16-bit paths (RND_* = SKETCH_RN / _SR / _DITHER)
enum : int { OUT_F32 = 0, OUT_F16 = 1, OUT_BF16 = 2 };
enum : int { RND_RN = 0, RND_SR = 1, RND_DITHER = 2 };


// What a tensor-memory word accumulates (template parameter MODE of k_tmem):
//   TM_F16         two binary16 halves, RN conversion once per element, sign as the +-1 multiplier of HFMA2 (the hot path)
//   TM_BF16        two bfloat16 halves, same structure with cvt.rn.bf16x2 / fma.rn.bf16x2 (the BF16 control)
//   TM_F16_SR      binary16, stochastic conversion of every SIGNED contribution (R13/R14): the sign must
//   TM_F16_DITHER  enter before the conversion, so the convert-once trick does not apply; Eq. (6) likewise (R20/R21)
//   TM_F32         one FP32 value per word: the FP32-accumulate path privatised the same way (what privatisation buys
//                  without the precision change, Eq. (5))
enum : int { TM_F16 = 0, TM_BF16 = 1, TM_F16_SR = 2, TM_F16_DITHER = 3, TM_F32 = 4 };
__host__ __device__ constexpr int tm_fw(int mode) { return mode == TM_F32 ? 1 : 2; }              // features per word
__host__ __device__ constexpr bool tm_perj(int mode) { return mode == TM_F16_SR || mode == TM_F16_DITHER; }
__host__ __device__ constexpr int tm_out(int mode) { return mode == TM_F32 ? OUT_F32 : mode == TM_BF16 ? OUT_BF16 : OUT_F16; }
__host__ __device__ constexpr uint32_t tm_one(int mode) { return mode == TM_F32 ? 0x3F800000u : mode == TM_BF16 ? 0x3F803F80u : 0x3C003C00u; }

struct ScatterArgs {
  const float* A;       // first row of the range
  int64_t lda;          // elements
  int64_t row_begin;    // global index of A's first row (hash counter base)
  int64_t rows;         // rows in the range
  void* B;              // d x n sketch (or base of the replicas)
  int64_t replica_stride;  // elements between replicas
  int32_t replicas;
  int32_t n;
  int32_t zeta;
  uint32_t db;          // d / zeta
  uint64_t seed;
  uint64_t sr_seed;
  float scale;          // fp32(1/sqrt(zeta)), correctly rounded on the host (R5)
  uint32_t cpr;         // chunks of VEC columns per row = n / VEC
  uint32_t cpr_magic;   // ceil(2^32 / cpr): c / cpr == umulhi(c, magic) while c * cpr < 2^32; 0 = cpr is 1; ~0 = use c / cpr
  int64_t odd_tail;     // k_generic, FP16 straight into B: index of the last element when d*n is odd (added by CAS), else -1
  const void* packed;   // hash_mode 2: packed entries for global rows, index i*zeta + j (ranked u16 or u32); else nullptr
};


struct SmemArgs {
  ScatterArgs s;
  int64_t rows_per_cta;  // multiple of the kernel's ring rows (NQ*4); so is ScatterArgs::rows for this kernel
  int32_t d;
  uint32_t zero;  // always 0; the kernel uses it to build a scheduling dependency ptxas cannot fold away
};

struct SmallArgs {
  ScatterArgs s;          // packed unused (hashes on the fly); n even, lda even, A 8-byte aligned, B 4-byte aligned
  int64_t rows_per_warp;  // multiple of 16
  int32_t d;
};

struct TmemArgs {
  ScatterArgs s;  // packed unused (the producer warp hashes on the fly); lda % 4 == 0, A and B 16-byte aligned
  int32_t d;
  // fused right-hand side: b[rows] FP32 (first row of the range) is sketched into Sb (FP32, d entries per
  // replica) with the hashes the producer computes anyway; nullptr = none
  const float* rhs;
  float* Sb;
  int64_t sb_stride;     // elements between the replicas of Sb
  int32_t sb_replicas;   // CTA x adds into replica x % sb_replicas
};

constexpr int kFlatThreads = 256;

}  // namespace sk
