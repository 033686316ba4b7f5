// args.h -- plain argument structs passed by value to the scatter kernels (host + device).
#pragma once
#include <stdint.h>

namespace sk {

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
};

constexpr int kFlatThreads = 256;

}  // namespace sk
