// sketch_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU restatement of what the sparse-sketch hot
// path computes (paper arxiv 2606.20195, "On the Robustness of Sparse
// Randomized Sketching to FP16 Rounding on GPUs").  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may build, load or call this file.  It shares no code, header, table or
// constant generator with paper_2606_20195_b200/csrc/ and includes nothing
// from it.
//
// Each function cites the passage it restates (PAPER.md:<line>, or
// BASELINE.json:north_star for the spec-defined counter hash, or a DESIGN.md
// "reading" Rk where the sources are silent).
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
//   splitmix64 ........ published test vector; survey-time Python-integer values
//   hash .............. tests/golden/hash_pins.txt, block-range invariant, Eq.(3) birthday law
//   rn16 / add16 ...... exhaustive vs x86 F16C + numpy.float16, PAPER.md:257 example, Cor.3 edge cases
//   F64 mode .......... dense materialised S*A (brute force), E||SA||^2=||A||^2 over 1000 seeds
//   SEQ16 mode ........ integer-valued input == F64 bit-exact; serial bound PAPER.md:261
//   BQ / BC modes ..... Proposition 1 (Eq. 8, 9)
//   SR ................ unbiasedness over all 2^24 draws; Cor. 3 Eq. (12) variance
//   bf16 rn / add ..... exhaustive (all 2^32 floats) vs the integer add-and-truncate rule, torch.bfloat16,
//                       worked example at u = 2^-8, serial bound; SEQ-BF16: integer-valued input == F64
//   xorshift64 ........ Marsaglia's published vector (tests/golden/xorshift64_vector.txt)
//   dither ............ c = 0 and u0 = 1/2 reduce to RN16; oddness; monotone in u0; closed-form
//                       jump probabilities over all 2^24 draws (Eq. 6)
// "parity unpinned" (bit-wise) for SEQ16 on generic inputs: the GPU order is
// arbitrary, so SEQ16 is one legal result, compared statistically.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -shared -fPIC -pthread  (oracle/__init__.py)

#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

namespace {

// ---------------------------------------------------------------------------
// splitmix64, first output of the generator started at state x (reading R1).
// BASELINE.json:north_star "h = splitmix64(seed ^ (i*zeta+j))".
// ---------------------------------------------------------------------------
inline uint64_t splitmix64(uint64_t x) {
  uint64_t z = x + 0x9E3779B97F4A7C15ULL;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
  return z ^ (z >> 31);
}

// (bucket, signbit) of input row i, stack block j.  PAPER.md:59 (uniform target
// in a block of d/zeta rows, equiprobable sign), instantiated by
// BASELINE.json:north_star: bucket = j*db + (((h>>32)*db)>>32), sign = h&1
// (readings R2, R3, R4: precedence, raw bit, 0-based).
inline void hash_ij(uint64_t seed, int64_t i, int32_t j, int32_t zeta, int32_t db,
                    int32_t* bucket, uint32_t* signbit) {
  uint64_t ctr = (uint64_t)i * (uint64_t)zeta + (uint64_t)j;
  uint64_t h = splitmix64(seed ^ ctr);
  uint64_t hi = h >> 32;
  *bucket = j * db + (int32_t)((hi * (uint64_t)(uint32_t)db) >> 32);
  *signbit = (uint32_t)(h & 1ULL);
}

// ---------------------------------------------------------------------------
// IEEE binary16 helpers, written from the format definition (no F16C, no
// compiler half type).  PAPER.md:144 (__float2half = round-to-nearest-even),
// PAPER.md:185-187 (.noftz: subnormals kept), reading R9 (overflow -> +-inf).
// ---------------------------------------------------------------------------
inline double half_to_double(uint16_t hbits) {
  uint32_t sign = hbits >> 15;
  uint32_t e = (hbits >> 10) & 0x1F;
  uint32_t f = hbits & 0x3FF;
  double v;
  if (e == 0) {
    v = std::ldexp((double)f, -24);            // subnormal: f * 2^-24
  } else if (e == 31) {
    v = f ? std::nan("") : INFINITY;
  } else {
    v = std::ldexp((double)(1024 + f), (int)e - 25);  // (1+f/1024)*2^(e-15)
  }
  return sign ? -v : v;
}

// Round a finite-or-not double to binary16, round-to-nearest ties-to-even,
// gradual underflow, |x| >= 65520 -> inf.  One rounding, done on the exact value.
inline uint16_t double_to_half_rn(double x) {
  uint16_t sign = std::signbit(x) ? 0x8000 : 0;
  if (std::isnan(x)) return (uint16_t)(sign | 0x7E00);
  double a = std::fabs(x);
  if (std::isinf(a)) return (uint16_t)(sign | 0x7C00);
  if (a == 0.0) return sign;
  int ex;
  (void)std::frexp(a, &ex);  // a = fr * 2^ex, fr in [0.5,1)  => a in [2^(ex-1), 2^ex)
  int e = ex - 1;            // unbiased exponent of a
  // quantum (spacing of the half grid around a): 2^(e-10) for normal, 2^-24 below 2^-14
  int qexp = (e < -14) ? -24 : (e - 10);
  double scaled = std::ldexp(a, -qexp);  // exact (power-of-two scale), < 2048
  double fl = std::floor(scaled);
  double rem = scaled - fl;              // exact
  uint64_t n = (uint64_t)fl;
  if (rem > 0.5 || (rem == 0.5 && (n & 1ULL))) n += 1;
  // n is the integer count of quanta; rebuild the bit pattern by arithmetic.
  // value = n * 2^qexp.  For subnormal grid (qexp=-24): bits = n (n<=1024 ok: 1024 -> exp field 1).
  uint32_t bits;
  if (qexp == -24) {
    bits = (uint32_t)n;  // n in [0,1024]; 1024 == smallest normal 0x0400
  } else {
    // n in [1024, 2048]; 2048 means carry to next binade.
    int be = e + 15;  // biased exponent
    if (n == 2048) { n = 1024; be += 1; }
    if (be >= 31) return (uint16_t)(sign | 0x7C00);
    bits = ((uint32_t)be << 10) | (uint32_t)(n - 1024);
  }
  return (uint16_t)(sign | bits);
}

// RN16 of an FP32 value (PAPER.md:127-129 `__float2half(s*a)`).
inline uint16_t float_to_half_rn(float p) { return double_to_half_rn((double)p); }

// z <- RN16(z + v): the exact sum of two binary16 values fits a double
// (span 2^-24..2^16 plus 11 bits < 53), rounded once.
// "z_k = RN16(z_{k-1} + v_k)".
inline uint16_t half_add_rn(uint16_t z, uint16_t v) {
  return double_to_half_rn(half_to_double(z) + half_to_double(v));
}

// Stochastic conversion of an FP32 product to binary16,
// reading R13: l = neighbour toward zero, v = neighbour away from zero,
// w = |v|-|l| (the grid spacing at |p|; 2^-24 in the subnormal range),
// t = (|p|-|l|)/w, u = (R24 + 1/2) * 2^-24, return v iff u < t.
// |p| >= 65536 -> inf; 65504 < |p| < 65536 may round up to inf.
inline uint16_t float_to_half_sr(float p, uint32_t r24) {
  uint16_t sign = std::signbit(p) ? 0x8000 : 0;
  if (std::isnan(p)) return (uint16_t)(sign | 0x7E00);
  double a = std::fabs((double)p);
  if (a >= 65536.0) return (uint16_t)(sign | 0x7C00);
  if (a == 0.0) return sign;
  int ex;
  (void)std::frexp(a, &ex);
  int e = ex - 1;
  int qexp = (e < -14) ? -24 : (e - 10);
  double scaled = std::ldexp(a, -qexp);  // exact
  double fl = std::floor(scaled);
  double t = scaled - fl;                // exact, in [0,1)
  uint64_t n = (uint64_t)fl;             // |l| in quanta
  if (t != 0.0) {
    double u = ((double)(r24 & 0xFFFFFFu) + 0.5) * std::ldexp(1.0, -24);
    if (u < t) n += 1;
  }
  uint32_t bits;
  if (qexp == -24) {
    bits = (uint32_t)n;
  } else {
    int be = e + 15;
    if (n == 2048) { n = 1024; be += 1; }
    if (be >= 31) return (uint16_t)(sign | 0x7C00);
    bits = ((uint32_t)be << 10) | (uint32_t)(n - 1024);
  }
  return (uint16_t)(sign | bits);
}


// ---------------------------------------------------------------------------
// bfloat16 control (PAPER.md:382 Fig. 7 "BF16 is a wider-range reference", :396 "BF16 remains
// finite throughout ... residual is about 20% larger").  Format: 1 sign, 8 exponent (bias 127,
// the FP32 range), 7 fraction bits; u = 2^-8; subnormal spacing 2^-133.  Written from the
// format definition like the binary16 routines above; subnormals kept, overflow -> +-inf.
// ---------------------------------------------------------------------------
inline double bf16_to_double(uint16_t b) {
  uint32_t sign = b >> 15;
  uint32_t e = (b >> 7) & 0xFF;
  uint32_t f = b & 0x7F;
  double v;
  if (e == 0) {
    v = std::ldexp((double)f, -133);                  // subnormal: f * 2^-133
  } else if (e == 255) {
    v = f ? std::nan("") : INFINITY;
  } else {
    v = std::ldexp((double)(128 + f), (int)e - 134);  // (1+f/128)*2^(e-127)
  }
  return sign ? -v : v;
}

// Round a double to bfloat16: nearest, ties to even, gradual underflow, one rounding on the
// exact value; |x| >= 2^128 (1 - 2^-9) -> inf.
inline uint16_t double_to_bf16_rn(double x) {
  uint16_t sign = std::signbit(x) ? 0x8000 : 0;
  if (std::isnan(x)) return (uint16_t)(sign | 0x7FC0);
  double a = std::fabs(x);
  if (std::isinf(a)) return (uint16_t)(sign | 0x7F80);
  if (a == 0.0) return sign;
  int ex;
  (void)std::frexp(a, &ex);
  int e = ex - 1;                                    // a in [2^e, 2^(e+1))
  int qexp = (e < -126) ? -133 : (e - 7);            // spacing of the bf16 grid around a
  double scaled = std::ldexp(a, -qexp);              // exact, < 256
  double fl = std::floor(scaled);
  double rem = scaled - fl;
  uint64_t n = (uint64_t)fl;
  if (rem > 0.5 || (rem == 0.5 && (n & 1ULL))) n += 1;
  uint32_t bits;
  if (qexp == -133) {
    bits = (uint32_t)n;                              // n in [0,128]; 128 == smallest normal 0x0080
  } else {
    int be = e + 127;
    if (n == 256) { n = 128; be += 1; }
    if (be >= 255) return (uint16_t)(sign | 0x7F80);
    bits = ((uint32_t)be << 7) | (uint32_t)(n - 128);
  }
  return (uint16_t)(sign | bits);
}

inline uint16_t float_to_bf16_rn(float p) { return double_to_bf16_rn((double)p); }

// z <- RN_bf16(z + v).  The sum is formed in double and rounded once to bf16.  When the exponents
// are at most 44 apart the double sum is exact (8 + 44 + 1 <= 53 bits).  Otherwise |v| < 2^-43 |z|,
// the exact sum lies strictly inside the rounding interval of z (half a bf16 spacing is >= 2^-10 |z|
// away), and so does its double rounding: both round to z.  Either way this is the correctly
// rounded bf16 sum (PAPER.md:253's recursion with u = 2^-8).
inline uint16_t bf16_add_rn(uint16_t z, uint16_t v) {
  return double_to_bf16_rn(bf16_to_double(z) + bf16_to_double(v));
}

// One FP32 multiply, single rounding (PAPER.md:127 `s * a0`).  volatile keeps
// the compiler from contracting or widening it.
inline float mul_f32(float s, float a) {
  volatile float r = s * a;
  return r;
}
// One FP32 add, single rounding.
inline float add_f32(float a, float b) {
  volatile float r = a + b;
  return r;
}

// ---------------------------------------------------------------------------
// Dither conversion, Eq. (6):  Q_dith(q) = RN16(q + (u0 - 1/2) c q),
// "a 24-bit variate u0 in [0,1) from an xorshift generator and the FP32 coefficient c written as
// 0.00097656f ...; the perturbation is evaluated in FP32".  Reading R20: every
// operation is one FP32 operation rounded to nearest, in the order the formula is written, no
// fused multiply-add:  t = u0 - 1/2 (exact: a 24-bit integer times 2^-24),  w = fl(t * c),
// e = fl(w * q),  q' = fl(q + e),  result RN16(q').
// ---------------------------------------------------------------------------
inline uint16_t float_to_half_dither(float q, uint32_t r24, float c) {
  float u0 = (float)(r24 & 0xFFFFFFu) * 5.9604644775390625e-08f;  // r24 * 2^-24, exact
  float t = u0 - 0.5f;                                            // exact
  float w = mul_f32(t, c);
  float e = mul_f32(w, q);
  float qp = add_f32(q, e);
  return float_to_half_rn(qp);
}

// One step of Marsaglia's xorshift64 generator (shifts 13, 7, 17; "Xorshift RNGs", 2003).
inline uint64_t xorshift64(uint64_t x) {
  x ^= x << 13;
  x ^= x >> 7;
  x ^= x << 17;
  return x;
}
// The 64 dither bits of one column pair, reading R21: a xorshift64 generator seeded per
// contribution pair from the counter hash (state 0, which xorshift cannot leave, is replaced by
// the SplitMix64 increment), first output.  Bits 63..40 -> column 2*pair, bits 39..16 -> 2*pair+1
// (the layout of reading R14).
inline uint64_t dither_bits(uint64_t sr_seed, uint64_t ctr) {
  uint64_t x = splitmix64(sr_seed ^ ctr);
  if (x == 0) x = 0x9E3779B97F4A7C15ULL;
  return xorshift64(x);
}
constexpr float kDitherC = 0.00097656f;  // PAPER.md:201, "approximately 2^-10"

// s = fp32(1/sqrt(zeta)), correctly rounded from FP64 (reading R5; PAPER.md:161
// "signed FP32 scale eps/sqrt(zeta)").
inline float scale_f32(int32_t zeta) { return (float)(1.0 / std::sqrt((double)zeta)); }


}  // namespace

extern "C" {

// --- scalar building blocks, exported so the pins can hit them directly -----
uint64_t orc_splitmix64(uint64_t x) { return splitmix64(x); }
uint16_t orc_rn16(float p) { return float_to_half_rn(p); }
uint16_t orc_rn16_from_double(double x) { return double_to_half_rn(x); }
double orc_half_to_double(uint16_t h) { return half_to_double(h); }
uint16_t orc_add16(uint16_t z, uint16_t v) { return half_add_rn(z, v); }
uint16_t orc_sr16(float p, uint32_t r24) { return float_to_half_sr(p, r24); }
float orc_scale_f32(int32_t zeta) { return scale_f32(zeta); }

uint16_t orc_bf16_rn(float p) { return float_to_bf16_rn(p); }
double orc_bf16_to_double(uint16_t b) { return bf16_to_double(b); }
uint16_t orc_bf16_add(uint16_t z, uint16_t v) { return bf16_add_rn(z, v); }
uint64_t orc_xorshift64(uint64_t x) { return xorshift64(x); }
float orc_dither_c(void) { return kDitherC; }
void orc_bf16_rn_array(const float* p, int64_t count, uint16_t* out) {
  for (int64_t k = 0; k < count; ++k) out[k] = float_to_bf16_rn(p[k]);
}
void orc_bf16_add_array(const uint16_t* z, const uint16_t* v, int64_t count, uint16_t* out) {
  for (int64_t k = 0; k < count; ++k) out[k] = bf16_add_rn(z[k], v[k]);
}
void orc_bf16_to_double_array(const uint16_t* b, int64_t count, double* out) {
  for (int64_t k = 0; k < count; ++k) out[k] = bf16_to_double(b[k]);
}
// Eq. (6) with an explicit coefficient, so the pins can set c = 0
void orc_dither16_array(const float* p, const uint32_t* r24, float c, int64_t count, uint16_t* out) {
  for (int64_t k = 0; k < count; ++k) out[k] = float_to_half_dither(p[k], r24[k], c);
}

void orc_rn16_array(const float* p, int64_t count, uint16_t* out) {
  for (int64_t k = 0; k < count; ++k) out[k] = float_to_half_rn(p[k]);
}
void orc_add16_array(const uint16_t* z, const uint16_t* v, int64_t count, uint16_t* out) {
  for (int64_t k = 0; k < count; ++k) out[k] = half_add_rn(z[k], v[k]);
}
void orc_sr16_array(const float* p, const uint32_t* r24, int64_t count, uint16_t* out) {
  for (int64_t k = 0; k < count; ++k) out[k] = float_to_half_sr(p[k], r24[k]);
}

// --- hash stage ---------------------------------------------
// bucket[(i-row_begin)*zeta + j], signbit[...] for i in [row_begin,row_begin+rows).
int orc_hash(uint64_t seed, int32_t d, int32_t zeta, int64_t row_begin, int64_t rows,
             int32_t* bucket, uint8_t* signbit) {
  if (d <= 0 || zeta < 1 || d % zeta != 0) return -1;  // PAPER.md:59 "d divisible by zeta"
  int32_t db = d / zeta;
  for (int64_t r = 0; r < rows; ++r) {
    for (int32_t j = 0; j < zeta; ++j) {
      int32_t b;
      uint32_t sb;
      hash_ij(seed, row_begin + r, j, zeta, db, &b, &sb);
      bucket[r * zeta + j] = b;
      signbit[r * zeta + j] = (uint8_t)sb;
    }
  }
  return 0;
}

// --- dense S, Eq. (1): d x m FP64 row-major, entry eps/sqrt(zeta)
int orc_dense_S(uint64_t seed, int64_t m, int32_t d, int32_t zeta, double* S) {
  if (d <= 0 || zeta < 1 || d % zeta != 0) return -1;
  int32_t db = d / zeta;
  for (int64_t k = 0; k < (int64_t)d * m; ++k) S[k] = 0.0;
  double sc = 1.0 / std::sqrt((double)zeta);
  for (int64_t i = 0; i < m; ++i)
    for (int32_t j = 0; j < zeta; ++j) {
      int32_t b;
      uint32_t sb;
      hash_ij(seed, i, j, zeta, db, &b, &sb);
      S[(int64_t)b * m + i] += sb ? -sc : sc;  // reading R3: bit 0 -> +1, bit 1 -> -1
    }
  return 0;
}

// --- FP64 contribution sums --------------------------------------------------
// mode 0 IDEAL: B  = S*A of Eq. (1): sum eps*(double)a, *caller* multiplies by
//               1/sqrt(zeta) once at the end via orc_f64_finalize (reading R7,
//               PAPER.md:217 "ideal sketch").
// mode 1 BQ:    B_q of PAPER.md:217: exact sum of the actual signed FP32 products.
// mode 2 BC:    B_c of PAPER.md:217: exact sum of their individually RN16-converted values.
// Accumulates into B (d x n row-major FP64, caller-zeroed) so rows can be streamed
// in chunks: rows [row_begin, row_begin+rows) of the matrix, A points at row_begin.
static void f64_accumulate_range(uint64_t seed, int32_t d, int32_t zeta, int mode, const float* A,
                                 int64_t row_begin, int64_t rows, int32_t n, int64_t lda, double* B) {
  int32_t db = d / zeta;
  float s = scale_f32(zeta);
  for (int64_t r = 0; r < rows; ++r) {
    const float* arow = A + r * lda;
    for (int32_t j = 0; j < zeta; ++j) {
      int32_t b;
      uint32_t sb;
      hash_ij(seed, row_begin + r, j, zeta, db, &b, &sb);
      double* brow = B + (int64_t)b * n;
      if (mode == 0) {
        double eps = sb ? -1.0 : 1.0;
        for (int32_t c = 0; c < n; ++c) brow[c] += eps * (double)arow[c];
      } else {
        float es = sb ? -s : s;  // reading R6: (eps*s)*a
        for (int32_t c = 0; c < n; ++c) {
          float p = mul_f32(es, arow[c]);
          brow[c] += (mode == 1) ? (double)p : half_to_double(float_to_half_rn(p));
        }
      }
    }
  }
}

int orc_f64_accumulate(uint64_t seed, int32_t d, int32_t zeta, int mode, const float* A,
                       int64_t row_begin, int64_t rows, int32_t n, int64_t lda, double* B,
                       int32_t threads) {
  if (d <= 0 || zeta < 1 || d % zeta != 0 || n <= 0 || lda < n || mode < 0 || mode > 2) return -1;
  if (threads <= 1 || rows < 4 * (int64_t)threads) {
    f64_accumulate_range(seed, d, zeta, mode, A, row_begin, rows, n, lda, B);
    return 0;
  }
  // Row-chunk-private FP64 partial sketches, summed at the end in chunk order
  // (SURVEY 8d "CPU baseline (b)").  FP64 makes the order immaterial (~L*2^-53).
  std::vector<std::vector<double>> part(threads, std::vector<double>((size_t)d * n, 0.0));
  std::vector<std::thread> pool;
  int64_t per = (rows + threads - 1) / threads;
  for (int32_t t = 0; t < threads; ++t) {
    int64_t r0 = t * per, r1 = std::min<int64_t>(rows, r0 + per);
    if (r0 >= r1) break;
    pool.emplace_back([=, &part]() {
      f64_accumulate_range(seed, d, zeta, mode, A + r0 * lda, row_begin + r0, r1 - r0, n, lda,
                           part[t].data());
    });
  }
  for (auto& th : pool) th.join();
  for (int32_t t = 0; t < threads; ++t)
    for (int64_t k = 0; k < (int64_t)d * n; ++k) B[k] += part[t][k];
  return 0;
}

// multiply the IDEAL-mode sums by the FP64 scale 1/sqrt(zeta), once (reading R7)
void orc_f64_finalize(int32_t zeta, int64_t count, double* B) {
  double sc = 1.0 / std::sqrt((double)zeta);
  for (int64_t k = 0; k < count; ++k) B[k] *= sc;
}

// --- SEQ16: one legal FP16 result (Listing 2 + PAPER.md:253) -----
// rows ascending, blocks ascending (reading R8), every column:
//   p = fp32(eps*s * a);  v = RN16(p) [or SR16(p, bits) if rounding==1, or Q_dith(p) of Eq. (6) if
//   rounding==2: same counter, bits through one xorshift64 step, reading R21];  D = RN16(D + v).
// D is d x n row-major binary16 bit patterns, caller-initialised (+0 for a fresh sketch),
// so rows can be streamed in chunks.  SR bits (reading R14):
//   R = splitmix64(sr_seed ^ ((i*zeta+j)*ceil(n/2) + pair)); bits 63..40 -> column 2*pair,
//   bits 39..16 -> column 2*pair+1.
int orc_seq16_accumulate(uint64_t seed, int32_t d, int32_t zeta, const float* A, int64_t row_begin,
                         int64_t rows, int32_t n, int64_t lda, int rounding, uint64_t sr_seed,
                         uint16_t* D) {
  if (d <= 0 || zeta < 1 || d % zeta != 0 || n <= 0 || lda < n) return -1;
  int32_t db = d / zeta;
  float s = scale_f32(zeta);
  uint64_t npairs = (uint64_t)((n + 1) / 2);
  for (int64_t r = 0; r < rows; ++r) {
    const float* arow = A + r * lda;
    int64_t i = row_begin + r;
    for (int32_t j = 0; j < zeta; ++j) {
      int32_t b;
      uint32_t sb;
      hash_ij(seed, i, j, zeta, db, &b, &sb);
      float es = sb ? -s : s;
      uint16_t* drow = D + (int64_t)b * n;
      for (int32_t c = 0; c < n; ++c) {
        float p = mul_f32(es, arow[c]);
        uint16_t v;
        if (rounding == 0) {
          v = float_to_half_rn(p);
        } else if (rounding == 2) {
          uint64_t ctr = ((uint64_t)i * (uint64_t)zeta + (uint64_t)j) * npairs + (uint64_t)(c >> 1);
          uint64_t R = dither_bits(sr_seed, ctr);
          uint32_t r24 = (c & 1) ? (uint32_t)((R >> 16) & 0xFFFFFFu) : (uint32_t)(R >> 40);
          v = float_to_half_dither(p, r24, kDitherC);
        } else {
          uint64_t ctr = ((uint64_t)i * (uint64_t)zeta + (uint64_t)j) * npairs + (uint64_t)(c >> 1);
          uint64_t R = splitmix64(sr_seed ^ ctr);
          uint32_t r24 = (c & 1) ? (uint32_t)((R >> 16) & 0xFFFFFFu) : (uint32_t)(R >> 40);
          v = float_to_half_sr(p, r24);
        }
        drow[c] = half_add_rn(drow[c], v);
      }
    }
  }
  return 0;
}

// --- SEQ-BF16: the same sequential loop with bfloat16 conversion and accumulation (the BF16
// control of PAPER.md:382, :396): p = fp32(eps*s*a); v = RN_bf16(p); D = RN_bf16(D + v).
// D is d x n row-major bfloat16 bit patterns, caller-initialised.
int orc_seqbf16_accumulate(uint64_t seed, int32_t d, int32_t zeta, const float* A, int64_t row_begin,
                           int64_t rows, int32_t n, int64_t lda, uint16_t* D) {
  if (d <= 0 || zeta < 1 || d % zeta != 0 || n <= 0 || lda < n) return -1;
  int32_t db = d / zeta;
  float s = scale_f32(zeta);
  for (int64_t r = 0; r < rows; ++r) {
    const float* arow = A + r * lda;
    for (int32_t j = 0; j < zeta; ++j) {
      int32_t b;
      uint32_t sb;
      hash_ij(seed, row_begin + r, j, zeta, db, &b, &sb);
      float es = sb ? -s : s;
      uint16_t* drow = D + (int64_t)b * n;
      for (int32_t c = 0; c < n; ++c) drow[c] = bf16_add_rn(drow[c], float_to_bf16_rn(mul_f32(es, arow[c])));
    }
  }
  return 0;
}

// --- SEQ32: the same loop with an FP32 running sum (Listing 1's
// atomicAdd(&B[r*n+col], val*a) in ascending order); one legal FP32 result.
int orc_seq32_accumulate(uint64_t seed, int32_t d, int32_t zeta, const float* A, int64_t row_begin,
                         int64_t rows, int32_t n, int64_t lda, float* B) {
  if (d <= 0 || zeta < 1 || d % zeta != 0 || n <= 0 || lda < n) return -1;
  int32_t db = d / zeta;
  float s = scale_f32(zeta);
  for (int64_t r = 0; r < rows; ++r) {
    const float* arow = A + r * lda;
    for (int32_t j = 0; j < zeta; ++j) {
      int32_t b;
      uint32_t sb;
      hash_ij(seed, row_begin + r, j, zeta, db, &b, &sb);
      float es = sb ? -s : s;
      float* brow = B + (int64_t)b * n;
      for (int32_t c = 0; c < n; ++c) {
        float p = mul_f32(es, arow[c]);
        volatile float z = brow[c] + p;
        brow[c] = z;
      }
    }
  }
  return 0;
}

// --- range counters for the rescaling study (reading R18; Eq. 9 N_sub, Cor. 3) -----
// per contribution p = fp32(eps*s*a): counts[0] += 0<|p|<2^-14 (N_sub),
// counts[1] += p!=0 && RN16(p)==0 (erased), counts[2] += |p|>=65520 (RN -> inf),
// counts[3] += number of contributions examined.
int orc_range_counts(int32_t zeta, const float* A, int64_t rows, int32_t n, int64_t lda,
                     int64_t* counts) {
  if (zeta < 1 || n <= 0 || lda < n) return -1;
  float s = scale_f32(zeta);
  for (int64_t r = 0; r < rows; ++r)
    for (int32_t c = 0; c < n; ++c) {
      float p = mul_f32(s, A[r * lda + c]);  // RN is odd: sign irrelevant to the class
      double a = std::fabs((double)p);
      int64_t sub = (a > 0.0 && a < std::ldexp(1.0, -14)) ? 1 : 0;
      int64_t zero = (a > 0.0 && (float_to_half_rn(p) & 0x7FFF) == 0) ? 1 : 0;
      int64_t inf = (a >= 65520.0) ? 1 : 0;
      counts[0] += sub * zeta;
      counts[1] += zero * zeta;
      counts[2] += inf * zeta;
      counts[3] += zeta;
    }
  return 0;
}

}  // extern "C"
