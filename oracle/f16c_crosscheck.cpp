// f16c_crosscheck.cpp -- TEST INFRASTRUCTURE.  A pin for the oracle's own
// binary16 routines, not part of its arithmetic: compares orc_rn16 / orc_add16
// (written from the format definition in sketch_oracle.cpp) against the x86
// F16C hardware conversion `_cvtss_sh(x, round-to-nearest-even)`, exhaustively.
// Compiled with -mf16c into its own translation unit; tests skip it when the
// host CPU has no F16C.
#include <immintrin.h>

#include <atomic>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

extern "C" uint16_t orc_rn16(float p);
extern "C" uint16_t orc_add16(uint16_t z, uint16_t v);

namespace {
inline bool is_nan16(uint16_t h) { return (h & 0x7C00) == 0x7C00 && (h & 0x3FF) != 0; }
inline bool same16(uint16_t a, uint16_t b) { return a == b || (is_nan16(a) && is_nan16(b)); }
inline uint16_t hw_rn16(float x) {
  return (uint16_t)_cvtss_sh(x, _MM_FROUND_TO_NEAREST_INT | _MM_FROUND_NO_EXC);
}
inline float hw_h2f(uint16_t h) { return _cvtsh_ss(h); }
}  // namespace

extern "C" {

// Every FP32 bit pattern first, first+stride, ... (count of them); returns the
// number of mismatches and the first offending pattern.
int64_t orc_x_rn16_vs_f16c(uint32_t first, uint64_t count, uint32_t stride, int32_t threads,
                           uint32_t* first_bad) {
  std::atomic<int64_t> bad{0};
  std::atomic<uint64_t> badpat{~0ULL};
  if (threads < 1) threads = 1;
  std::vector<std::thread> pool;
  uint64_t per = (count + threads - 1) / threads;
  for (int32_t t = 0; t < threads; ++t) {
    uint64_t k0 = t * per, k1 = k0 + per < count ? k0 + per : count;
    if (k0 >= k1) break;
    pool.emplace_back([=, &bad, &badpat]() {
      for (uint64_t k = k0; k < k1; ++k) {
        uint32_t bits = first + (uint32_t)(k * stride);
        float x;
        std::memcpy(&x, &bits, 4);
        if (!same16(orc_rn16(x), hw_rn16(x))) {
          bad.fetch_add(1);
          uint64_t cur = badpat.load();
          while (bits < cur && !badpat.compare_exchange_weak(cur, bits)) {
          }
        }
      }
    });
  }
  for (auto& th : pool) th.join();
  if (first_bad) *first_bad = (uint32_t)badpat.load();
  return bad.load();
}

// z over all 2^16 patterns, v over patterns v0, v0+v_stride, ...: float add of
// two halves is exact-or-correctly-rounded-once after F16C rounding (24 >= 2*11+2).
int64_t orc_x_add16_vs_f16c(uint32_t v0, uint32_t v_stride, int32_t threads, uint32_t* first_bad) {
  std::atomic<int64_t> bad{0};
  std::atomic<uint64_t> badpat{~0ULL};
  if (threads < 1) threads = 1;
  if (v_stride == 0) v_stride = 1;
  std::vector<std::thread> pool;
  for (int32_t t = 0; t < threads; ++t) {
    pool.emplace_back([=, &bad, &badpat]() {
      for (uint32_t z = t; z < 65536u; z += threads)
        for (uint32_t v = v0; v < 65536u; v += v_stride) {
          uint16_t want = hw_rn16(hw_h2f((uint16_t)z) + hw_h2f((uint16_t)v));
          uint16_t got = orc_add16((uint16_t)z, (uint16_t)v);
          if (!same16(got, want)) {
            bad.fetch_add(1);
            uint64_t pat = ((uint64_t)z << 16) | v, cur = badpat.load();
            while (pat < cur && !badpat.compare_exchange_weak(cur, pat)) {
            }
          }
        }
    });
  }
  for (auto& th : pool) th.join();
  if (first_bad) *first_bad = (uint32_t)badpat.load();
  return bad.load();
}

}  // extern "C"
