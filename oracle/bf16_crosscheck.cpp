// bf16_crosscheck.cpp -- TEST INFRASTRUCTURE.  A pin for the oracle's bfloat16 conversion, not part
// of its arithmetic: compares orc_bf16_rn (written from the format definition in sketch_oracle.cpp)
// with the textbook integer rule "add 0x7FFF plus the lowest kept bit to the FP32 pattern, keep the
// upper 16 bits" over every FP32 bit pattern, and orc_bf16_add with "add in FP32, round to bf16"
// (innocuous double rounding: 24 >= 2*8 + 2).
#include <atomic>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

extern "C" uint16_t orc_bf16_rn(float p);
extern "C" uint16_t orc_bf16_add(uint16_t z, uint16_t v);

namespace {
inline bool is_nan_bf(uint16_t b) { return (b & 0x7F80) == 0x7F80 && (b & 0x7F) != 0; }
inline bool same_bf(uint16_t a, uint16_t b) { return a == b || (is_nan_bf(a) && is_nan_bf(b)); }
inline uint16_t bits_rn(uint32_t x) {
  if ((x & 0x7FFFFFFFu) > 0x7F800000u) return (uint16_t)((x >> 16) | 0x0040);  // NaN stays NaN
  return (uint16_t)((x + 0x7FFFu + ((x >> 16) & 1u)) >> 16);
}
inline float bf_to_float(uint16_t b) {
  uint32_t x = (uint32_t)b << 16;
  float f;
  std::memcpy(&f, &x, 4);
  return f;
}
}  // namespace

extern "C" {

int64_t orc_x_bf16_vs_bits(uint32_t first, uint64_t count, uint32_t stride, int32_t threads, uint32_t* first_bad) {
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
        if (!same_bf(orc_bf16_rn(x), bits_rn(bits))) {
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

// z over all 2^16 patterns, v over v0, v0 + v_stride, ...
int64_t orc_x_bf16_add_vs_float(uint32_t v0, uint32_t v_stride, int32_t threads, uint32_t* first_bad) {
  std::atomic<int64_t> bad{0};
  std::atomic<uint64_t> badpat{~0ULL};
  if (threads < 1) threads = 1;
  if (v_stride == 0) v_stride = 1;
  std::vector<std::thread> pool;
  for (int32_t t = 0; t < threads; ++t) {
    pool.emplace_back([=, &bad, &badpat]() {
      for (uint32_t z = t; z < 65536u; z += threads)
        for (uint32_t v = v0; v < 65536u; v += v_stride) {
          volatile float sum = bf_to_float((uint16_t)z) + bf_to_float((uint16_t)v);
          float sf = sum;
          uint32_t sb;
          std::memcpy(&sb, &sf, 4);
          uint16_t want = bits_rn(sb);
          uint16_t got = orc_bf16_add((uint16_t)z, (uint16_t)v);
          if (!same_bf(got, want)) {
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
