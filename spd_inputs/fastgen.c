/* fastgen.c — seeded N(0, std) bf16 matrix filler for the synthetic weights (inputs only; none of
 * the SPD arithmetic).  Counter-based: element pair j of a tensor keyed `key` is a Box-Muller
 * transform of two 24-bit uniforms hashed from (key, j), so any slice can be generated in parallel
 * and the bytes depend only on (key, index), never on the thread count. */
#include <math.h>
#include <stdint.h>
#include <string.h>

static inline uint64_t mix64(uint64_t x) {
  x += 0x9e3779b97f4a7c15ull;
  x = (x ^ (x >> 30)) * 0xbf58476d1ce4e5b9ull;
  x = (x ^ (x >> 27)) * 0x94d049bb133111ebull;
  return x ^ (x >> 31);
}

static inline uint16_t to_bf16(float x) {
  uint32_t u;
  memcpy(&u, &x, 4);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

void fastgen_normal_bf16(uint16_t *out, uint64_t n, uint64_t key, float std) {
  const float two_pi = 6.28318530717958647692f;
  uint64_t pairs = (n + 1) / 2;
#pragma omp parallel for schedule(static)
  for (uint64_t j = 0; j < pairs; ++j) {
    uint64_t h = mix64(key ^ mix64(j));
    float u1 = ((float)(uint32_t)(h >> 40) + 0.5f) * (1.0f / 16777216.0f);
    float u2 = ((float)(uint32_t)((h >> 16) & 0xffffffu) + 0.5f) * (1.0f / 16777216.0f);
    float r = sqrtf(-2.0f * logf(u1)) * std;
    float a = two_pi * u2;
    out[2 * j] = to_bf16(r * cosf(a));
    if (2 * j + 1 < n) out[2 * j + 1] = to_bf16(r * sinf(a));
  }
}
