/* Seeded random sequential placement of N sphere centres in a periodic cube.
 *
 * Input generator only (serves the CUDA library and the CPU oracle alike): it holds none of the
 * method's arithmetic.  RNG: splitmix64.  Candidates are rounded to float32 first (the stored
 * precision) and then tested in double with a relative margin, so the result is overlap-free under
 * any fp32 distance predicate.  Returns the number placed (== N on success).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static uint64_t sm64(uint64_t* s) {
  uint64_t z = (*s += 0x9E3779B97F4A7C15ull);
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

int64_t rsa_place(int64_t N, double L, double sigma, uint64_t seed, float* pos4, int64_t max_tries) {
  int g = (int)floor(L / (sigma * 1.0001));
  if (g < 1) g = 1;
  const double wg = L / g;
  const int K = 8;
  const int64_t ncell = (int64_t)g * g * g;
  int32_t* slots = (int32_t*)malloc(sizeof(int32_t) * ncell * K);
  uint8_t* cnt = (uint8_t*)calloc(ncell, 1);
  if (!slots || !cnt) { free(slots); free(cnt); return -1; }
  const double d2min = sigma * (1.0 + 5e-5) * sigma * (1.0 + 5e-5);
  const float Lf = (float)L;
  uint64_t s = seed;
  int64_t placed = 0, tries = 0;
  const int span = g >= 3 ? 1 : 0;
  while (placed < N && tries < max_tries) {
    ++tries;
    float c[3];
    int ci[3];
    for (int a = 0; a < 3; ++a) {
      c[a] = (float)((double)(sm64(&s) >> 11) * (1.0 / 9007199254740992.0) * L);
      if (c[a] >= Lf || c[a] < 0.0f) c[a] = 0.0f;
      ci[a] = (int)((double)c[a] / wg);
      if (ci[a] >= g) ci[a] = g - 1;
    }
    int ok = 1;
    for (int dz = -span; dz <= span && ok; ++dz)
      for (int dy = -span; dy <= span && ok; ++dy)
        for (int dx = -span; dx <= span && ok; ++dx) {
          int64_t lin;
          if (g >= 3) {
            const int jx = (ci[0] + dx + g) % g, jy = (ci[1] + dy + g) % g, jz = (ci[2] + dz + g) % g;
            lin = ((int64_t)jz * g + jy) * g + jx;
          } else lin = -1;
          const int64_t lo = lin >= 0 ? lin : 0, hi = lin >= 0 ? lin + 1 : ncell;
          for (int64_t cl = lo; cl < hi && ok; ++cl)
            for (int k = 0; k < cnt[cl]; ++k) {
              const float* p = pos4 + 4 * (int64_t)slots[cl * K + k];
              double d2 = 0.0;
              for (int a = 0; a < 3; ++a) {
                double d = (double)p[a] - (double)c[a];
                d -= L * nearbyint(d / L);
                d2 += d * d;
              }
              if (d2 < d2min) { ok = 0; break; }
            }
        }
    if (!ok) continue;
    const int64_t own = ((int64_t)ci[2] * g + ci[1]) * g + ci[0];
    if (cnt[own] >= K) continue;
    slots[own * K + cnt[own]++] = (int32_t)placed;
    pos4[4 * placed] = c[0]; pos4[4 * placed + 1] = c[1]; pos4[4 * placed + 2] = c[2]; pos4[4 * placed + 3] = 0.0f;
    ++placed;
  }
  free(slots); free(cnt);
  return placed;
}
