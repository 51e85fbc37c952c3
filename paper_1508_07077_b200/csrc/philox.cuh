// philox.cuh -- counter-based RNG of the hot path: Philox4x32-10 (Salmon et al., SC'11) keyed by
// (seed, step) with counter (id, k, trial|dir<<16, purpose|colour<<8|attempt<<16).
// BASELINE.json north_star ("Randomness comes from counter-based Philox4x32-10 keyed by (seed, step,
// sub-lattice, colloid id, trial, depletant index)"); reading R-S20.
#pragma once
#include <cstdint>

namespace hpmc {

enum : uint32_t { P_SWEEP = 0, P_SELECT = 1, P_MOVE = 2, P_NDEP = 3, P_DEPPOS = 4, P_CBPOS = 5, P_ACCEPT = 6, P_FREEVOL = 7 };

struct Key10 {  // the ten round keys of one (seed, step): hoisted out of every block computation
  uint32_t k0[10], k1[10];
};

__host__ __device__ inline Key10 make_key(uint32_t seed, uint32_t step) {
  Key10 k;
  uint32_t a = seed, b = step;
#pragma unroll
  for (int r = 0; r < 10; ++r) { k.k0[r] = a; k.k1[r] = b; a += 0x9E3779B9u; b += 0xBB67AE85u; }
  return k;
}

struct Block4 { uint32_t x, y, z, w; };

__host__ __device__ __forceinline__ uint32_t ctr_word3(uint32_t purpose, uint32_t colour, uint32_t attempt) {
  return purpose + (colour << 8) + (attempt << 16);
}

__host__ __device__ __forceinline__ Block4 philox(const Key10& key, uint32_t c0, uint32_t c1, uint32_t c2,
                                                   uint32_t c3) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
#ifdef __CUDA_ARCH__
    const uint32_t lo0 = 0xD2511F53u * c0, hi0 = __umulhi(0xD2511F53u, c0);
    const uint32_t lo1 = 0xCD9E8D57u * c2, hi1 = __umulhi(0xCD9E8D57u, c2);
#else
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t lo0 = (uint32_t)p0, hi0 = (uint32_t)(p0 >> 32), lo1 = (uint32_t)p1, hi1 = (uint32_t)(p1 >> 32);
#endif
    const uint32_t n0 = hi1 ^ c1 ^ key.k0[r];
    const uint32_t n2 = hi0 ^ c3 ^ key.k1[r];
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
  }
  return Block4{c0, c1, c2, c3};
}

// u32 -> s = 2u-1 with u = ((x>>9)+0.5) 2^-23: every operation exact in binary32 (R-S4)
__host__ __device__ __forceinline__ float sym_unit(uint32_t x) {
  return ((float)(x >> 9) + 0.5f) * 2.384185791015625e-07f - 1.0f;
}
__host__ __device__ __forceinline__ float unit01(uint32_t x) {
  return ((float)(x >> 9) + 0.5f) * 1.1920928955078125e-07f;
}

}  // namespace hpmc
