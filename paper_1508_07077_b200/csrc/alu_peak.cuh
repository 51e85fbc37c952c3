// alu_peak.cuh -- micro-benchmark of the plain ALU pipes (SURVEY 8(d) "Peaks to use").
//
// The move kernel is bound by integer (Philox) and non-FMA fp32 instruction issue, and MEASURED_PEAKS.json holds
// no ALU figure, so the roofline denominator is measured on the device the library runs on: dependency-free
// streams of ONE instruction kind (8 independent chains per thread, 32 warps per SM) timed with clock64(), giving
// thread-instructions per SM per clock, which is clock-independent.  Kinds: FADD, FMUL, FFMA (context only: the
// path runs with --fmad=false), IMAD, the pair IMAD.WIDE.U32 + LOP3 (one half of a Philox round: wide multiply, then
// hi ^ lo ^ key; counted as 2 instructions), LOP3 alone, an alternating FADD/LOP3 stream (both pipes at once: the issue limit), and the Philox4x32-10
// block function itself with 1, 2 and 4 independent blocks per thread.
#pragma once
#include <cstdint>
#include "philox.cuh"

namespace hpmc {

enum : int { AK_FADD = 0, AK_FMUL, AK_FFMA, AK_IMAD, AK_IMADW_XOR, AK_LOP3, AK_MIX, AK_PHILOX1, AK_PHILOX2, AK_PHILOX4, AK_COUNT };

constexpr int AK_THREADS = 512;     // x 2 CTAs per SM = 32 warps per SM
constexpr int AK_CHAINS = 8;

template <int KIND>
__global__ void __launch_bounds__(AK_THREADS) k_alu_peak(int iters, uint32_t a, uint32_t b, float fa, float fb, Key10 key,
                                                         unsigned long long* __restrict__ cycles,
                                                         uint32_t* __restrict__ sink) {
  uint32_t x[AK_CHAINS];
  float f[AK_CHAINS];
#pragma unroll
  for (int c = 0; c < AK_CHAINS; ++c) {
    x[c] = threadIdx.x * 2654435761u + (uint32_t)c * 40503u + a;
    f[c] = (float)(threadIdx.x + c) * fa;
  }
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
#pragma unroll
      for (int c = 0; c < AK_CHAINS; ++c) {
        if (KIND == AK_FADD) f[c] = f[c] + fb;
        if (KIND == AK_FMUL) f[c] = f[c] * fb;
        if (KIND == AK_FFMA) f[c] = fmaf(f[c], fb, fa);
        if (KIND == AK_IMAD) asm("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x[c]) : "r"(a), "r"(b));   // opaque to the compiler: x a^4 + k cannot be folded
        if (KIND == AK_IMADW_XOR) {               // one Philox half-round: wide multiply, then hi ^ lo ^ key (2 instructions)
          const unsigned long long w = (unsigned long long)x[c] * 0xD2511F53u;
          x[c] = (uint32_t)(w >> 32) ^ (uint32_t)w ^ b;
        }
        if (KIND == AK_LOP3) asm("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[c]) : "r"(a), "r"(b));
        if (KIND == AK_MIX) {
          if (c & 1) f[c] = f[c] + fb;
          else asm("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[c]) : "r"(a), "r"(b));
        }
      }
    }
    if (KIND == AK_PHILOX1 || KIND == AK_PHILOX2 || KIND == AK_PHILOX4) {
      constexpr int NB = KIND == AK_PHILOX1 ? 1 : (KIND == AK_PHILOX2 ? 2 : 4);
#pragma unroll
      for (int c = 0; c < NB; ++c) {
        const Block4 r = philox(key, x[c], (uint32_t)it, x[c + 4], b);
        x[c] = r.x ^ r.z; x[c + 4] = r.y ^ r.w;
      }
    }
  }
  const long long t1 = clock64();
  uint32_t acc = 0;
#pragma unroll
  for (int c = 0; c < AK_CHAINS; ++c) acc ^= x[c] ^ __float_as_uint(f[c]);
  if (acc == 0x12345678u) sink[0] = acc;       // keeps every chain alive; practically never taken
  if ((threadIdx.x & 31) == 0) atomicMax(&cycles[blockIdx.x], (unsigned long long)(t1 - t0));   // slowest warp of the CTA
}

}  // namespace hpmc
