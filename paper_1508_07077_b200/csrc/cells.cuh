// cells.cuh -- step a2: cell-list build (K-A).  PAPER.md L180 (checkerboard grid, "grid lines are randomly
// shifted"); BASELINE.json north_star (2).  Deterministic layout: occupants of a cell in ascending particle id,
// cells in ascending linear index (ix fastest), so a row of 3 x-neighbour cells is one contiguous span.
//   k_bin_count   cell id + arrival rank per particle (atomic), counts per cell
//   k_scan_*      exclusive scan of the counts -> cell_start            (3 small kernels)
//   k_fill        scatter particle ids to cell_start[c] + rank
//   k_sort_write  per cell: sort its few ids ascending (removes the atomics' arrival order) and write the
//                 cell-ordered pose copy cpos = (x,y,z,pid) and, for anisotropic shapes, caxis = body z axis
// (measured and dropped in round 2: k_fill scattering the 16-byte pose copy itself and a sort pass over the cells with
//  >= 2 occupants only: 24.3 + 10.4 us against 12.5 + 18.1 us for this split at C3)
#pragma once
#include <cstdint>
#include "geometry.cuh"

namespace hpmc {

__global__ void __launch_bounds__(256) k_bin_count(const float4* __restrict__ pos, int N, Geo g, float sx, float sy,
                                                   float sz, uint32_t* __restrict__ cid, uint32_t* __restrict__ rank,
                                                   uint32_t* __restrict__ counts, uint8_t* __restrict__ outcome) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  outcome[i] = 0;                      // outcome codes of the sweep this build belongs to: "not tried"
  const float4 p = pos[i];
  const int ix = cell_axis(g, p.x, sx), iy = cell_axis(g, p.y, sy), iz = cell_axis(g, p.z, sz);
  const uint32_t c = ((uint32_t)iz * g.nc + iy) * g.nc + ix;
  cid[i] = c;
  rank[i] = atomicAdd(&counts[c], 1u);
}

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* s_warp, uint32_t& block_total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t incl = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  if (lane == 31) s_warp[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    uint32_t w = (lane < (int)(blockDim.x >> 5)) ? s_warp[lane] : 0u;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += t;
    }
    s_warp[lane] = w;   // inclusive over warps
  }
  __syncthreads();
  const uint32_t warp_off = wid ? s_warp[wid - 1] : 0u;
  block_total = s_warp[(blockDim.x >> 5) - 1];
  return warp_off + incl - v;
}

// counts[] is padded to a multiple of SCAN_TILE and 16-byte aligned (cudaMalloc), so every thread moves its 8
// consecutive words as two uint4: fully coalesced 16-byte accesses.
__device__ __forceinline__ void load8(const uint32_t* __restrict__ p, uint32_t v[8]) {
  const uint4 a = reinterpret_cast<const uint4*>(p)[0], b = reinterpret_cast<const uint4*>(p)[1];
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w; v[4] = b.x; v[5] = b.y; v[6] = b.z; v[7] = b.w;
}

__global__ void __launch_bounds__(SCAN_THREADS) k_scan_tiles(const uint32_t* __restrict__ counts, int n,
                                                             uint32_t* __restrict__ tile_sums) {
  __shared__ uint32_t s_warp[32];
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS], s = 0;
  load8(counts + base, v);                       // the padding beyond n is kept zero
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) s += v[k];
  uint32_t total;
  block_exclusive_scan(s, s_warp, total);
  if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) k_scan_top(uint32_t* __restrict__ tile_sums, int ntiles) {
  __shared__ uint32_t s_warp[32];
  uint32_t carry = 0;
  for (int base = 0; base < ntiles; base += 1024) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < ntiles ? tile_sums[i] : 0u;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan(v, s_warp, total);
    if (i < ntiles) tile_sums[i] = carry + ex;
    carry += total;
    __syncthreads();
  }
}

// FUSED_TOP: tile_sums holds the raw tile totals and every CTA adds up the totals of the tiles before it (a few
// hundred words from L2: cheaper than a launch of k_scan_top); otherwise tile_sums is already the exclusive scan.
// The counts are consumed here for the last time and re-zeroed for the next build.
template <bool FUSED_TOP>
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_apply(uint32_t* __restrict__ counts, int n,
                                                             const uint32_t* __restrict__ tile_sums,
                                                             uint32_t* __restrict__ cell_start) {
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_off;
  uint32_t off;
  if (FUSED_TOP) {
    uint32_t part = 0;
    for (int i = threadIdx.x; i < (int)blockIdx.x; i += SCAN_THREADS) part += tile_sums[i];
    uint32_t tot;
    block_exclusive_scan(part, s_warp, tot);
    if (threadIdx.x == 0) s_off = tot;
    __syncthreads();
    off = s_off;
  } else {
    off = tile_sums[blockIdx.x];
  }
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS], s = 0;
  load8(counts + base, v);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) s += v[k];
  reinterpret_cast<uint4*>(counts + base)[0] = make_uint4(0u, 0u, 0u, 0u);     // re-zeroed for the next build
  reinterpret_cast<uint4*>(counts + base)[1] = make_uint4(0u, 0u, 0u, 0u);
  uint32_t total;
  uint32_t run = off + block_exclusive_scan(s, s_warp, total);
  uint32_t o[SCAN_ITEMS];
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) { o[k] = run; run += v[k]; }
  // cell_start is padded like counts (the words beyond n + 1 are scratch), so the store is two uint4 as well
  reinterpret_cast<uint4*>(cell_start + base)[0] = make_uint4(o[0], o[1], o[2], o[3]);
  reinterpret_cast<uint4*>(cell_start + base)[1] = make_uint4(o[4], o[5], o[6], o[7]);
  // cell_start[n] = N: inside the padding it is written above (padding counts are zero); if n is a whole number of tiles
  // the last thread adds it
  if (base + SCAN_ITEMS == n) cell_start[n] = run;
}

__global__ void __launch_bounds__(256) k_fill(const uint32_t* __restrict__ cid, const uint32_t* __restrict__ rank,
                                              const uint32_t* __restrict__ cell_start, int N,
                                              uint32_t* __restrict__ cell_pid) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  cell_pid[cell_start[cid[i]] + rank[i]] = (uint32_t)i;
}

template <int SHAPE>
__global__ void __launch_bounds__(256) k_sort_write(const uint32_t* __restrict__ cell_start, int ncell,
                                                    uint32_t* __restrict__ cell_pid, const float4* __restrict__ pos,
                                                    const float4* __restrict__ quat, float4* __restrict__ cpos,
                                                    float4* __restrict__ caxis) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  const uint32_t b = cell_start[c], e = cell_start[c + 1];
  for (uint32_t s = b + 1; s < e; ++s) {          // insertion sort, a handful of entries at most
    const uint32_t v = cell_pid[s];
    uint32_t t = s;
    while (t > b && cell_pid[t - 1] > v) { cell_pid[t] = cell_pid[t - 1]; --t; }
    cell_pid[t] = v;
  }
  for (uint32_t s = b; s < e; ++s) {
    const uint32_t i = cell_pid[s];
    float4 p = pos[i];
    p.w = __uint_as_float(i);
    cpos[s] = p;
    if (SHAPE != SH_SPHERE) caxis[s] = as_f4(ori_of<SHAPE>(as_q(quat[i])));     // body axis, or the quaternion (tetrahedron)
  }
}

}  // namespace hpmc
