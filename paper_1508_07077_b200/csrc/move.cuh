// move.cuh -- steps a3..a10: the checkerboard move kernel (K-B).
//
// One warp per non-empty active cell (persistent warps stride over the active cells of the pass):
//   a3  pick one occupant uniformly                                  (north_star)
//   a4  trial translation / Cayley rotation, wrap, confinement       (L66, L78, L180)
//   a5  stage the 27-cell neighbourhood in shared memory in the frame of the new centre
//   a6  hard-overlap test, neighbours across lanes                   (Eq. 5)
//   a7  N_d ~ Poisson(n_R V_ins) by table inversion                  (L67, L156)
//   a8  depletants across lanes, __ballot_sync early exit on the first rejecting one (L68, L72, L156)
//   a9  configurational-bias reinsertions across lanes               (Sec. III.D, Eq. 16)
//   a10 commit pose, outcome code, counters                          (App. A "flagged for rejection")
// The paper's GPU design (App. A: separate trial-move, insertion and CB kernels with global round trips) is
// fused into this single kernel.
#pragma once
#include <cstdint>
#include "geometry.cuh"
#include "philox.cuh"

namespace hpmc {

enum : int { C_TRIALS_TRANS, C_ACCEPT_TRANS, C_TRIALS_ROT, C_ACCEPT_ROT, C_REJ_BOUNDARY, C_REJ_HARD,
             C_REJ_DEPLETANT, C_REJ_CB, C_DEP_DRAWN, C_DEP_NEEDED, C_DEP_EVALUATED, C_CB_REINSERTIONS,
             C_PHILOX_BLOCKS, C_COUNT };
enum : int { OUT_NONE = 0, OUT_ACCEPT = 1, OUT_BOUNDARY = 2, OUT_HARD = 3, OUT_DEPLETANT = 4, OUT_CB = 5 };

constexpr int MOVE_WARPS = 8;          // warps per CTA
constexpr int MAXNB = 64;              // staged neighbours per move

struct MoveArgs {
  Geo g;
  Key10 key;
  float sx, sy, sz;                    // grid shift of this sweep
  uint32_t colour;                     // active sub-lattice (bit0: x parity, bit1: y, bit2: z)
  int hc;                              // n_c / 2
  int nact;                            // hc^3 active cells
  float d_max, a_max, a_max2;
  int n_trial;
  float4* pos;                         // [N] canonical poses (updated on accept)
  float4* quat;
  float4* cpos;                        // [N] cell-ordered (x,y,z,pid)
  float4* caxis;                       // [N] cell-ordered body axes (anisotropic shapes)
  const uint32_t* cell_start;
  const unsigned long long* ptable;    // Poisson thresholds
  int pt_n;
  uint32_t pt_klo;
  uint8_t* outcome;
  unsigned long long* counters;
  int* err_flag;
  uint32_t* acc_count;                 // host-buffer path: list of the particles accepted this sweep (nullptr: not kept)
  uint32_t* acc_list;
  uint32_t options;                    // OPT_SHELL | OPT_ROSENBLUTH (hpmc_set_options)
  float sh_Rin3, sh_dR3;               // shell option (R-N1): R_in^3 and R^3 - R_in^3
};

enum : uint32_t { OPT_SHELL = 1u, OPT_ROSENBLUTH = 2u };

// cube root by +, x, / only (R-N1: no libdevice transcendental on the parity path): exponent/3 seed, four Newton steps
__device__ __forceinline__ float cbrt_fixed(float t) {
  float y = __uint_as_float(__float_as_uint(t) / 3u + 0x2a514067u);
#pragma unroll
  for (int it = 0; it < 4; ++it) { const float q = __fdiv_rn(t, y * y); y = ((y + y) + q) * 0.33333334f; }
  return y;
}

// One attempt of the shell sampler (R-N1) from one Philox block: direction by cube rejection (words 0-2), radius
// (R_in^3 + u dR^3)^(1/3) from word 3.  Returns false if the attempt is rejected.
__device__ __forceinline__ bool shell_attempt(const Block4& r, float Rin3, float dR3, V3& d) {
  const V3 v = V3{sym_unit(r.x), sym_unit(r.y), sym_unit(r.z)};
  const float n2 = dot3(v, v);
  if (!(n2 <= 1.0f && n2 >= 1e-6f)) return false;
  const float t = Rin3 + unit01(r.w) * dR3;
  d = v * __fdiv_rn(cbrt_fixed(t), __fsqrt_rn(n2));
  return true;
}


// uniform point in the ball (R-S3): cube rejection, one Philox block per attempt, cap 64 then the origin
__device__ __forceinline__ V3 ball_sample(const Key10& key, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3base,
                                          float radius, float radius2, uint32_t& nblocks) {
  for (uint32_t a = 0; a < 64; ++a) {
    const Block4 r = philox(key, c0, c1, c2, c3base + (a << 16));
    ++nblocks;
    const V3 d = V3{radius * sym_unit(r.x), radius * sym_unit(r.y), radius * sym_unit(r.z)};
    if (dot3(d, d) <= radius2) return d;
  }
  return V3{0.0f, 0.0f, 0.0f};
}

// position of depletant k about the new centre: the whole insertion ball (L156) or, with OPT_SHELL, its shell (L158)
__device__ __forceinline__ V3 dep_position(const MoveArgs& A, uint32_t pid, uint32_t k, uint32_t c3dep, uint32_t& nblocks) {
  if (!(A.options & OPT_SHELL)) return ball_sample(A.key, pid, k, 0, c3dep, A.g.Rins, A.g.Rins2, nblocks);
  for (uint32_t a = 0; a < 64; ++a) {
    const Block4 r = philox(A.key, pid, k, 0, c3dep + (a << 16));
    ++nblocks;
    V3 d;
    if (shell_attempt(r, A.sh_Rin3, A.sh_dR3, d)) return d;
  }
  return V3{A.g.Rins, 0.0f, 0.0f};
}

template <int SHAPE>
struct MoveCtx {       // per-move state shared by the depletant predicates
  V3 rho_old;
  Ori a_old, a_new;
  const float4* nb;    // shared memory: neighbour centres relative to the new centre
  const float4* ax;    // shared memory: neighbour axes
  int nnb;
};

template <int SHAPE>
__device__ __forceinline__ bool free_of_nbrs(const Geo& g, const MoveCtx<SHAPE>& m, V3 d) {
  for (int j = 0; j < m.nnb; ++j) {
    const float4 r = m.nb[j];
    Ori a = Ori{0.0f, 0.0f, 1.0f, 0.0f};
    if (SHAPE != SH_SPHERE) a = as_ori(m.ax[j]);
    if (dep_overlap<SHAPE>(g, d - V3{r.x, r.y, r.z}, a)) return false;
  }
  return true;
}
template <int SHAPE>
__device__ __forceinline__ bool new_only(const Geo& g, const MoveCtx<SHAPE>& m, V3 d) {
  return dep_overlap<SHAPE>(g, d, m.a_new) && !dep_overlap<SHAPE>(g, d - m.rho_old, m.a_old);
}
template <int SHAPE>
__device__ __forceinline__ bool old_only(const Geo& g, const MoveCtx<SHAPE>& m, V3 d) {
  return dep_overlap<SHAPE>(g, d - m.rho_old, m.a_old) && !dep_overlap<SHAPE>(g, d, m.a_new);
}

// Free-volume measurement (hpmc_free_volume; Sec. IV.A): one test depletant per thread at a uniform point of
// the box; free iff it overlaps no colloid of the 27 cells around it (9 x-rows, each one or two spans of the
// cell-ordered arrays).  Integer result: a count, accumulated per warp.
template <int SHAPE>
__global__ void __launch_bounds__(256) k_free_volume(Geo g, Key10 key, float sx, float sy, float sz, long long n,
                                                     const float4* __restrict__ cpos, const float4* __restrict__ caxis,
                                                     const uint32_t* __restrict__ cell_start,
                                                     unsigned long long* __restrict__ count) {
  const int nc = g.nc;
  unsigned long long mine = 0;
  for (long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += (long long)gridDim.x * blockDim.x) {
    const Block4 r = philox(key, (uint32_t)((unsigned long long)s & 0xffffffffull), (uint32_t)((unsigned long long)s >> 32), 0,
                            ctr_word3(P_FREEVOL, 0, 0));
    const V3 p = V3{unit01(r.x) * g.L, unit01(r.y) * g.L, unit01(r.z) * g.L};
    const int ix = cell_axis(g, p.x, sx), iy = cell_axis(g, p.y, sy), iz = cell_axis(g, p.z, sz);
    bool is_free = true;
    for (int row = 0; row < 9 && is_free; ++row) {
      int jy = iy + row % 3 - 1, jz = iz + row / 3 - 1;
      jy += (jy < 0) ? nc : 0; jy -= (jy >= nc) ? nc : 0;
      jz += (jz < 0) ? nc : 0; jz -= (jz >= nc) ? nc : 0;
      const uint32_t rb = ((uint32_t)jz * nc + jy) * nc;
      int x0 = ix - 1, n0 = 3, n1 = 0;
      if (ix == 0) { x0 = nc - 1; n0 = 1; n1 = 2; }
      else if (ix == nc - 1) { x0 = nc - 2; n0 = 2; n1 = 1; }
      for (int part = 0; part < (n1 != 0 ? 2 : 1) && is_free; ++part) {
        const uint32_t b = part == 0 ? cell_start[rb + x0] : cell_start[rb];
        const uint32_t e = part == 0 ? cell_start[rb + x0 + n0] : cell_start[rb + n1];
        for (uint32_t t = b; t < e; ++t) {
          const float4 c = cpos[t];
          Ori a = Ori{0.0f, 0.0f, 1.0f, 0.0f};
          if (SHAPE != SH_SPHERE) a = as_ori(caxis[t]);
          const V3 d = V3{minimg1(g, p.x - c.x), minimg1(g, p.y - c.y), minimg1(g, p.z - c.z)};
          if (dep_overlap<SHAPE>(g, d, a)) { is_free = false; break; }
        }
      }
    }
    mine += is_free ? 1ull : 0ull;
  }
  for (int o = 16; o >= 1; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
  if ((threadIdx.x & 31) == 0 && mine) atomicAdd(count, mine);
}

// Host-buffer path (hpmc_step_host): the poses of the n accepted particles, packed for one small device-to-host copy.
__global__ void __launch_bounds__(256) k_gather_accepted(const uint32_t* __restrict__ list, uint32_t n, const float4* __restrict__ pos,
                                                         const float4* __restrict__ quat, float4* __restrict__ pack) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t pid = list[i];
  pack[i] = pos[pid];
  if (quat) pack[n + i] = quat[pid];
}

template <int SHAPE, bool CB>
__global__ void __launch_bounds__(MOVE_WARPS * 32) k_move(const MoveArgs A) {
  __shared__ int s_excl[MOVE_WARPS][32];
  __shared__ uint32_t s_start[MOVE_WARPS][32];
  __shared__ float4 s_nb[MOVE_WARPS][MAXNB];
  __shared__ float4 s_ax[MOVE_WARPS][SHAPE == SH_SPHERE ? 1 : MAXNB];

  const Geo& g = A.g;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned FULL = 0xffffffffu;
  const int nwarps = gridDim.x * MOVE_WARPS;
  const int nc = g.nc;
  const int px = A.colour & 1, py = (A.colour >> 1) & 1, pz = (A.colour >> 2) & 1;
  const uint32_t colw = A.colour << 8;

  // per-thread counters; uniform quantities are counted by lane 0 only
  uint32_t cnt[C_COUNT];
#pragma unroll
  for (int k = 0; k < C_COUNT; ++k) cnt[k] = 0;
  unsigned long long cnt_drawn = 0, cnt_needed = 0, cnt_eval = 0, cnt_blocks = 0, cnt_cb = 0;

  for (int a = blockIdx.x * MOVE_WARPS + wid; a < A.nact; a += nwarps) {
    const int ax_ = a % A.hc, ay_ = (a / A.hc) % A.hc, az_ = a / (A.hc * A.hc);
    const int ix = 2 * ax_ + px, iy = 2 * ay_ + py, iz = 2 * az_ + pz;
    const uint32_t cell = ((uint32_t)iz * nc + iy) * nc + ix;
    const uint32_t cb = A.cell_start[cell], ce = A.cell_start[cell + 1];
    const uint32_t nocc = ce - cb;
    if (nocc == 0) continue;

    // ---- a3: pick
    const Block4 rs = philox(A.key, cell, 0, 0, P_SELECT + colw);
    const uint32_t slot = cb + __umulhi(rs.x, nocc);
    const float4 p0 = A.cpos[slot];
    const uint32_t pid = __float_as_uint(p0.w);
    const V3 r0 = V3{p0.x, p0.y, p0.z};
    Q4 q0 = Q4{1.0f, 0.0f, 0.0f, 0.0f};
    if (SHAPE != SH_SPHERE) q0 = as_q(A.quat[pid]);

    // ---- a4: trial pose
    const Block4 rm = philox(A.key, pid, 0, 0, P_MOVE + colw);
    uint32_t ublocks = 2;                         // warp-uniform Philox blocks of this move
    const bool rot = (A.a_max > 0.0f) && (rm.w & 1u);
    V3 r1 = r0;
    Q4 q1 = q0;
    if (!rot) {
      r1 = V3{wrap1(g, r0.x + A.d_max * sym_unit(rm.x)), wrap1(g, r0.y + A.d_max * sym_unit(rm.y)),
              wrap1(g, r0.z + A.d_max * sym_unit(rm.z))};
    } else {
      const V3 v = ball_sample(A.key, pid, 0, 0, P_MOVE + colw + (1u << 16), A.a_max, A.a_max2, ublocks);
      q1 = rotate_cayley(q0, v);
    }
    int out = OUT_NONE;
    // confinement (L180)
    {
      const int jx = cell_axis(g, r1.x, A.sx), jy = cell_axis(g, r1.y, A.sy), jz = cell_axis(g, r1.z, A.sz);
      if (jx != ix || jy != iy || jz != iz) out = OUT_BOUNDARY;
    }

    uint32_t Nd = 0, needed = 0, lane_eval = 0, lane_blocks = 0, cbre = 0;
    if (out == OUT_NONE) {
      // ---- a5: stage the 27-cell neighbourhood (local frame of the new centre)
      uint32_t nstart = 0;
      int ncnt = 0;
      if (lane < 27) {
        const int dz = lane / 9 - 1, dy = (lane / 3) % 3 - 1, dx = lane % 3 - 1;
        int jx = ix + dx, jy = iy + dy, jz = iz + dz;
        jx += (jx < 0) ? nc : 0; jx -= (jx >= nc) ? nc : 0;
        jy += (jy < 0) ? nc : 0; jy -= (jy >= nc) ? nc : 0;
        jz += (jz < 0) ? nc : 0; jz -= (jz >= nc) ? nc : 0;
        const uint32_t cj = ((uint32_t)jz * nc + jy) * nc + jx;
        nstart = A.cell_start[cj];
        ncnt = (int)(A.cell_start[cj + 1] - nstart);
      }
      int incl = ncnt;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += t;
      }
      const int total = __shfl_sync(FULL, incl, 31);
      s_excl[wid][lane] = incl - ncnt;
      s_start[wid][lane] = nstart;
      __syncwarp();
      int nnb = 0;
      for (int base = 0; base < total; base += 32) {
        const int t = base + lane;
        bool keep = false;
        float4 pj = make_float4(0.f, 0.f, 0.f, 0.f);
        uint32_t sj = 0;
        V3 rho = V3{0.f, 0.f, 0.f};
        if (t < total) {
          int c = 0;                              // largest c with s_excl[c] <= t
#pragma unroll
          for (int step = 16; step >= 1; step >>= 1)
            if (c + step < 27 && s_excl[wid][c + step] <= t) c += step;
          sj = s_start[wid][c] + (uint32_t)(t - s_excl[wid][c]);
          pj = A.cpos[sj];
          rho = V3{minimg1(g, pj.x - r1.x), minimg1(g, pj.y - r1.y), minimg1(g, pj.z - r1.z)};
          keep = (__float_as_uint(pj.w) != pid) && (dot3(rho, rho) < g.rcut2);
        }
        const unsigned km = __ballot_sync(FULL, keep);
        if (keep) {
          const int at = nnb + __popc(km & ((1u << lane) - 1u));
          if (at < MAXNB) {
            s_nb[wid][at] = make_float4(rho.x, rho.y, rho.z, 0.0f);
            if (SHAPE != SH_SPHERE) s_ax[wid][at] = A.caxis[sj];
          }
        }
        nnb += __popc(km);
      }
      if (nnb > MAXNB) {
        if (lane == 0) atomicMax(A.err_flag, 1);
        nnb = MAXNB;
      }
      __syncwarp();

      MoveCtx<SHAPE> m;
      m.rho_old = V3{minimg1(g, r0.x - r1.x), minimg1(g, r0.y - r1.y), minimg1(g, r0.z - r1.z)};
      m.a_old = ori_of<SHAPE>(q0);
      m.a_new = ori_of<SHAPE>(q1);
      m.nb = s_nb[wid];
      m.ax = s_ax[wid];
      m.nnb = nnb;

      // ---- a6: hard overlap, neighbours across lanes
      bool hard = false;
      for (int j = lane; j < nnb; j += 32) {
        const float4 r = s_nb[wid][j];
        Ori aB = Ori{0.0f, 0.0f, 1.0f, 0.0f};
        if (SHAPE != SH_SPHERE) aB = as_ori(s_ax[wid][j]);
        if (pair_overlap<SHAPE>(g, V3{r.x, r.y, r.z}, m.a_new, aB)) hard = true;
      }
      if (__any_sync(FULL, hard)) out = OUT_HARD;

      if (out == OUT_NONE) {
        // ---- a7: N_d by table inversion
        if (A.pt_n > 0) {
          const Block4 rn = philox(A.key, pid, 0, 0, P_NDEP + colw);
          ++ublocks;
          const unsigned long long U = ((unsigned long long)rn.x << 32) | rn.y;
          int lo = 0, hi = A.pt_n;
          while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (__ldg(&A.ptable[mid]) <= U) lo = mid + 1; else hi = mid;
          }
          Nd = A.pt_klo + (uint32_t)lo;
        }
        const uint32_t c3dep = P_DEPPOS + colw;
        const uint32_t c3cb = P_CBPOS + colw;
        needed = Nd;
        if (!CB) {
          // ---- a8: plain rule; 32 consecutive depletants per step, exit on the first rejecting one
          bool rejected = false;
          for (uint32_t base = 0; base < Nd && !rejected; base += 32) {
            const uint32_t k = base + lane;
            bool rej = false;
            if (k < Nd) {
              const V3 d = dep_position(A, pid, k, c3dep, lane_blocks);
              ++lane_eval;
              rej = new_only<SHAPE>(g, m, d) && free_of_nbrs<SHAPE>(g, m, d);
            }
            const unsigned rm_ = __ballot_sync(FULL, rej);
            if (rm_) { needed = base + (uint32_t)__ffs(rm_); rejected = true; }
          }
          out = rejected ? OUT_DEPLETANT : OUT_ACCEPT;
        } else {
          // ---- a8 + a9: configurational bias, Eq. 16 with readings G1-G3
          float P = 1.0f;
          bool any = false, zero = false;
          const uint32_t ne = 2u * (uint32_t)A.n_trial;
          // OPT_ROSENBLUTH (R-N4): the last reverse reinsertion is not drawn (the original depletant takes its place)
          const bool rosen = (A.options & OPT_ROSENBLUTH) != 0u;
          const uint32_t e_skip = rosen ? ne - 1u : 0xffffffffu;
          for (uint32_t base = 0; base < Nd && !zero; base += 32) {
            const uint32_t k = base + lane;
            bool rej = false;
            if (k < Nd) {
              const V3 d = dep_position(A, pid, k, c3dep, lane_blocks);
              ++lane_eval;
              rej = new_only<SHAPE>(g, m, d) && free_of_nbrs<SHAPE>(g, m, d);
            }
            unsigned rmask = __ballot_sync(FULL, rej);
            while (rmask) {
              const uint32_t kk = base + (uint32_t)__ffs(rmask) - 1u;
              rmask &= rmask - 1u;
              any = true;
              uint32_t Ni = 0, Npins = 0, Npi = 0, Nins = 0;
              for (uint32_t e0 = 0; e0 < ne; e0 += 32) {
                const uint32_t e = e0 + lane;
                bool valid = false, fr = false;
                const uint32_t dir = e & 1u, t = e >> 1;
                if (e < ne && e != e_skip) {
                  V3 s = ball_sample(A.key, pid, kk, t + (dir << 16), c3cb, g.Rins, g.Rins2, lane_blocks);
                  if (dir == 0) {                 // forward: about the old centre, must overlap the old pose only
                    s = s + m.rho_old;
                    valid = old_only<SHAPE>(g, m, s);
                  } else {                        // reverse: about the new centre, must overlap the new pose only
                    valid = new_only<SHAPE>(g, m, s);
                  }
                  fr = valid && free_of_nbrs<SHAPE>(g, m, s);
                }
                const unsigned vm = __ballot_sync(FULL, valid), fm = __ballot_sync(FULL, fr);
                Ni += __popc(vm & 0x55555555u);   Npi += __popc(vm & 0xAAAAAAAAu);
                Npins += __popc(fm & 0x55555555u); Nins += __popc(fm & 0xAAAAAAAAu);
              }
              cbre += rosen ? ne - 1u : ne;
              if (Npins == 0) { zero = true; needed = kk + 1u; break; }
              const float wk = rosen ? __fdiv_rn((float)Npins, (float)(Nins + 1u))
                                     : __fdiv_rn((float)(Npins * (Npi + 1u)), (float)((Nins + 1u) * Ni));
              P = P * wk;
            }
          }
          if (zero) out = OUT_CB;
          else if (!any) out = OUT_ACCEPT;
          else {
            const Block4 ra = philox(A.key, pid, 0, 0, P_ACCEPT + colw);
            ++ublocks;
            out = (unit01(ra.x) < P) ? OUT_ACCEPT : OUT_CB;
          }
        }
      }
    }

    // ---- a10: commit
    if (lane == 0) {
      A.outcome[pid] = (uint8_t)out;
      if (out == OUT_ACCEPT) {
        float4 pn = A.pos[pid];
        pn.x = r1.x; pn.y = r1.y; pn.z = r1.z;
        A.pos[pid] = pn;
        if (A.acc_list) A.acc_list[atomicAdd(A.acc_count, 1u)] = pid;
        A.cpos[slot] = make_float4(r1.x, r1.y, r1.z, p0.w);
        if (SHAPE != SH_SPHERE && rot) {
          A.quat[pid] = as_f4(q1);
          A.caxis[slot] = as_f4(ori_of<SHAPE>(q1));
        }
      }
      ++cnt[rot ? C_TRIALS_ROT : C_TRIALS_TRANS];
      if (out == OUT_ACCEPT) ++cnt[rot ? C_ACCEPT_ROT : C_ACCEPT_TRANS];
      else if (out == OUT_BOUNDARY) ++cnt[C_REJ_BOUNDARY];
      else if (out == OUT_HARD) ++cnt[C_REJ_HARD];
      else if (out == OUT_DEPLETANT) ++cnt[C_REJ_DEPLETANT];
      else ++cnt[C_REJ_CB];
      if (out != OUT_BOUNDARY && out != OUT_HARD) { cnt_drawn += Nd; cnt_needed += needed; }
      cnt_cb += cbre;
      cnt_blocks += ublocks;
    }
    cnt_eval += lane_eval;
    cnt_blocks += lane_blocks;
    __syncwarp();
  }

  // ---- counters: warp reduction, one atomic per warp and counter
  for (int o = 16; o >= 1; o >>= 1) {
    cnt_eval += __shfl_xor_sync(FULL, cnt_eval, o);
    cnt_blocks += __shfl_xor_sync(FULL, cnt_blocks, o);
  }
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < C_REJ_CB + 1; ++k)
      if (cnt[k]) atomicAdd(&A.counters[k], (unsigned long long)cnt[k]);
    if (cnt_drawn) atomicAdd(&A.counters[C_DEP_DRAWN], cnt_drawn);
    if (cnt_needed) atomicAdd(&A.counters[C_DEP_NEEDED], cnt_needed);
    if (cnt_eval) atomicAdd(&A.counters[C_DEP_EVALUATED], cnt_eval);
    if (cnt_cb) atomicAdd(&A.counters[C_CB_REINSERTIONS], cnt_cb);
    if (cnt_blocks) atomicAdd(&A.counters[C_PHILOX_BLOCKS], cnt_blocks);
  }
}

}  // namespace hpmc
