// moveq.cuh -- steps a3..a10, item-queue design of the checkerboard move kernel (K-B).
//
// C3 has 175,616 active cells per pass and a B200 holds ~150k resident threads of this kernel, so a pass is ONE wave
// of work.  Every phase is spread over all T lanes of the CTA and every dependent-load chain is kept short:
//   tiling   every CTA owns a contiguous range of active cells, sized by the host so that all CTAs are resident at
//            once (one wave, no tile counter), and handles it as one tile of <= CPT*T cells (more tiles only for
//            systems too large for one wave); C3: 1179 CTAs x 149 cells, ~73 moves per 128 lanes.
//   phase 1a one THREAD per active cell: pick (a3), trial pose + confinement (a4).  Moves that stay in their cell are
//            compacted into a dense list in shared memory (empty cells and boundary rejections drop out here).
//   phase 1b one thread per (move, x-row) item, 9 rows per move: the row's 3 cells are one contiguous span of the
//            cell-ordered array (two spans when the row wraps); four particle loads are in flight per item, rows with
//            more particles hand their rest to an overflow queue that a second pass spreads over all lanes; the sphere
//            hard-overlap test runs inline (a5, a6), neighbours that a depletant of the move can touch are pushed on
//            the move's linked list in a CTA-wide shared-memory pool.  Moves more than two cells away from the
//            coordinate wrap skip the minimum image (the plain difference is the minimum image there).
//   phase 1c (convex shapes) the (move, neighbour) pairs inside the circumsphere distance are items of their own;
//            the CTA's lanes run the support-function test on them side by side.
//   phase 1d one thread per move: N_d by table inversion (a7), one 16-byte load instead of an eleven-step binary
//            search thanks to a 4096-bucket guide table indexed by the top 12 bits of the uniform.
//   phase 2  the depletant insertions of ALL surviving moves of the tile are one pool of items
//            (move m, depletant k, attempt a).  Every lane repeatedly claims the next k of the move it is
//            attached to (shared-memory atomic), computes ONE Philox block per loop trip, and on an accepted
//            cube-rejection attempt applies the free-volume test (L68, L72); a rejecting k is folded in with
//            atomicMin.  A lane whose move is exhausted re-attaches to any unfinished move of the tile, so short
//            moves (the common case: ~14 needed insertions) cost ~14 lane-items instead of a 32-lane batch, and
//            long ones (accepted moves test all N_d ~ 2.8k at C3) are shared by up to T lanes.
//   commit   the owner thread writes outcome, pose, counters (a10).
// Results are identical to the sequential definition: the outcome depends only on whether a rejecting depletant
// exists, and dep_needed = (smallest rejecting k) + 1 is exact because k's are claimed in ascending order and a
// claimed k below the current minimum is never abandoned.  The order of a move's neighbour list does not matter:
// "overlaps no other colloid" is a disjunction.
//
// PAPER.md: move rule L64-68, Fig. 2 L72; insertion sphere L156; checkerboard + confinement L180; the paper's
// own GPU layout (App. A: one kernel for trial moves, one thread GROUP per depletant) is prior art.
#pragma once
#include <cstdint>
#include "geometry.cuh"
#include "move.cuh"
#include "philox.cuh"

namespace hpmc {

struct QArgs {
  MoveArgs m;
  unsigned long long magic_hc;     // floor(2^64 / hc) + 1: exact a / hc by __umul64hi for a < 2^32
  const uint4* pguide;             // [4096] guide table of the Poisson thresholds (poisson_count), or nullptr
  float wlo, whi;                  // 2.1 w and L - 2.1 w: centres in between need no minimum image (phase 1b)
  float ramp;                      // share of the first / last CTA relative to the average: 1 + ramp / 1 - ramp
  int tile_cells;                  // a CTA works through its share in tiles of tile_cells <= CPT*T cells (normally one)
  // ---- one launch per sweep (npass = 8): a CTA keeps its share of the active-cell index space for all 8 colours
  // and runs the passes back to back.  Instead of a grid-wide barrier it waits, before the neighbourhood walk of pass
  // p, only for the CTAs whose shares touch its own 27-cell neighbourhoods to have published pass p-1 (done[b] >= seq0 + p).
  int npass;                       // 1: the colour in m.colour (one launch per pass); 8: colours[0..7] in this launch
  uint32_t colours[8];
  const uint32_t* cta_first;       // [gridDim.x + 1] first active-cell index of every CTA's share (host table, with the ramp)
  uint32_t* done;                  // [gridDim.x] passes published so far (monotone over the sweeps of a context)
  uint32_t seq0;                   // value of done[] before this sweep
#ifdef HPMC_PHASE_CLOCKS
  unsigned long long* phase_clk;   // tuning build: [8] clock64 sums of thread 0 over the phases of every tile
#endif
  float rlist2;                    // neighbours farther than this from the new centre cannot touch any depletant
                                   // of the move: (sigma_c + sigma_d + 1e-3)^2 for the plain rule (insertion
                                   // sphere about the new centre only), r_cut^2 of R-3.4 otherwise
};

// s = 2u - 1 with u = ((x >> 9) + 0.5) 2^-23 (R-S4).  Every step is exact in binary32, so this three-instruction
// form gives the same bits as the (float)(x >> 9) form: f = 1 + n 2^-23, t = f - 1.5, s = 2 t + 2^-23.
__device__ __forceinline__ float sym_unit_bits(uint32_t x) {
  const float f = __uint_as_float((x >> 9) | 0x3f800000u);
  return fmaf(f - 1.5f, 2.0f, 1.1920928955078125e-07f);
}

#ifndef HPMC_WALK_DEFER
#define HPMC_WALK_DEFER 1
#endif
// One-launch sweep: how long (wall clock, %globaltimer) a CTA waits for a neighbouring CTA's pass before it abandons the
// sweep with error code 2 (HPMC_E_CUDA).  Not a tuning knob: the cooperative launch makes every wait finite, so this only
// turns a lost CTA into an error instead of a hang.  (The abandon path is tested with a build that sets it to microseconds.)
#ifndef HPMC_WAIT_LIMIT_NS
#define HPMC_WAIT_LIMIT_NS 60000000000ull
#endif
#ifndef HPMC_WALK_SLOTS
#define HPMC_WALK_SLOTS 4         // phase 1b: particle loads in flight per (move, row) item
#endif

#ifdef HPMC_PHASE_CLOCKS
__device__ unsigned long long g_dbg_trips[2];    // tuning build: loop trips of thread 0 in phase 2, tiles
#endif

template <int SHAPE>
struct QLayout {
  static constexpr bool ANISO = SHAPE != SH_SPHERE;
  static constexpr int ENTRY = ANISO ? 2 : 1;                 // float4 per neighbour entry
  static constexpr int POOL_PER_MOVE = ANISO ? 12 : 6;        // pool capacity = this x T entries (tile average)
  static constexpr int HCAP_PER_MOVE = 4;                     // hard-test items (convex shapes) = this x T
  static constexpr int MIN_CTAS = ANISO ? 1 : 8;              // resident CTAs per SM the register allocation must allow
};

// shared-memory carve-up for a CTA of T threads handling tiles of up to M = CPT*T active cells (hence <= M moves)
#ifndef HPMC_CB_WINDOW
#define HPMC_CB_WINDOW 32          // configurational bias: depletant indices examined per round and move (speculation bound)
#endif

template <int SHAPE, int T, int CPT, bool CB = false>
struct QSmem {
  using Lq = QLayout<SHAPE>;
  static constexpr int M = CPT * T;
  static constexpr int POOL = Lq::POOL_PER_MOVE * T;
  static constexpr int HCAP = Lq::ANISO ? Lq::HCAP_PER_MOVE * T : 0;
  static constexpr size_t o_r1 = 0;                                             // float4[M]  r1.xyz, slot bits (phase 1b reads only this)
  static constexpr size_t o_rho = o_r1 + sizeof(float4) * M;                    // float4[M]  rho_old.xyz, pid bits (phase 2 reads only this + head)
  static constexpr size_t o_q1 = o_rho + sizeof(float4) * M;                    // float4[M]  new quaternion (aniso)
  static constexpr size_t o_aold = o_q1 + (Lq::ANISO ? sizeof(float4) * M : 0); // float4[M]
  static constexpr size_t o_anew = o_aold + (Lq::ANISO ? sizeof(float4) * M : 0);
  static constexpr size_t o_pool = o_anew + (Lq::ANISO ? sizeof(float4) * M : 0);
  static constexpr size_t o_cell = o_pool + sizeof(float4) * (size_t)POOL * Lq::ENTRY;   // u32[M] ix|iy<<10|iz<<20|rot<<30|interior<<31
  static constexpr size_t o_Nd = o_cell + 4 * M;
  static constexpr size_t o_knext = o_Nd + 4 * M;
  static constexpr size_t o_rejmin = o_knext + 4 * M;
  static constexpr size_t o_head = o_rejmin + 4 * M;
  static constexpr size_t o_state = o_head + 4 * M;                             // u32[M] outcome code so far
  static constexpr size_t o_todo = o_state + 4 * M;                             // u32[M/32]
  static constexpr size_t o_hitems = o_todo + 4 * (M / 32);
  static constexpr size_t o_scal = o_hitems + 4 * HCAP;                         // u32[8]
  static constexpr size_t o_alive = o_scal + 32;                                // u16[M]
  static constexpr size_t o_ovf = o_alive + 2 * M;                              // u32[T] overflow queue of phase 1b
  static constexpr size_t o_cnt = o_ovf + 4 * T;                                // u32[16] CTA totals of the counters
  static constexpr size_t o_tcnt = o_cnt + 64;                                  // u32[4] phase-1a counters of the tile in flight
  static constexpr int NBMAP_WORDS = T <= 64 ? 160 : 40;                                        // bitmap over <= 1280 CTAs (8 per SM on 148 SMs fit; the 28,160 B that allow 8 CTAs per SM leave no more room)
  static constexpr size_t o_nbmap = o_tcnt + 16;                                // u32[NBMAP_WORDS] CTAs this one must wait for
  // configurational bias (a9): per move the product so far, the rejecting depletants handled, the window start, the
  // head of its job list; per job (one rejecting depletant of the current window) k, move | next, packed counts
  static constexpr int JCAP = CB ? 4 * T : 0;
  // the job-overflow redo of the CB stage halves the window down to one depletant per move and relies on "one job per
  // move always fits": without this a larger CPT (HPMC_QCPT) would make that loop spin for ever
  static_assert(!CB || M <= JCAP, "configurational bias: a tile must not hold more moves than job slots");
  static constexpr size_t o_P = o_nbmap + 4 * NBMAP_WORDS;                       // float[M]
  static constexpr size_t o_cbre = o_P + (CB ? 4 * M : 0);                       // u32[M] jobs counted (x 2 n_trial = reinsertions)
  static constexpr size_t o_klo = o_cbre + (CB ? 4 * M : 0);                     // u32[M]
  static constexpr size_t o_jhead = o_klo + (CB ? 4 * M : 0);                    // int[M]
  static constexpr size_t o_jk = o_jhead + (CB ? 4 * M : 0);                     // u32[JCAP]
  static constexpr size_t o_jm = o_jk + 4 * JCAP;                                // u32[JCAP] move | (next job + 1) << 16
  static constexpr size_t o_jc = o_jm + 4 * JCAP;                                // uint2[JCAP] (N_i | N'_ins << 16, N'_i | N_ins << 16)
  static constexpr size_t bytes = o_jc + 8 * JCAP;
};

template <int SHAPE>
__device__ __forceinline__ bool q_new_only(const Geo& g, V3 d, V3 rho_old, Ori a_old, Ori a_new) {
  return dep_overlap<SHAPE>(g, d, a_new) && !dep_overlap<SHAPE>(g, d - rho_old, a_old);
}

template <int SHAPE>
__device__ __forceinline__ bool q_free_of_nbrs(const Geo& g, const float4* pool, int head, V3 d) {
  constexpr int E = QLayout<SHAPE>::ENTRY;
  for (int e = head; e >= 0;) {
    const float4 r = pool[e * E];
    Ori a = Ori{0.0f, 0.0f, 1.0f, 0.0f};
    if (SHAPE != SH_SPHERE) a = as_ori(pool[e * E + 1]);
    if (dep_overlap<SHAPE>(g, d - V3{r.x, r.y, r.z}, a)) return false;
    e = __float_as_int(r.w);
  }
  return true;
}

// N_d = k_lo + #{j : T[j] <= U} (R-S2).  Guide table: bucket b = U >> 52 holds {lo = #{T < b 2^52}, n = number of
// thresholds inside the bucket, T[lo] as two words}: one 16-byte load answers the common case (n <= 1); a bucket with
// more thresholds (the far tails of the distribution) falls back to a binary search over its n entries.
__device__ __forceinline__ uint32_t poisson_count(const unsigned long long* __restrict__ T, int n,
                                                  const uint4* __restrict__ guide, unsigned long long U) {
  int lo = 0, hi = n;
  if (guide) {
    const uint4 gb = __ldg(&guide[(uint32_t)(U >> 52)]);
    const unsigned long long t0 = ((unsigned long long)gb.w << 32) | gb.z;
    if (gb.y == 0u || U < t0) return gb.x;
    if (gb.y == 1u) return gb.x + 1u;
    lo = (int)gb.x + 1; hi = (int)(gb.x + gb.y);
  }
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (__ldg(&T[mid]) <= U) lo = mid + 1; else hi = mid;
  }
  return (uint32_t)lo;
}

// Pointers to the phase-2 tables of one CTA.
struct QTables {
  const float4* r1; const float4* rho; const float4* aold; const float4* anew; const float4* pool;
  uint32_t* knext; uint32_t* rejmin; const int* head; uint32_t* todo; const uint16_t* alive;
  // configurational bias: job list of the current window
  uint32_t* jk; uint32_t* jm; uint2* jc; int* jhead; uint32_t* njobs; int jcap;
  // OPT_SHELL (R-N1): depletants in the shell R_in < |d| <= R instead of the whole ball
  float sh_Rin3, sh_dR3;
};

#ifndef HPMC_LANES_PER_OPEN_MOVE
#define HPMC_LANES_PER_OPEN_MOVE 0      // > 0: a lane looking for work retires once t >= this x (open moves): fewer helpers at the end of a tile
#endif

// Phase 2 (a8): the depletant item queue over the `nalive` surviving moves described by `tb`; returns when no move
// of the tile has unclaimed work left and this thread's last item is done.  rejmin[m] starts at N_d and only
// decreases, so "k < rejmin[m]" is the one test for "this depletant still matters".
template <int SHAPE, bool CB, bool SHELL>
__device__ __forceinline__ void q_depletant_queue(const QTables& tb, int nalive, const Geo& g, const Key10& key,
                                                  uint32_t c3dep, int t, uint32_t& n_eval, uint32_t& n_blocks) {
  constexpr bool ANISO = SHAPE != SH_SPHERE;
  if (nalive <= 0) return;
  const int nw_alive = (nalive + 31) >> 5;
  int j = t % nalive;
  uint32_t m = tb.alive[j];
  int c_head = tb.head[m];
  float4 c_rho = tb.rho[m];
  uint32_t c_pid = __float_as_uint(c_rho.w);
  Ori c_aold = Ori{0.f, 0.f, 1.f, 0.f}, c_anew = Ori{0.f, 0.f, 1.f, 0.f};
  if (ANISO) { c_aold = as_ori(tb.aold[m]); c_anew = as_ori(tb.anew[m]); }
  volatile uint32_t* v_rejmin = tb.rejmin;
  volatile uint32_t* v_todo = tb.todo;
  uint32_t k = 0, c3 = c3dep, trip = 0;
  bool have = false, active = true;
  for (;;) {
    // ---- claim (divergent, short): lanes without an item take the next k of their move, or re-attach
    if (active && !have) {
#pragma unroll 1
      for (;;) {
        k = atomicAdd(&tb.knext[m], 1u);
        if (k < v_rejmin[m]) { c3 = c3dep; have = true; break; }
        // this move has no unclaimed work left: retire its bit (idempotent), attach to an unfinished move of the tile
        atomicAnd(&tb.todo[j >> 5], ~(1u << (j & 31)));
        int found = -1;
        int wi = j >> 5;
        uint32_t open = 0;
#pragma unroll 1
        for (int i = 0; i < nw_alive; ++i) {            // only the words that ever held a bit
          const uint32_t w = v_todo[wi];
          if (HPMC_LANES_PER_OPEN_MOVE > 0) open += __popc(w);
          if (w && found < 0) {
            const int r = t & 31;
            const uint32_t w2 = __funnelshift_r(w, w, r);
            found = wi * 32 + ((__ffs(w2) - 1 + r) & 31);
            if (HPMC_LANES_PER_OPEN_MOVE == 0) break;
          }
          wi = (wi + 1 == nw_alive) ? 0 : wi + 1;
        }
        if (HPMC_LANES_PER_OPEN_MOVE > 0 && (uint32_t)t >= HPMC_LANES_PER_OPEN_MOVE * open) found = -1;
        if (found < 0) { active = false; break; }
        j = found;
        m = tb.alive[j];
        c_head = tb.head[m]; c_rho = tb.rho[m]; c_pid = __float_as_uint(c_rho.w);
        if (ANISO) { c_aold = as_ori(tb.aold[m]); c_anew = as_ori(tb.anew[m]); }
      }
    }
    // the vote is also the reconvergence point: the Philox block below runs with the whole warp together
    // (checked every fourth trip: a warp that has run dry idles through at most three cheap trips)
    if ((++trip & 3u) == 0u && !__any_sync(0xffffffffu, active)) {
#ifdef HPMC_PHASE_CLOCKS
      if (t == 0) { atomicAdd(&g_dbg_trips[0], (unsigned long long)trip); atomicAdd(&g_dbg_trips[1], 1ull); }
#endif
      break;
    }
    if (active) {
      // one Philox block = one cube-rejection attempt of depletant k (R-S3); c3 carries the attempt number
      const Block4 r = philox(key, c_pid, k, 0, c3);
      ++n_blocks;
      V3 d;
      float d2;
      bool inside;
      if (!SHELL) {
        d = V3{g.Rins * sym_unit_bits(r.x), g.Rins * sym_unit_bits(r.y), g.Rins * sym_unit_bits(r.z)};
        d2 = dot3(d, d);
        inside = d2 <= g.Rins2;
        if (!inside && c3 >= c3dep + (63u << 16)) { d = V3{0.f, 0.f, 0.f}; d2 = 0.0f; inside = true; }
      } else {
        inside = shell_attempt(r, tb.sh_Rin3, tb.sh_dR3, d);
        if (!inside && c3 >= c3dep + (63u << 16)) { d = V3{g.Rins, 0.f, 0.f}; inside = true; }
        d2 = inside ? dot3(d, d) : 0.0f;
      }
      if (inside) {
        ++n_eval;
        const V3 ro = V3{c_rho.x, c_rho.y, c_rho.z};
        // new-only (L72): overlaps the new pose (|d|^2 < R^2 is dep_overlap's own first test, same value as d2) ...
        bool hit;
        if (ANISO) hit = q_new_only<SHAPE>(g, d, ro, c_aold, c_anew);
        else { const V3 e = d - ro; hit = (d2 < g.Rins2) && !(dot3(e, e) < g.Rins2); }
        if (hit && q_free_of_nbrs<SHAPE>(g, tb.pool, c_head, d)) {
          if (!CB) {
            atomicMin(&tb.rejmin[m], k);
            atomicAnd(&tb.todo[j >> 5], ~(1u << (j & 31)));   // every k below this one is already claimed: closed for newcomers
          } else {
            // Sec. III.D: a rejecting depletant does not end the move; it becomes a reinsertion job of this window
            const uint32_t jb = atomicAdd(tb.njobs, 1u);
            if (jb < (uint32_t)tb.jcap) {
              const int prev = atomicExch(&tb.jhead[m], (int)jb);
              tb.jk[jb] = k; tb.jm[jb] = m | ((uint32_t)(prev + 1) << 16); tb.jc[jb] = make_uint2(0u, 0u);
            }
          }
        }
        have = false;
      } else {
        c3 += 1u << 16;
        if (k > v_rejmin[m]) have = false;     // a lower k already rejects: this one cannot matter
      }
    }
  }
}

#ifdef HPMC_PHASE_CLOCKS      // tuning build (profiles/*_summary.md "phase split"): thread 0 sums clock64 deltas per phase
#define HPMC_PHASE_MARK(i) do { if (threadIdx.x == 0) { const long long c_ = clock64(); pclk[i] += (unsigned long long)(c_ - pclk_t); pclk_t = c_; } } while (0)
#else
#define HPMC_PHASE_MARK(i) do { } while (0)
#endif

template <int SHAPE, int T, int CPT, bool CB>
__global__ void __launch_bounds__(T, (CB ? 1 : QLayout<SHAPE>::MIN_CTAS * (T < 128 ? 128 / T : 1))) k_moveq(const QArgs Q) {
#ifdef HPMC_PHASE_CLOCKS
  unsigned long long pclk[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  long long pclk_t = clock64();
#endif
  using Lq = QLayout<SHAPE>;
  using S = QSmem<SHAPE, T, CPT, CB>;
  constexpr bool ANISO = Lq::ANISO;
  constexpr int E = Lq::ENTRY;
  constexpr int M = S::M, POOL = S::POOL, HCAP = S::HCAP, NW = M / 32;
  constexpr int SLOTS = HPMC_WALK_SLOTS;
  constexpr bool DEFER = HPMC_WALK_DEFER && !ANISO && (9 * M < 65536);   // overflow queue of phase 1b
  const MoveArgs& A = Q.m;
  const Geo& g = A.g;

  extern __shared__ float4 q_smem[];
  char* sb_ = reinterpret_cast<char*>(q_smem);
  float4* s_r1 = reinterpret_cast<float4*>(sb_ + S::o_r1);
  float4* s_rho = reinterpret_cast<float4*>(sb_ + S::o_rho);
  float4* s_q1 = reinterpret_cast<float4*>(sb_ + S::o_q1);
  float4* s_aold = reinterpret_cast<float4*>(sb_ + S::o_aold);
  float4* s_anew = reinterpret_cast<float4*>(sb_ + S::o_anew);
  float4* s_pool = reinterpret_cast<float4*>(sb_ + S::o_pool);
  uint32_t* s_cell = reinterpret_cast<uint32_t*>(sb_ + S::o_cell);
  uint32_t* s_Nd = reinterpret_cast<uint32_t*>(sb_ + S::o_Nd);
  uint32_t* s_knext = reinterpret_cast<uint32_t*>(sb_ + S::o_knext);
  uint32_t* s_rejmin = reinterpret_cast<uint32_t*>(sb_ + S::o_rejmin);
  int* s_head = reinterpret_cast<int*>(sb_ + S::o_head);
  uint32_t* s_state = reinterpret_cast<uint32_t*>(sb_ + S::o_state);
  uint32_t* s_todo = reinterpret_cast<uint32_t*>(sb_ + S::o_todo);
  uint32_t* s_hitems = reinterpret_cast<uint32_t*>(sb_ + S::o_hitems);
  uint32_t* s_scal = reinterpret_cast<uint32_t*>(sb_ + S::o_scal);   // [0] nalive [1] pool top [3] nhard [4] nlist
  uint16_t* s_alive = reinterpret_cast<uint16_t*>(sb_ + S::o_alive);
  uint32_t* s_ovf = reinterpret_cast<uint32_t*>(sb_ + S::o_ovf);
  uint32_t* s_cnt = reinterpret_cast<uint32_t*>(sb_ + S::o_cnt);
  uint32_t* s_tcnt = reinterpret_cast<uint32_t*>(sb_ + S::o_tcnt);  // [0] trials_trans [1] trials_rot [2] rej_boundary of this tile
  float* s_P = reinterpret_cast<float*>(sb_ + S::o_P);               // configurational bias only (CB)
  uint32_t* s_cbre = reinterpret_cast<uint32_t*>(sb_ + S::o_cbre);
  uint32_t* s_klo = reinterpret_cast<uint32_t*>(sb_ + S::o_klo);
  int* s_jhead = reinterpret_cast<int*>(sb_ + S::o_jhead);
  uint32_t* s_jk = reinterpret_cast<uint32_t*>(sb_ + S::o_jk);
  uint32_t* s_jm = reinterpret_cast<uint32_t*>(sb_ + S::o_jm);
  uint2* s_jc = reinterpret_cast<uint2*>(sb_ + S::o_jc);

  const int t = threadIdx.x;
  const int nc = g.nc, hc = A.hc;
  // per-thread counters (reduced once at the end of the kernel): the two that tick in the hot loop live in
  // registers; the per-move ones go to CTA totals in shared memory (far below 2^32)
  uint32_t n_eval = 0, n_blocks = 0;
  if (t < C_COUNT) s_cnt[t] = 0u;               // ordered before the first use by the barrier at the top of the tile loop
  if (t == 0) s_scal[6] = 0u;                   // "a neighbour wait timed out", likewise

  // CTA b owns the active-cell indices [cta_first[b], cta_first[b+1]) for every colour; the host table gives the
  // first-launched CTAs a larger share (the SM's warp arbitration favours them; see setup_moveq).
  const uint32_t cta_lo = Q.cta_first[blockIdx.x];
  const uint32_t cta_hi = Q.cta_first[blockIdx.x + 1u];

  // ---- neighbour CTAs (npass > 1): every CTA whose share holds a cell of the x-rows (az+dz, ay+dy), dz, dy in
  // {-1,0,1}, of the rows this share touches -- a superset of the 27-cell neighbourhoods of its cells.  Bitmap over CTAs.
  uint32_t* s_nbmap = reinterpret_cast<uint32_t*>(sb_ + S::o_nbmap);
  if (Q.npass > 1) {
    for (int w = t; w < S::NBMAP_WORDS; w += T) s_nbmap[w] = 0u;
    __syncthreads();
    if (cta_hi > cta_lo) {
      const int r_lo = (int)(cta_lo / (uint32_t)hc), r_hi = (int)((cta_hi - 1u) / (uint32_t)hc);
      const int nrow = r_hi - r_lo + 1;
      for (int it = t; it < nrow * 9; it += T) {
        const int r = r_lo + it / 9, o = it % 9;
        int az = r / hc + (o / 3 - 1), ay = r % hc + (o % 3 - 1);
        az += (az < 0) ? hc : 0; az -= (az >= hc) ? hc : 0;
        ay += (ay < 0) ? hc : 0; ay -= (ay >= hc) ? hc : 0;
        const uint32_t a0 = (uint32_t)(az * hc + ay) * (uint32_t)hc, a1 = a0 + (uint32_t)hc - 1u;
        // CTAs owning a0 and a1: largest b with cta_first[b] <= a
        uint32_t b0 = 0, b1 = 0;
        {
          uint32_t lo = 0, hi = gridDim.x;
          while (hi - lo > 1u) { const uint32_t mid = (lo + hi) >> 1; if (Q.cta_first[mid] <= a0) lo = mid; else hi = mid; }
          b0 = lo; lo = b0; hi = gridDim.x;
          while (hi - lo > 1u) { const uint32_t mid = (lo + hi) >> 1; if (Q.cta_first[mid] <= a1) lo = mid; else hi = mid; }
          b1 = lo;
        }
        for (uint32_t b = b0; b <= b1; ++b)
          if (b != blockIdx.x) atomicOr(&s_nbmap[b >> 5], 1u << (b & 31));
      }
    }
    __syncthreads();
  }

  uint32_t tile_cap = (uint32_t)Q.tile_cells;     // halved (for the rest of this CTA's share) when a tile's neighbour pool overflows
  bool gave_up = false;                           // a neighbour wait ran into HPMC_WAIT_LIMIT_NS (CTA-uniform)
#pragma unroll 1
  for (int pass = 0; pass < Q.npass; ++pass) {
  const uint32_t colour = Q.npass > 1 ? Q.colours[pass] : A.colour;
  const int px = colour & 1, py = (colour >> 1) & 1, pz = (colour >> 2) & 1;
  const uint32_t colw = colour << 8;
  const uint32_t c3dep = P_DEPPOS + colw;
  bool must_wait = pass > 0;                      // pass 0 follows the cell build in stream order
  for (uint32_t cur = cta_lo; cur < cta_hi;) {
    const uint32_t tile_n = min(tile_cap, cta_hi - cur);
    const uint32_t tile_lo = cur;
    cur += tile_n;
    if (t == 0) { s_scal[0] = 0; s_scal[1] = 0; s_scal[3] = 0; s_scal[4] = 0; s_scal[7] = 0; }
    if (t < 4) s_tcnt[t] = 0u;
    __syncthreads();
    HPMC_PHASE_MARK(0);        // idle/tile setup (incl. the publish of the previous pass)

    // ================================================================ phase 1a: one thread per active cell
#pragma unroll 1
    for (uint32_t c = t; c < tile_n; c += T) {
      const uint32_t a = tile_lo + c;
      {
        const uint32_t q1d = (uint32_t)__umul64hi((unsigned long long)a, Q.magic_hc);        // a / hc
        const uint32_t q2d = (uint32_t)__umul64hi((unsigned long long)q1d, Q.magic_hc);      // a / hc^2
        const int ix = 2 * (int)(a - q1d * hc) + px, iy = 2 * (int)(q1d - q2d * hc) + py, iz = 2 * (int)q2d + pz;
        const uint32_t cell = ((uint32_t)iz * nc + iy) * nc + ix;
        const uint32_t cb = A.cell_start[cell], ce = A.cell_start[cell + 1];
        const uint32_t nocc = ce - cb;
        if (nocc != 0) {
          // ---- a3: pick
          const Block4 rs = philox(A.key, cell, 0, 0, P_SELECT + colw);
          const uint32_t slot = cb + __umulhi(rs.x, nocc);
          const float4 p0 = A.cpos[slot];
          const uint32_t pid = __float_as_uint(p0.w);
          const V3 r0 = V3{p0.x, p0.y, p0.z};
          Q4 q0 = Q4{1.0f, 0.0f, 0.0f, 0.0f};
          if (ANISO) q0 = as_q(A.quat[pid]);
          // ---- a4: trial pose
          const Block4 rm = philox(A.key, pid, 0, 0, P_MOVE + colw);
          n_blocks += 2;
          const bool rot = (A.a_max > 0.0f) && (rm.w & 1u);
          V3 r1 = r0;
          Q4 q1 = q0;
          if (!rot) {
            r1 = V3{wrap1(g, r0.x + A.d_max * sym_unit_bits(rm.x)), wrap1(g, r0.y + A.d_max * sym_unit_bits(rm.y)),
                    wrap1(g, r0.z + A.d_max * sym_unit_bits(rm.z))};
            atomicAdd(&s_tcnt[0], 1u);
          } else {
            const V3 v = ball_sample(A.key, pid, 0, 0, P_MOVE + colw + (1u << 16), A.a_max, A.a_max2, n_blocks);
            q1 = rotate_cayley(q0, v);
            atomicAdd(&s_tcnt[1], 1u);
          }
          const int jx = cell_axis(g, r1.x, A.sx), jy = cell_axis(g, r1.y, A.sy), jz = cell_axis(g, r1.z, A.sz);
          if (jx != ix || jy != iy || jz != iz) {        // confinement (L180)
            A.outcome[pid] = (uint8_t)OUT_BOUNDARY;
            atomicAdd(&s_tcnt[2], 1u);
          } else {
            const uint32_t e = atomicAdd(&s_scal[4], 1u);
            s_r1[e] = make_float4(r1.x, r1.y, r1.z, __uint_as_float(slot));
            s_rho[e] = make_float4(minimg1(g, r0.x - r1.x), minimg1(g, r0.y - r1.y), minimg1(g, r0.z - r1.z), p0.w);
            // interior: the new centre is more than two cell widths from the coordinate wrap on every axis, so the
            // minimum image of any neighbour of the 27 cells is the plain difference (|d| < 2w <= L/3 < L/2; n_c >= 6)
            const bool interior = nc >= 6 && r1.x > Q.wlo && r1.x < Q.whi && r1.y > Q.wlo && r1.y < Q.whi &&
                                  r1.z > Q.wlo && r1.z < Q.whi;
            s_cell[e] = (uint32_t)ix | ((uint32_t)iy << 10) | ((uint32_t)iz << 20) | (rot ? (1u << 30) : 0u) |
                        (interior ? (1u << 31) : 0u);
            s_head[e] = -1;
            s_state[e] = OUT_NONE;
            if (ANISO) {
              s_q1[e] = as_f4(q1);
              s_aold[e] = as_f4(ori_of<SHAPE>(q0));
              s_anew[e] = as_f4(ori_of<SHAPE>(q1));
            }
          }
        }
      }
    }
    // ---- passes after the first: the neighbourhood walk reads cells that neighbouring CTAs wrote in the previous
    // pass (and they must be done reading ours): wait for their published pass counter.  Acquire loads by the
    // polling threads + the barrier make their writes visible to the whole CTA.  Phase 1a above touched only this
    // CTA's own cells, so it ran ahead of the wait.  The launch is cooperative, so the neighbour is resident and WILL
    // publish, however slow its pass is (n_trial up to 65535, a clustered share, a debugger): the wait is not bounded in
    // polls.  The wall-clock bound (HPMC_WAIT_LIMIT_NS, looked at every 4096 polls) only guards against a lost CTA, and
    // when it strikes this CTA does not go on against cells its neighbour may still be writing: it raises the error
    // flag and abandons the rest of the sweep (see "gave_up" below).
    HPMC_PHASE_MARK(1);        // phase 1a (thread 0's own share of it)
    if (must_wait) {
      must_wait = false;
      const uint32_t target = Q.seq0 + (uint32_t)pass;
      bool polled = false;
      for (uint32_t b = (uint32_t)t; b < gridDim.x; b += T) {
        if (!((s_nbmap[b >> 5] >> (b & 31)) & 1u)) continue;
        uint32_t v, spins = 0;
        unsigned long long t_first = 0ull;
        for (;;) {       // relaxed polls (no L1 invalidation while spinning), one acquire fence at the end
          asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(Q.done + b) : "memory");
          if ((int32_t)(v - target) >= 0) break;
          if ((++spins & 4095u) == 0u) {
            unsigned long long now;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
            if (t_first == 0ull) t_first = now;
            else if (now - t_first > (unsigned long long)(HPMC_WAIT_LIMIT_NS)) { atomicMax(A.err_flag, 2); s_scal[6] = 1u; break; }
          }
          __nanosleep(spins < 64u ? 40u : 200u);      // short waits are the rule (small systems are latency-bound); back off on long ones
        }
        polled = true;
      }
      if (polled) asm volatile("fence.acq_rel.gpu;" ::: "memory");
    }
    __syncthreads();
    if (Q.npass > 1 && s_scal[6]) { gave_up = true; break; }      // nothing of this tile is committed
    HPMC_PHASE_MARK(2);        // neighbour wait + barrier after 1a
    const int nlist = (int)s_scal[4];

    // ================================================================ phase 1b: one thread per (move, x-row) item
    // Two passes over work units: first every item's leading SLOTS particles; an item with more particles in its row
    // (8 % of the rows at C3, but some lane of nearly every warp) does not make its whole warp loop again: it defers
    // the rest to an overflow queue, and the second pass spreads those leftovers over all lanes of the CTA.
    int n_units = nlist * 9;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
#pragma unroll 1
    for (int un = t; un < n_units; un += T) {
      int it = un;
      uint32_t i_first = 0;
      if (pass != 0) { const uint32_t wq = s_ovf[un]; it = (int)(wq & 0xffffu); i_first = wq >> 16; }
      const int e = it / 9, row = it - 9 * e;
      const float4 r1f = s_r1[e];
      const V3 r1 = V3{r1f.x, r1f.y, r1f.z};
      const uint32_t slot = __float_as_uint(r1f.w);
      const uint32_t cw = s_cell[e];
      const int ix = cw & 1023, iy = (cw >> 10) & 1023, iz = (cw >> 20) & 1023;
      const bool interior = (cw >> 31) != 0u;
      const int dz = row / 3 - 1, dy = row - 3 * (row / 3) - 1;
      int jy = iy + dy, jz = iz + dz;
      jy += (jy < 0) ? nc : 0; jy -= (jy >= nc) ? nc : 0;
      jz += (jz < 0) ? nc : 0; jz -= (jz >= nc) ? nc : 0;
      const uint32_t rb = ((uint32_t)jz * nc + jy) * nc;
      // ---- a5: the row's 3 cells are one contiguous span unless the row wraps in x
      int x0 = ix - 1, n0 = 3, n1 = 0;
      if (ix == 0) { x0 = nc - 1; n0 = 1; n1 = 2; }
      else if (ix == nc - 1) { x0 = nc - 2; n0 = 2; n1 = 1; }
      // one virtual span: the main part [sb0, sb0+len0) followed by the wrapped part [sb1, sb1+len1) (rare)
      const uint32_t sb0 = A.cell_start[rb + x0], len0 = A.cell_start[rb + x0 + n0] - sb0;
      uint32_t sb1 = 0, len1 = 0;
      if (n1 != 0) { sb1 = A.cell_start[rb]; len1 = A.cell_start[rb + n1] - sb1; }
      const uint32_t len = len0 + len1;
      // SLOTS particles in flight per trip (a row holds 2.2 particles on average at C3; more slots cost registers and
      // with them a resident CTA per SM: 4 and 5 measured equal, 6 and 8 slower)
#pragma unroll 1
      for (uint32_t i0 = i_first; i0 < len; i0 += SLOTS) {
        if (DEFER && pass == 0 && i0 != 0) {
          const uint32_t qi = atomicAdd(&s_scal[7], 1u);
          if (qi < (uint32_t)T) { s_ovf[qi] = (uint32_t)it | (i0 << 16); break; }   // queue full: finish inline
        }
        float4 pj[SLOTS];
#pragma unroll
        for (int u = 0; u < SLOTS; ++u) {
          const uint32_t i = i0 + u;
          if (i < len) pj[u] = A.cpos[i < len0 ? sb0 + i : sb1 + (i - len0)];
        }
#pragma unroll
        for (int u = 0; u < SLOTS; ++u) {
          const uint32_t i = i0 + u;
          const uint32_t s = i < len0 ? sb0 + i : sb1 + (i - len0);
          if (i >= len || s == slot) continue;
          V3 rho = V3{pj[u].x - r1.x, pj[u].y - r1.y, pj[u].z - r1.z};
          if (!interior) rho = V3{minimg1(g, rho.x), minimg1(g, rho.y), minimg1(g, rho.z)};
          const float r2 = dot3(rho, rho);
          if (!(r2 < Q.rlist2)) continue;
          if (!ANISO && r2 < g.dcirc2) { s_state[e] = OUT_HARD; continue; }     // a6 (spheres)
          const int pe = (int)atomicAdd(&s_scal[1], 1u);
          if (pe >= POOL) continue;            // the tile is split and redone below (nothing is committed before that)
          const int prev = atomicExch(&s_head[e], pe);
          s_pool[pe * E] = make_float4(rho.x, rho.y, rho.z, __int_as_float(prev));
          if (ANISO) {
            const float4 axj = A.caxis[s];
            s_pool[pe * E + 1] = axj;
            if (r2 < g.dcirc2) {
              const uint32_t hi = atomicAdd(&s_scal[3], 1u);
              if (hi < (uint32_t)HCAP) s_hitems[hi] = ((uint32_t)e << 16) | (uint32_t)pe;
              else {
                if (mpr_overlap<SHAPE>(g, rho, as_ori(s_anew[e]), as_ori(axj))) s_state[e] = OUT_HARD;
              }
            }
          }
        }
      }
    }
      if (!DEFER) break;
      __syncthreads();
      n_units = (int)min(s_scal[7], (uint32_t)T);
    }
    // ================================================================ phase 1c: convex hard-overlap items (a6)
    if (ANISO) {
      __syncthreads();
      const uint32_t nh = min(s_scal[3], (uint32_t)HCAP);
      for (uint32_t i = t; i < nh; i += T) {
        const uint32_t itm = s_hitems[i];
        const uint32_t sl = itm >> 16, pe = itm & 0xffffu;
        const float4 r = s_pool[pe * E], ax = s_pool[pe * E + 1], an = s_anew[sl];
        if (mpr_overlap<SHAPE>(g, V3{r.x, r.y, r.z}, as_ori(an), as_ori(ax)))
          s_state[sl] = OUT_HARD;
      }
    }
    __syncthreads();
    HPMC_PHASE_MARK(3);        // phase 1b + 1c + barrier
    // ---- neighbour pool overflow (a locally dense tile, e.g. a cluster in a dilute box): nothing of this tile is
    // committed yet (boundary outcomes are idempotent, its counters are tile-local), so halve the tile and redo it
    if (s_scal[1] > (uint32_t)POOL) {
      if (tile_n > 1u) { tile_cap = max(1u, tile_n >> 1); cur = tile_lo; __syncthreads(); continue; }
      if (t == 0) atomicMax(A.err_flag, 1);      // ONE move with more listed neighbours than the whole pool holds
    }
    // ================================================================ phase 1d: N_d by table inversion (a7)
#pragma unroll 1
    for (int e = t; e < nlist; e += T) {
      uint32_t Nd = 0;
      if (s_state[e] == OUT_NONE && A.pt_n > 0) {
        const uint32_t pid = __float_as_uint(s_rho[e].w);
        const Block4 rn = philox(A.key, pid, 0, 0, P_NDEP + colw);
        ++n_blocks;
        const unsigned long long U = ((unsigned long long)rn.x << 32) | rn.y;
        Nd = A.pt_klo + poisson_count(A.ptable, A.pt_n, Q.pguide, U);
      }
      s_Nd[e] = Nd; s_knext[e] = 0; s_rejmin[e] = Nd;        // rejmin: smallest rejecting k so far, N_d = none
      if (s_state[e] == OUT_NONE && Nd != 0) s_alive[atomicAdd(&s_scal[0], 1u)] = (uint16_t)e;
    }
    __syncthreads();
    HPMC_PHASE_MARK(4);        // phase 1d + barrier
    if (!CB) {
    const int nalive = (int)s_scal[0];
    for (int w = t; w < NW; w += T) {
      const int rem = nalive - 32 * w;
      s_todo[w] = rem >= 32 ? 0xffffffffu : (rem > 0 ? ((1u << rem) - 1u) : 0u);
    }
    __syncthreads();
    // ================================================================ phase 2: depletant items (a8)
    {
      QTables tb;
      tb.r1 = s_r1; tb.rho = s_rho; tb.aold = s_aold; tb.anew = s_anew; tb.pool = s_pool;
      tb.knext = s_knext; tb.rejmin = s_rejmin; tb.head = s_head; tb.todo = s_todo; tb.alive = s_alive;
      tb.sh_Rin3 = A.sh_Rin3; tb.sh_dR3 = A.sh_dR3;
      if (A.options & OPT_SHELL) q_depletant_queue<SHAPE, false, true>(tb, nalive, g, A.key, c3dep, t, n_eval, n_blocks);
      else q_depletant_queue<SHAPE, false, false>(tb, nalive, g, A.key, c3dep, t, n_eval, n_blocks);
    }
    __syncthreads();
    } else {
    // ================================================================ phase 2 + 3: configurational bias (a8 + a9, Eq. 16)
    // Rounds over windows of W depletant indices per move.  Round: (A) the item queue examines k in [k_lo, k_lo + W)
    // of every running move; rejecting depletants become jobs.  (B) the 2 n_trial reinsertions of every job are items
    // (job, t, dir) spread over the lanes; counts by shared atomics.  (C) one thread per move folds its jobs in
    // ASCENDING k into the fp32 product (the order is part of the definition) and stops at the first zero weight
    // (R-G3), which also fixes dep_needed and the reinsertion count exactly as the sequential definition does.
    const uint32_t ne = 2u * (uint32_t)A.n_trial;
    const uint32_t c3cb = P_CBPOS + colw;
    // OPT_ROSENBLUTH (R-N4): weight N'_ins / (N_ins + 1), the last reverse reinsertion is not drawn
    const bool rosen = (A.options & OPT_ROSENBLUTH) != 0u;
    uint32_t W = HPMC_CB_WINDOW;
    for (int e = t; e < nlist; e += T) { s_P[e] = 1.0f; s_cbre[e] = 0u; s_klo[e] = 0u; }
    __syncthreads();
    for (;;) {
      if (t == 0) { s_scal[0] = 0; s_scal[5] = 0; }
      __syncthreads();
      for (int e = t; e < nlist; e += T) {
        const uint32_t klo = s_klo[e], Nd = s_Nd[e];
        if (s_state[e] == OUT_NONE && klo < Nd) {
          s_alive[atomicAdd(&s_scal[0], 1u)] = (uint16_t)e;
          s_knext[e] = klo; s_rejmin[e] = min(Nd, klo + W); s_jhead[e] = -1;
        }
      }
      __syncthreads();
      const int nalive = (int)s_scal[0];
      if (nalive == 0) break;
      for (int w = t; w < NW; w += T) {
        const int rem = nalive - 32 * w;
        s_todo[w] = rem >= 32 ? 0xffffffffu : (rem > 0 ? ((1u << rem) - 1u) : 0u);
      }
      __syncthreads();
      {
        QTables tb;
        tb.r1 = s_r1; tb.rho = s_rho; tb.aold = s_aold; tb.anew = s_anew; tb.pool = s_pool;
        tb.knext = s_knext; tb.rejmin = s_rejmin; tb.head = s_head; tb.todo = s_todo; tb.alive = s_alive;
        tb.jk = s_jk; tb.jm = s_jm; tb.jc = s_jc; tb.jhead = s_jhead; tb.njobs = &s_scal[5]; tb.jcap = S::JCAP;
        tb.sh_Rin3 = A.sh_Rin3; tb.sh_dR3 = A.sh_dR3;
        if (A.options & OPT_SHELL) q_depletant_queue<SHAPE, true, true>(tb, nalive, g, A.key, c3dep, t, n_eval, n_blocks);
        else q_depletant_queue<SHAPE, true, false>(tb, nalive, g, A.key, c3dep, t, n_eval, n_blocks);
      }
      __syncthreads();
      const uint32_t njobs = s_scal[5];
      if (njobs > (uint32_t)S::JCAP) {       // more rejecting depletants than job slots: redo the round with half the window
        W = max(1u, W >> 1);                 // (W = 1 gives at most one job per move: always fits)
        __syncthreads();
        continue;
      }
      // ---- (B) reinsertion items
      const uint32_t nitems = njobs * ne;
#pragma unroll 1
      for (uint32_t i = t; i < nitems; i += T) {
        const uint32_t jb = i / ne, e2 = i - jb * ne;
        const uint32_t m = s_jm[jb] & 0xffffu, kk = s_jk[jb];
        const uint32_t dir = e2 & 1u, tt = e2 >> 1;
        if (rosen && e2 == ne - 1u) continue;
        const float4 r1f = s_r1[m], rof = s_rho[m];
        const V3 ro = V3{rof.x, rof.y, rof.z};
        Ori ao = Ori{0.f, 0.f, 1.f, 0.f}, an = Ori{0.f, 0.f, 1.f, 0.f};
        if (ANISO) { ao = as_ori(s_aold[m]); an = as_ori(s_anew[m]); }
        V3 sp = ball_sample(A.key, __float_as_uint(rof.w), kk, tt + (dir << 16), c3cb, g.Rins, g.Rins2, n_blocks);
        bool valid;
        if (dir == 0) {                  // forward: about the old centre, must overlap the old pose only (R-G2)
          sp = sp + ro;
          valid = dep_overlap<SHAPE>(g, sp - ro, ao) && !dep_overlap<SHAPE>(g, sp, an);
        } else {                         // reverse: about the new centre, must overlap the new pose only
          valid = q_new_only<SHAPE>(g, sp, ro, ao, an);
        }
        if (valid) {
          const bool fr = q_free_of_nbrs<SHAPE>(g, s_pool, s_head[m], sp);
          atomicAdd(dir == 0 ? &s_jc[jb].x : &s_jc[jb].y, fr ? 0x10001u : 1u);
        }
      }
      __syncthreads();
      // ---- (C) fold the jobs of every running move in ascending k
#pragma unroll 1
      for (int j = t; j < nalive; j += T) {
        const uint32_t e = s_alive[j];
        float P = s_P[e];
        uint32_t cbre = s_cbre[e];
        long long last = -1;
        bool zero = false;
        for (;;) {
          int best = -1; uint32_t bk = 0xffffffffu;
          for (int jb = s_jhead[e]; jb >= 0; jb = (int)(s_jm[jb] >> 16) - 1) {
            const uint32_t kk = s_jk[jb];
            if ((long long)kk > last && kk < bk) { bk = kk; best = jb; }
          }
          if (best < 0) break;
          last = (long long)bk;
          const uint2 c = s_jc[best];
          const uint32_t Ni = c.x & 0xffffu, Npins = c.x >> 16, Npi = c.y & 0xffffu, Nins = c.y >> 16;
          ++cbre;
          if (Npins == 0u) { zero = true; s_state[e] = OUT_CB; s_rejmin[e] = bk + 1u; break; }   // R-G3; dep_needed = k + 1
          P = P * (rosen ? __fdiv_rn((float)Npins, (float)(Nins + 1u))                           // R-N4
                         : __fdiv_rn((float)(Npins * (Npi + 1u)), (float)((Nins + 1u) * Ni)));   // Eq. 16, R-G1
        }
        s_P[e] = P; s_cbre[e] = cbre;
        if (!zero) s_klo[e] = s_rejmin[e];     // window end
      }
      __syncthreads();
    }
    }
    HPMC_PHASE_MARK(5);        // phase 2 (+ CB) + barrier
    // ================================================================ commit (a10)
#pragma unroll 1
    for (int e = t; e < nlist; e += T) {
      int out = (int)s_state[e];
      const float4 r1f = s_r1[e];
      const uint32_t pid = __float_as_uint(s_rho[e].w);
      const bool rot = (s_cell[e] >> 30) & 1u;
      if (!CB && out == OUT_NONE) {
        const uint32_t Nd = s_Nd[e], rm_ = s_rejmin[e];
        const bool rej = rm_ < Nd;
        out = rej ? OUT_DEPLETANT : OUT_ACCEPT;
        atomicAdd(&s_cnt[C_DEP_DRAWN], Nd);
        atomicAdd(&s_cnt[C_DEP_NEEDED], rej ? rm_ + 1u : Nd);
      }
      if (CB && (out == OUT_NONE || out == OUT_CB)) {
        const uint32_t Nd = s_Nd[e], cbre = s_cbre[e];
        atomicAdd(&s_cnt[C_DEP_DRAWN], Nd);
        atomicAdd(&s_cnt[C_DEP_NEEDED], out == OUT_CB ? s_rejmin[e] : Nd);
        if (cbre) atomicAdd(&s_cnt[C_CB_REINSERTIONS], cbre * (2u * (uint32_t)A.n_trial - ((A.options & OPT_ROSENBLUTH) ? 1u : 0u)));
        if (out == OUT_NONE) {
          if (cbre == 0u) out = OUT_ACCEPT;          // no rejecting depletant at all
          else {
            const Block4 ra = philox(A.key, pid, 0, 0, P_ACCEPT + colw);
            ++n_blocks;
            out = (unit01(ra.x) < s_P[e]) ? OUT_ACCEPT : OUT_CB;
          }
        }
      }
      A.outcome[pid] = (uint8_t)out;
      if (out == OUT_ACCEPT) {
        const uint32_t slot = __float_as_uint(r1f.w);
        float4 pn = A.pos[pid];
        pn.x = r1f.x; pn.y = r1f.y; pn.z = r1f.z;
        A.pos[pid] = pn;
        if (A.acc_list) A.acc_list[atomicAdd(A.acc_count, 1u)] = pid;
        A.cpos[slot] = make_float4(r1f.x, r1f.y, r1f.z, __uint_as_float(pid));
        if (ANISO && rot) {
          A.quat[pid] = s_q1[e];
          A.caxis[slot] = s_anew[e];
        }
        atomicAdd(&s_cnt[rot ? C_ACCEPT_ROT : C_ACCEPT_TRANS], 1u);
      } else atomicAdd(&s_cnt[out == OUT_HARD ? C_REJ_HARD : (out == OUT_CB ? C_REJ_CB : C_REJ_DEPLETANT)], 1u);
    }
    if (t == 0) {
      atomicAdd(&s_cnt[C_TRIALS_TRANS], s_tcnt[0]); atomicAdd(&s_cnt[C_TRIALS_ROT], s_tcnt[1]);
      atomicAdd(&s_cnt[C_REJ_BOUNDARY], s_tcnt[2]);
    }
    __syncthreads();
    HPMC_PHASE_MARK(6);        // commit + barrier
  }
  // ---- publish the pass: every commit of this CTA is ordered before the counter by the barrier above + the release
  // (a CTA without cells in this pass has nothing to wait for: it reads and writes no cell.)  A CTA that gave up
  // publishes the counter's end-of-sweep value at once, so that no neighbour waits for passes it will never run and the
  // host's sequence number stays valid for the next sweep; the poses of this sweep are invalid and the flag says so.
  if (Q.npass > 1) {
    if (t == 0) {
      const uint32_t v = Q.seq0 + (uint32_t)(gave_up ? Q.npass : pass + 1);
      asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(Q.done + blockIdx.x), "r"(v) : "memory");
    }
  }
  if (gave_up) break;
  }   // pass

  // ---- counters: REDUX for the two register counters, then one global atomic per CTA and counter
  {
    const unsigned FULL = 0xffffffffu;
    const uint32_t xe = __reduce_add_sync(FULL, n_eval), xb = __reduce_add_sync(FULL, n_blocks);
    if ((t & 31) == 0) {
      if (xe) atomicAdd(&s_cnt[C_DEP_EVALUATED], xe);
      if (xb) atomicAdd(&s_cnt[C_PHILOX_BLOCKS], xb);
    }
  }
  __syncthreads();
  if (t < C_COUNT && s_cnt[t]) atomicAdd(&A.counters[t], (unsigned long long)s_cnt[t]);
#ifdef HPMC_PHASE_CLOCKS
  if (t == 0)
    for (int i = 0; i < 8; ++i) atomicAdd(&Q.phase_clk[i], pclk[i]);
#endif
}

}  // namespace hpmc
