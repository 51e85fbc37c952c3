// hpmc_lib.cu -- host driver and C-ABI (include/hpmc.h) of the B200 implicit-depletant HPMC library.
//
// Per sweep:
//   hpmc_build_cells: host draws the grid shift from Philox(seed, step, SWEEP) -> K-A kernels (cells.cuh)
//   hpmc_sweep:       host draws the colour permutation, builds/caches the Poisson threshold table (fp64, R-S2)
//                     -> ONE cooperative launch of the item-queue move kernel (moveq.cuh) for the 8 sub-lattice passes;
//                     the warp-per-cell kernel (move.cuh: configurational bias with few reinsertions on small systems,
//                     or HPMC_MOVE_KERNEL=warp) takes 8 launches, one per pass, stream ordered.
// No host synchronisation inside a sweep; no CPU fallback anywhere.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/hpmc.h"
#include "alu_peak.cuh"
#include "cells.cuh"
#include "move.cuh"
#include "moveq.cuh"

using namespace hpmc;

namespace {

thread_local std::string g_init_error;

struct PoissonTable {
  double lambda = -1.0;
  uint32_t k_lo = 0;
  int n = 0;
  unsigned long long* d_T = nullptr;
  uint4* d_G = nullptr;                 // guide table (4096 buckets, see poisson_count in moveq.cuh)
  bool has_guide = false;
  size_t cap = 0;
};

struct QPlan {                         // how the item-queue move kernel is tiled over the active cells (moveq.cuh)
  int ctas = 0;                        // CTAs, all resident at once
  float ramp = 0.0f;                   // work ramp over the CTAs (one launch per pass only)
  int cpc = 0, big = 0;                // average active cells per CTA, tile size
  uint32_t* d_cta_first = nullptr;     // [ctas + 1] first active-cell index of every CTA's share
  uint32_t* d_done = nullptr;          // [ctas] pass counters of the one-launch-per-sweep kernel
  uint32_t seq = 0;                    // value of d_done[] before the next sweep
  bool one_launch = false;             // all 8 passes in one cooperative launch (HPMC_SWEEP_LAUNCHES=8: one launch per pass)
};

struct EventPair { cudaEvent_t a, b; int n = 8; };

}  // namespace

struct hpmc_ctx {
  hpmc_params p;
  Geo g;
  int64_t N = 0;
  int ncell = 0;
  cudaStream_t stream = nullptr;
  bool own_pose = false;
  float4* d_pos = nullptr;
  float4* d_quat = nullptr;
  float4* d_cpos = nullptr;
  float4* d_caxis = nullptr;
  uint32_t *d_cid = nullptr, *d_rank = nullptr, *d_counts = nullptr, *d_cell_start = nullptr, *d_cell_pid = nullptr,
           *d_tile_sums = nullptr;
  int ntiles = 0;
  uint8_t* d_outcome = nullptr;
  unsigned long long* d_counters = nullptr;
  int* d_err = nullptr;
  float shift[3] = {0, 0, 0};
  bool built = false;
  uint32_t b_seed = 0, b_step = 0;
  std::vector<PoissonTable> tables;     // small cache keyed by lambda (C2 sweeps four densities)
  size_t table_rr = 0;
  int num_sms = 148;
  int move_ctas = 0;
  QPlan plan[2];                       // launch plans of the item-queue move kernel: [0] plain rule, [1] configurational bias
  uint32_t options = 0;                // hpmc_set_options
  // host-buffer path: accepted-particle list of the sweep in flight, packed poses, pinned staging (hpmc_step_host)
  uint32_t *d_acc_count = nullptr, *d_acc_list = nullptr, *h_acc_list = nullptr;
  float4 *d_acc_pack = nullptr, *h_acc_pack = nullptr;
  uint32_t* h_acc_count = nullptr;
  bool track_accepts = false;          // set by hpmc_step_host for the sweep it issues
  size_t acc_cap = 0;                  // entries the sparse download may carry (beyond: full copy)
  int64_t last_h2d = 0, last_d2h = 0;  // bytes of the last hpmc_step_host
  bool use_queue = true;               // HPMC_MOVE_KERNEL=warp selects the first (warp-per-cell) design
  int cb_kernel = 0;                   // configurational bias: 0 = choose per sweep (n_trial, N), 1 = warp-per-cell kernel, 2 = item-queue kernel (HPMC_CB_KERNEL=warp|queue)
  int64_t launches = 0;
#ifdef HPMC_PHASE_CLOCKS
  unsigned long long* d_phase_clk = nullptr;   // tuning build: per-phase clock sums of the move kernel (printed by hpmc_destroy)
  int64_t phase_ctas = 0;
#endif
  bool timing = false;
  std::vector<EventPair> ev;
  size_t ev_used = 0;
  double ev_ms = 0.0;
  int64_t ev_launches = 0;
  std::string err;
};

namespace {

int fail(hpmc_ctx* c, int code, const std::string& msg) {
  if (c) c->err = msg; else g_init_error = msg;
  return code;
}

#define CU(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess)                                                                         \
      return fail(ctx, HPMC_E_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));           \
  } while (0)

Geo make_geo(const hpmc_params& p, int nc) {
  Geo g;
  g.L = p.box_L; g.halfL = 0.5f * p.box_L; g.nc = nc; g.w = p.box_L / (float)nc;
  g.rd = 0.5f * p.sigma_d;
  g.Rins = 0.5f * (p.sigma_c + p.sigma_d);
  g.Rins2 = g.Rins * g.Rins;
  g.dcirc2 = p.sigma_c * p.sigma_c;
  const float rcut = ((p.sigma_c + p.sigma_d) + p.d_max_cap * 1.7320508f) + 1e-3f;
  g.rcut2 = rcut * rcut;
  g.Rh = 0.5f * p.sigma_c;
  g.cen = 0.375f * g.Rh;
  g.adisk = p.disk_a; g.sdisk = p.disk_s;
  const float rs = p.disk_s + g.rd;
  g.rs2 = rs * rs;
  g.rd2 = g.rd * g.rd;
  return g;
}

// Poisson thresholds T[j] = floor(CDF(k_lo + j) 2^64), saturating (R-S2); fp64 on the host.
void poisson_thresholds(double lambda, uint32_t& k_lo, std::vector<unsigned long long>& T) {
  T.clear(); k_lo = 0;
  if (!(lambda > 0.0)) return;
  const double sq = std::sqrt(lambda);
  long long lo = (long long)std::floor(lambda - 10.0 * sq - 10.0);
  if (lo < 0) lo = 0;
  const long long hi = (long long)std::ceil(lambda + 10.0 * sq + 20.0);
  const long long n = hi - lo + 1;
  long long m = (long long)std::floor(lambda);
  if (m < lo) m = lo;
  std::vector<double> pm((size_t)n);
  pm[(size_t)(m - lo)] = std::exp((double)m * std::log(lambda) - lambda - std::lgamma((double)m + 1.0));
  for (long long k = m; k < hi; ++k) pm[(size_t)(k + 1 - lo)] = pm[(size_t)(k - lo)] * lambda / (double)(k + 1);
  for (long long k = m; k > lo; --k) pm[(size_t)(k - 1 - lo)] = pm[(size_t)(k - lo)] * (double)k / lambda;
  double S = 0.0;
  for (long long j = 0; j < n; ++j) S += pm[(size_t)j];
  k_lo = (uint32_t)lo;
  T.resize((size_t)n);
  double c = 0.0;
  for (long long j = 0; j < n; ++j) {
    c += pm[(size_t)j] / S;
    T[(size_t)j] = (c >= 1.0) ? 0xFFFFFFFFFFFFFFFFull : (unsigned long long)std::floor(c * 18446744073709551616.0);
  }
}

int get_table(hpmc_ctx* ctx, double lambda, PoissonTable** out) {
  for (auto& t : ctx->tables)
    if (t.lambda == lambda) { *out = &t; return 0; }
  PoissonTable* slot;
  if (ctx->tables.size() < 8) { ctx->tables.emplace_back(); slot = &ctx->tables.back(); }
  else {
    // evicting a table that may still be read by queued kernels: drain the stream first
    CU(cudaStreamSynchronize(ctx->stream));
    slot = &ctx->tables[ctx->table_rr++ % ctx->tables.size()];
  }
  std::vector<unsigned long long> T;
  uint32_t klo;
  poisson_thresholds(lambda, klo, T);
  if (T.size() > slot->cap) {
    if (slot->d_T) { CU(cudaStreamSynchronize(ctx->stream)); CU(cudaFree(slot->d_T)); slot->d_T = nullptr; }
    slot->cap = T.size() + 64;
    CU(cudaMalloc(&slot->d_T, slot->cap * sizeof(unsigned long long)));
  }
  slot->has_guide = false;
  if (!T.empty()) {
    // pageable source: the runtime stages it before returning, so T may go out of scope
    CU(cudaMemcpyAsync(slot->d_T, T.data(), T.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice, ctx->stream));
    {
      // guide table: bucket b covers uniforms U with U >> 52 == b; {lo = #{j : T[j] < b 2^52}, n = thresholds inside
      // the bucket, T[lo] low word, T[lo] high word}
      std::vector<uint4> G(4096);
      size_t j = 0;
      for (unsigned i = 0; i < 4096; ++i) {
        const unsigned long long edge = (unsigned long long)i << 52;
        while (j < T.size() && T[j] < edge) ++j;
        size_t j2 = j;
        if (i == 4095) j2 = T.size();
        else { const unsigned long long e2 = (unsigned long long)(i + 1) << 52; while (j2 < T.size() && T[j2] < e2) ++j2; }
        const unsigned long long t0 = j < T.size() ? T[j] : ~0ull;
        G[i] = make_uint4((unsigned)j, (unsigned)(j2 - j), (unsigned)(t0 & 0xffffffffull), (unsigned)(t0 >> 32));
      }
      if (!slot->d_G) CU(cudaMalloc(&slot->d_G, 4096 * sizeof(uint4)));
      CU(cudaMemcpyAsync(slot->d_G, G.data(), 4096 * sizeof(uint4), cudaMemcpyHostToDevice, ctx->stream));
      slot->has_guide = true;
    }
    CU(cudaStreamSynchronize(ctx->stream));
  }
  slot->lambda = lambda; slot->k_lo = klo; slot->n = (int)T.size();
  *out = slot;
  return 0;
}

#ifndef HPMC_QCPT
#define HPMC_QCPT 2
#endif
#ifndef HPMC_QT
#define HPMC_QT 128
#endif
constexpr int QT = HPMC_QT;                // threads per CTA of the item-queue kernel
template <int SHAPE> struct QCfg { static constexpr int CPT = SHAPE == SH_SPHERE ? HPMC_QCPT : 1; };   // tile capacity CPT*QT cells

// tuning builds only (HPMC_PHASE_CLOCKS): HPMC_SMEM_PAD bytes of unused dynamic shared memory lower the number of
// resident CTAs per SM, to time a CTA's phases without its neighbours on the SM
inline size_t smem_pad() {
#ifdef HPMC_PHASE_CLOCKS
  if (const char* o = getenv("HPMC_SMEM_PAD")) return (size_t)atol(o);
#endif
  return 0;
}

template <int SHAPE, bool CB>
int setup_moveq(hpmc_ctx* ctx) {
  QPlan& P = ctx->plan[CB ? 1 : 0];
  using SM = QSmem<SHAPE, QT, QCfg<SHAPE>::CPT, CB>;
  const size_t smem = SM::bytes + smem_pad();
  cudaError_t e = cudaFuncSetAttribute(k_moveq<SHAPE, QT, QCfg<SHAPE>::CPT, CB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return fail(ctx, HPMC_E_CUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e));
  int per_sm = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_moveq<SHAPE, QT, QCfg<SHAPE>::CPT, CB>, QT, smem);
  if (e != cudaSuccess || per_sm < 1) return fail(ctx, HPMC_E_CUDA, "k_moveq does not fit on an SM");
  // one wave: every CTA of a pass is resident at once (a pass is latency-, not throughput-bound) and owns
  // cells_per_cta active cells, worked through in nsub tiles of equal size
  const int nact = ctx->ncell / 8;
  const int resident = ctx->num_sms * per_sm;
  int cpc = (nact + resident - 1) / resident;
  int pool_cap = 1 << 30;
  {
    // keep the expected number of listed neighbours of a tile within the shared-memory pool: ideal-gas estimate of
    // the neighbours inside the list radius from the MEAN density, times 2 (contact shell of a dense hard-particle
    // fluid or crystal), for every non-empty cell of the tile.  Only a performance heuristic: a tile that overflows
    // anyway (a cluster in a dilute box) is halved and redone inside the kernel
    const double L = ctx->p.box_L, dens = (double)ctx->N / (L * L * L);
    const double rl = CB ? std::sqrt((double)ctx->g.rcut2) : (double)ctx->p.sigma_c + ctx->p.sigma_d + 1e-3;
    const double nbr = 2.0 * dens * (4.0 * M_PI / 3.0) * rl * rl * rl + 1.0;
    const double occ = (double)ctx->N / (double)ctx->ncell;
    const double pmove = occ < 1.0 ? occ : 1.0;
    pool_cap = (int)((double)SM::POOL / (nbr * pmove));
    if (getenv("HPMC_POOL_CAP_OFF")) pool_cap = 1 << 30;      // tests: rely on the in-kernel tile splitting alone
    if (cpc > pool_cap) cpc = pool_cap;
  }
  if (cpc < 8) cpc = 8;   // small systems are latency-bound: more, smaller CTAs (measured on C1, C2, C4)
  if (const char* o = getenv("HPMC_CELLS_PER_CTA")) { const int v = atoi(o); if (v >= 1) cpc = v; }
  constexpr int QM = QCfg<SHAPE>::CPT * QT;
  // work ramp: only when the pass is one full wave (then every SM holds per_sm CTAs launched in index order)
  float ramp = 0.0f;
  {
    int dev = 0, coop = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    const char* sl = getenv("HPMC_SWEEP_LAUNCHES");
    P.one_launch = coop != 0 && !(sl && atoi(sl) == 8);
  }
  // (the ramp only pays when all CTAs start a pass together, i.e. with one launch per pass: measured at C3 in the
  // one-launch kernel 0.2 / 0.1 / 0 -> 505 / 482 / 475 us per sweep)
  if (!P.one_launch && (nact + cpc - 1) / cpc > resident / 2) {
    ramp = 0.2f;    // measured at C3: 0 / 0.1 / 0.15 / 0.2 -> 66.7 / 65.3 / 64.2 / 63.7 us per pass
    if (const char* o = getenv("HPMC_RAMP")) ramp = (float)atof(o);
    if (ramp < 0.0f) ramp = 0.0f;
    if (ramp > 0.5f) ramp = 0.5f;
  }
  if ((double)cpc * (1.0 + ramp) > (double)pool_cap) cpc = (int)((double)pool_cap / (1.0 + ramp));
  if (cpc < 8) cpc = 8;
  P.ramp = ramp;
  const int cmax = (int)std::ceil((double)cpc * (1.0 + ramp)) + 1;     // largest share of a CTA
  int nsub = (cmax + QM - 1) / QM;
  int big = (cmax + nsub - 1) / nsub;
  if (big > QM) big = QM;
  if (const char* o = getenv("HPMC_TILE_BIG")) { const int v = atoi(o); if (v >= 1 && v <= QM) big = v; }
  P.cpc = cpc; P.big = big;
  P.ctas = (nact + cpc - 1) / cpc;
  {
    // shares: CTA i owns [first(i), first(i+1)), first(i) = nact (x + ramp x (1 - x)), x = i / n: the first CTAs get
    // (1 + ramp) times the average share, the last ones (1 - ramp) times
    const int n = P.ctas;
    std::vector<uint32_t> first((size_t)n + 1);
    for (int i = 0; i <= n; ++i) {
      const double x = (double)i / (double)n;
      const double v = (double)nact * (x + (double)ramp * x * (1.0 - x));
      first[(size_t)i] = i >= n ? (uint32_t)nact : std::min((uint32_t)v, (uint32_t)nact);
    }
    cudaError_t e2 = cudaMalloc(&P.d_cta_first, sizeof(uint32_t) * ((size_t)n + 1));
    if (e2 == cudaSuccess) e2 = cudaMalloc(&P.d_done, sizeof(uint32_t) * (size_t)n);
    if (e2 == cudaSuccess) e2 = cudaMemcpy(P.d_cta_first, first.data(), sizeof(uint32_t) * ((size_t)n + 1), cudaMemcpyHostToDevice);
    if (e2 == cudaSuccess) e2 = cudaMemset(P.d_done, 0, sizeof(uint32_t) * (size_t)n);
    if (e2 != cudaSuccess) return fail(ctx, HPMC_E_CUDA, std::string("setup_moveq: ") + cudaGetErrorString(e2));
    // every CTA of the one-launch kernel must be resident at once (its CTAs wait for one another)
    P.one_launch = P.one_launch && n <= resident && n <= 32 * SM::NBMAP_WORDS;
  }
  if (getenv("HPMC_VERBOSE"))
    fprintf(stderr, "k_moveq<%d,%d,%s>: smem %zu B, %d CTAs/SM, %d CTAs x %d cells on average (ramp %.2f), tiles of %d, %s\n", SHAPE,
            QT, CB ? "cb" : "plain", smem, per_sm, P.ctas, cpc, (double)ramp, big, P.one_launch ? "one launch per sweep" : "one launch per pass");
  return 0;
}

template <int SHAPE, bool CB>
int launch_moveq(hpmc_ctx* ctx, const MoveArgs& a, const PoissonTable* pt, const uint32_t* perm8) {
  QPlan& P = ctx->plan[CB ? 1 : 0];
  using SM = QSmem<SHAPE, QT, QCfg<SHAPE>::CPT, CB>;
  QArgs q;
  q.m = a;
  q.cta_first = P.d_cta_first; q.done = P.d_done; q.seq0 = P.seq;
  q.npass = perm8 ? 8 : 1;
  for (int i = 0; i < 8; ++i) q.colours[i] = perm8 ? perm8[i] : 0u;
  q.magic_hc = ~0ull / (unsigned long long)a.hc + 1ull;   // floor((2^64-1)/hc)+1 == floor(2^64/hc)+1 unless hc | 2^64
  if ((a.hc & (a.hc - 1)) == 0) q.magic_hc = (1ull << 63) / (unsigned long long)a.hc * 2ull + 1ull;
  q.pguide = pt->has_guide ? pt->d_G : nullptr;
  q.ramp = P.ramp; q.tile_cells = P.big;
  q.wlo = 2.1f * a.g.w; q.whi = a.g.L - 2.1f * a.g.w;
#ifdef HPMC_PHASE_CLOCKS
  if (!ctx->d_phase_clk) { cudaMalloc(&ctx->d_phase_clk, 64); cudaMemsetAsync(ctx->d_phase_clk, 0, 64, ctx->stream); }
  q.phase_clk = ctx->d_phase_clk; ctx->phase_ctas += (int64_t)P.ctas * q.npass;
#endif
  {
    const float rl = (ctx->p.sigma_c + ctx->p.sigma_d) + 1e-3f;
    q.rlist2 = rl * rl;
    if (CB || q.rlist2 > a.g.rcut2) q.rlist2 = a.g.rcut2;      // CB also samples about the OLD centre: the full r_cut of R-3.4
  }
  if (perm8) {
    // cooperative launch: the runtime guarantees that all CTAs are resident, which the neighbour waits rely on
    void* args[] = {(void*)&q};
    const cudaError_t e = cudaLaunchCooperativeKernel((const void*)k_moveq<SHAPE, QT, QCfg<SHAPE>::CPT, CB>, dim3(P.ctas),
                                                      dim3(QT), args, SM::bytes + smem_pad(), ctx->stream);
    if (e != cudaSuccess) return fail(ctx, HPMC_E_CUDA, std::string("cudaLaunchCooperativeKernel: ") + cudaGetErrorString(e));
    P.seq += 8u;
    return 0;
  }
  k_moveq<SHAPE, QT, QCfg<SHAPE>::CPT, CB><<<P.ctas, QT, SM::bytes + smem_pad(), ctx->stream>>>(q);
  return 0;
}

template <int SHAPE>
int launch_move(hpmc_ctx* ctx, const MoveArgs& a, bool cb) {
  const dim3 grid(ctx->move_ctas), block(MOVE_WARPS * 32);
  if (cb) k_move<SHAPE, true><<<grid, block, 0, ctx->stream>>>(a);
  else k_move<SHAPE, false><<<grid, block, 0, ctx->stream>>>(a);
  return 0;
}

}  // namespace

extern "C" {

int hpmc_init(hpmc_ctx** out, const hpmc_params* p, int64_t N, float* d_pos4, float* d_quat4, void* cuda_stream) {
  hpmc_ctx* ctx = nullptr;
  if (!out || !p) return fail(nullptr, HPMC_E_BADARG, "hpmc_init: NULL argument");
  *out = nullptr;
  if (N <= 0 || N > 0x7fffffff) return fail(nullptr, HPMC_E_BADARG, "hpmc_init: N out of range");
  if (!(p->box_L > 0.0f) || !(p->sigma_c > 0.0f) || p->sigma_d < 0.0f || p->d_max_cap < 0.0f)
    return fail(nullptr, HPMC_E_BADARG, "hpmc_init: bad geometry parameters");
  if (p->shape < HPMC_SPHERE || p->shape > HPMC_TETRAHEDRON) return fail(nullptr, HPMC_E_BADARG, "hpmc_init: bad shape");
  if (p->shape == HPMC_ELLIPSOID) {
    // oblate spheroid (disk_a, disk_a, disk_s): sigma_c is the circumsphere diameter 2 disk_a
    if (!(p->disk_s > 0.0f) || !(p->disk_a >= p->disk_s) ||
        std::fabs((double)p->sigma_c - 2.0 * (double)p->disk_a) > 1e-5 * (double)p->sigma_c)
      return fail(nullptr, HPMC_E_BADARG, "hpmc_init: ellipsoid needs disk_a >= disk_s > 0 and sigma_c == 2 disk_a");
    // the depletant test finds the closest point of the ellipse with a FIXED six Newton steps (geometry.cuh): converged to
    // fp32 rounding for aspect ratios up to 4, off by up to 1e-4 of a diameter at 10
    if (p->disk_a > 4.0f * p->disk_s)
      return fail(nullptr, HPMC_E_BADARG, "hpmc_init: ellipsoid aspect ratio disk_a / disk_s above 4 is not supported");
  }
  if (p->shape == HPMC_SPHERODISK) {
    // sigma_c is the circumsphere diameter 2 (a + s): the insertion radius, the cell width and the list radius derive from it
    if (!(p->disk_a >= 0.0f) || !(p->disk_s >= 0.0f) || !(p->disk_a + p->disk_s > 0.0f) ||
        std::fabs((double)p->sigma_c - 2.0 * ((double)p->disk_a + (double)p->disk_s)) > 1e-5 * (double)p->sigma_c)
      return fail(nullptr, HPMC_E_BADARG, "hpmc_init: spherodisk needs disk_a, disk_s >= 0 and sigma_c == 2 (disk_a + disk_s)");
  }
  if (p->shape != HPMC_SPHERE && d_pos4 && !d_quat4)
    return fail(nullptr, HPMC_E_BADARG, "hpmc_init: anisotropic shape needs orientations");
  if (!d_pos4 && d_quat4) return fail(nullptr, HPMC_E_BADARG, "hpmc_init: d_quat4 without d_pos4");
  const double wmin = (double)p->sigma_c + (double)p->sigma_d + 2.0 * (double)p->d_max_cap;
  long long n = (long long)std::floor((double)p->box_L / wmin);
  n &= ~1ll;
  if (n < 4) return fail(nullptr, HPMC_E_GEOMETRY, "hpmc_init: fewer than 4 cells per axis");
  if (n > 1024) return fail(nullptr, HPMC_E_GEOMETRY, "hpmc_init: more than 1024 cells per axis");
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return fail(nullptr, HPMC_E_CUDA, std::string("hpmc_init: no usable CUDA device: ") + cudaGetErrorString(cudaGetLastError()));

  ctx = new hpmc_ctx();
  ctx->p = *p; ctx->N = N; ctx->stream = (cudaStream_t)cuda_stream; ctx->num_sms = sms;
  ctx->g = make_geo(*p, (int)n);
  ctx->ncell = (int)(n * n * n);
  ctx->ntiles = (ctx->ncell + SCAN_TILE - 1) / SCAN_TILE;
  auto bail = [&](const std::string& m) { g_init_error = m; hpmc_destroy(ctx); return HPMC_E_CUDA; };
#define CUI(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return bail(std::string(#call) + ": " + cudaGetErrorString(e_)); } while (0)
  if (!d_pos4) {
    ctx->own_pose = true;
    CUI(cudaMalloc(&ctx->d_pos, sizeof(float4) * N));
    CUI(cudaMalloc(&ctx->d_quat, sizeof(float4) * N));
    CUI(cudaMemsetAsync(ctx->d_pos, 0, sizeof(float4) * N, ctx->stream));
    CUI(cudaMemsetAsync(ctx->d_quat, 0, sizeof(float4) * N, ctx->stream));
  } else {
    ctx->d_pos = (float4*)d_pos4; ctx->d_quat = (float4*)d_quat4;
  }
  CUI(cudaMalloc(&ctx->d_cpos, sizeof(float4) * N));
  if (p->shape != HPMC_SPHERE) CUI(cudaMalloc(&ctx->d_caxis, sizeof(float4) * N));
  CUI(cudaMalloc(&ctx->d_cid, sizeof(uint32_t) * N));
  CUI(cudaMalloc(&ctx->d_rank, sizeof(uint32_t) * N));
  CUI(cudaMalloc(&ctx->d_cell_pid, sizeof(uint32_t) * N));
  // counts and cell_start are padded to whole scan tiles (+ one tile for cell_start[ncell]): the scan kernels move uint4
  const size_t padded = (size_t)ctx->ntiles * SCAN_TILE;
  CUI(cudaMalloc(&ctx->d_counts, sizeof(uint32_t) * padded));
  CUI(cudaMalloc(&ctx->d_cell_start, sizeof(uint32_t) * (padded + SCAN_TILE)));
  CUI(cudaMalloc(&ctx->d_tile_sums, sizeof(uint32_t) * (size_t)ctx->ntiles));
  CUI(cudaMalloc(&ctx->d_outcome, (size_t)N));
  CUI(cudaMalloc(&ctx->d_counters, sizeof(unsigned long long) * (C_COUNT + 1)));   // + 1: the tally of hpmc_free_volume
  CUI(cudaMalloc(&ctx->d_err, sizeof(int)));
  CUI(cudaMemsetAsync(ctx->d_outcome, 0, (size_t)N, ctx->stream));
  CUI(cudaMemsetAsync(ctx->d_counts, 0, sizeof(uint32_t) * padded, ctx->stream));   // kept zero between builds by k_scan_apply
  CUI(cudaMemsetAsync(ctx->d_counters, 0, sizeof(unsigned long long) * C_COUNT, ctx->stream));
  CUI(cudaMemsetAsync(ctx->d_err, 0, sizeof(int), ctx->stream));
#undef CUI
  // persistent warps: a whole number of CTAs per SM, capped by the work available
  const int nact = ctx->ncell / 8;
  int ctas = sms * 8;
  const int need = (nact + MOVE_WARPS - 1) / MOVE_WARPS;
  if (ctas > need) ctas = need;
  if (ctas < 1) ctas = 1;
  ctx->move_ctas = ctas;
  {
    const char* sel = getenv("HPMC_MOVE_KERNEL");
    ctx->use_queue = !(sel && std::string(sel) == "warp");
    // Configurational bias: two kernels, same bits, both covered by the parity tests.  Measured on spherodisks
    // (profiles/r2_cb_kernels.md): the warp-per-cell kernel wins for few reinsertions on small systems (n_trial = 4,
    // 32,768 particles: 252 against 480 us per sweep), the item-queue kernel, which spreads the 2 n_trial reinsertions of
    // every rejecting depletant over the whole CTA, from n_trial ~ 16 on (n_trial = 40: 1.6 against 2.2 ms; 100: 3.3
    // against 4.8 ms) and on large systems (262,144 particles: 813 against 830 us at n_trial = 4).
    const char* cbk = getenv("HPMC_CB_KERNEL");
    ctx->cb_kernel = (cbk && std::string(cbk) == "queue") ? 2 : ((cbk && std::string(cbk) == "warp") ? 1 : 0);
    int rc = 0;
    switch (p->shape) {
      case HPMC_SPHERE: rc = setup_moveq<SH_SPHERE, false>(ctx); if (!rc) rc = setup_moveq<SH_SPHERE, true>(ctx); break;
      case HPMC_HALFBALL: rc = setup_moveq<SH_HALFBALL, false>(ctx); if (!rc) rc = setup_moveq<SH_HALFBALL, true>(ctx); break;
      case HPMC_SPHERODISK: rc = setup_moveq<SH_SPHERODISK, false>(ctx); if (!rc) rc = setup_moveq<SH_SPHERODISK, true>(ctx); break;
      case HPMC_ELLIPSOID: rc = setup_moveq<SH_ELLIPSOID, false>(ctx); if (!rc) rc = setup_moveq<SH_ELLIPSOID, true>(ctx); break;
      default: rc = setup_moveq<SH_TETRAHEDRON, false>(ctx); if (!rc) rc = setup_moveq<SH_TETRAHEDRON, true>(ctx); break;
    }
    if (rc) { g_init_error = ctx->err; hpmc_destroy(ctx); return rc; }
  }
  *out = ctx;
  return HPMC_OK;
}

void hpmc_destroy(hpmc_ctx* ctx) {
  if (!ctx) return;
  cudaStreamSynchronize(ctx->stream);
#ifdef HPMC_PHASE_CLOCKS
  if (ctx->d_phase_clk) {
    unsigned long long h[8], tr[2] = {0, 0};
    cudaMemcpy(h, ctx->d_phase_clk, 64, cudaMemcpyDeviceToHost);
    cudaMemcpyFromSymbol(tr, g_dbg_trips, sizeof(tr));
    static const char* nm[8] = {"setup", "1a", "wait", "1b+1c", "1d", "2", "commit", "-"};
    fprintf(stderr, "phase clocks per CTA and pass (thread 0):");
    for (int i = 0; i < 7; ++i) fprintf(stderr, " %s %.0f", nm[i], (double)h[i] / (double)std::max<int64_t>(1, ctx->phase_ctas));
    fprintf(stderr, "; phase 2: %.2f loop trips per tile\n", (double)tr[0] / (double)std::max(1ull, tr[1]));
    cudaFree(ctx->d_phase_clk);
  }
#endif
  if (ctx->own_pose) { cudaFree(ctx->d_pos); cudaFree(ctx->d_quat); }
  cudaFree(ctx->d_cpos); cudaFree(ctx->d_caxis); cudaFree(ctx->d_cid); cudaFree(ctx->d_rank);
  cudaFree(ctx->d_cell_pid); cudaFree(ctx->d_counts); cudaFree(ctx->d_cell_start); cudaFree(ctx->d_tile_sums);
  cudaFree(ctx->d_outcome); cudaFree(ctx->d_counters); cudaFree(ctx->d_err);
  cudaFree(ctx->d_acc_count); cudaFree(ctx->d_acc_list); cudaFree(ctx->d_acc_pack);
  if (ctx->h_acc_list) cudaFreeHost(ctx->h_acc_list);
  if (ctx->h_acc_pack) cudaFreeHost(ctx->h_acc_pack);
  if (ctx->h_acc_count) cudaFreeHost(ctx->h_acc_count);
  for (auto& pl : ctx->plan) { cudaFree(pl.d_cta_first); cudaFree(pl.d_done); }
  for (auto& t : ctx->tables) { cudaFree(t.d_T); cudaFree(t.d_G); }
  for (auto& e : ctx->ev) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  delete ctx;
}

int hpmc_build_cells(hpmc_ctx* ctx, uint32_t seed, uint32_t step) {
  if (!ctx) return HPMC_E_BADARG;
  const Key10 key = make_key(seed, step);
  const Block4 r = philox(key, 0, 0, 0, ctr_word3(P_SWEEP, 0, 0));
  ctx->shift[0] = unit01(r.x) * ctx->g.w;
  ctx->shift[1] = unit01(r.y) * ctx->g.w;
  ctx->shift[2] = unit01(r.z) * ctx->g.w;
  const int N = (int)ctx->N, nb = (N + 255) / 256;
  cudaStream_t st = ctx->stream;
  // d_counts is zero here: hpmc_init clears it once and k_scan_apply re-zeroes it after its last read
  k_bin_count<<<nb, 256, 0, st>>>(ctx->d_pos, N, ctx->g, ctx->shift[0], ctx->shift[1], ctx->shift[2], ctx->d_cid,
                                  ctx->d_rank, ctx->d_counts, ctx->d_outcome);
  k_scan_tiles<<<ctx->ntiles, SCAN_THREADS, 0, st>>>(ctx->d_counts, ctx->ncell, ctx->d_tile_sums);
  if (ctx->ntiles <= 4096) {
    k_scan_apply<true><<<ctx->ntiles, SCAN_THREADS, 0, st>>>(ctx->d_counts, ctx->ncell, ctx->d_tile_sums, ctx->d_cell_start);
    ctx->launches += 5;
  } else {
    k_scan_top<<<1, 1024, 0, st>>>(ctx->d_tile_sums, ctx->ntiles);
    k_scan_apply<false><<<ctx->ntiles, SCAN_THREADS, 0, st>>>(ctx->d_counts, ctx->ncell, ctx->d_tile_sums, ctx->d_cell_start);
    ctx->launches += 6;
  }
  k_fill<<<nb, 256, 0, st>>>(ctx->d_cid, ctx->d_rank, ctx->d_cell_start, N, ctx->d_cell_pid);
  const int cbk = (ctx->ncell + 255) / 256;
  if (ctx->p.shape == HPMC_SPHERE)
    k_sort_write<SH_SPHERE><<<cbk, 256, 0, st>>>(ctx->d_cell_start, ctx->ncell, ctx->d_cell_pid, ctx->d_pos, ctx->d_quat,
                                                 ctx->d_cpos, ctx->d_caxis);
  else if (ctx->p.shape == HPMC_TETRAHEDRON)       // cell-ordered orientation = the quaternion itself
    k_sort_write<SH_TETRAHEDRON><<<cbk, 256, 0, st>>>(ctx->d_cell_start, ctx->ncell, ctx->d_cell_pid, ctx->d_pos, ctx->d_quat,
                                                      ctx->d_cpos, ctx->d_caxis);
  else                                             // bodies of revolution: the body z axis
    k_sort_write<SH_HALFBALL><<<cbk, 256, 0, st>>>(ctx->d_cell_start, ctx->ncell, ctx->d_cell_pid, ctx->d_pos, ctx->d_quat,
                                                   ctx->d_cpos, ctx->d_caxis);
  CU(cudaGetLastError());
  ctx->built = true; ctx->b_seed = seed; ctx->b_step = step;
  return HPMC_OK;
}

int hpmc_sweep(hpmc_ctx* ctx, uint32_t seed, uint32_t step, double n_R, float d_max, float a_max, int32_t n_trial) {
  if (!ctx) return HPMC_E_BADARG;
  if (!(d_max >= 0.0f) || !(n_R >= 0.0) || !(a_max >= 0.0f) || n_trial < 0 || n_trial > 65535)
    return fail(ctx, HPMC_E_BADARG, "hpmc_sweep: bad argument");
  if (d_max > ctx->p.d_max_cap) return fail(ctx, HPMC_E_DMAX, "hpmc_sweep: d_max exceeds d_max_cap");
  if (!ctx->built || ctx->b_seed != seed || ctx->b_step != step)
    return fail(ctx, HPMC_E_STATE, "hpmc_sweep: call hpmc_build_cells(seed, step) first");
  const double Rd = (double)ctx->g.Rins;
  double lambda = n_R * ((4.0 * M_PI / 3.0) * (Rd * Rd * Rd));
  // HPMC_OPT_SHELL (R-N1, L158): R_in = max(0, r_in - sqrt(3) d_max), r_in = inradius of the dilated shape about its centre
  float sh_Rin = 0.0f;
  if (ctx->options & HPMC_OPT_SHELL) {
    float rin = ctx->g.Rins;
    if (ctx->p.shape == HPMC_HALFBALL) rin = ctx->g.rd;
    else if (ctx->p.shape == HPMC_SPHERODISK || ctx->p.shape == HPMC_ELLIPSOID) rin = ctx->g.sdisk + ctx->g.rd;
    else if (ctx->p.shape == HPMC_TETRAHEDRON) rin = ctx->g.Rh * 0.33333334f + ctx->g.rd;
    sh_Rin = rin - 1.7320508f * d_max;
    if (sh_Rin < 0.0f) sh_Rin = 0.0f;
    const double Ri = (double)sh_Rin;
    lambda = n_R * ((4.0 * M_PI / 3.0) * (Rd * Rd * Rd - Ri * Ri * Ri));
  }
  PoissonTable* pt = nullptr;
  const int rc = get_table(ctx, lambda, &pt);
  if (rc) return rc;

  const Key10 key = make_key(seed, step);
  // colour permutation (R-2): Fisher-Yates from SWEEP blocks 1 and 2
  uint32_t perm[8] = {0, 1, 2, 3, 4, 5, 6, 7};
  const Block4 b1 = philox(key, 0, 0, 0, ctr_word3(P_SWEEP, 0, 1));
  const Block4 b2 = philox(key, 0, 0, 0, ctr_word3(P_SWEEP, 0, 2));
  const uint32_t wds[7] = {b1.x, b1.y, b1.z, b1.w, b2.x, b2.y, b2.z};
  for (int i = 7, j = 0; i >= 1; --i, ++j) {
    const uint32_t r = (uint32_t)(((uint64_t)wds[j] * (uint32_t)(i + 1)) >> 32);
    const uint32_t t = perm[i]; perm[i] = perm[r]; perm[r] = t;
  }

  MoveArgs a;
  a.g = ctx->g; a.key = key;
  a.sx = ctx->shift[0]; a.sy = ctx->shift[1]; a.sz = ctx->shift[2];
  a.hc = ctx->g.nc / 2; a.nact = a.hc * a.hc * a.hc;
  a.d_max = d_max; a.a_max = a_max; a.a_max2 = a_max * a_max; a.n_trial = n_trial;
  a.pos = ctx->d_pos; a.quat = ctx->d_quat; a.cpos = ctx->d_cpos; a.caxis = ctx->d_caxis;
  a.cell_start = ctx->d_cell_start;
  a.ptable = pt->d_T; a.pt_n = pt->n; a.pt_klo = pt->k_lo;
  a.outcome = ctx->d_outcome; a.counters = ctx->d_counters; a.err_flag = ctx->d_err;
  a.options = ctx->options;
  a.acc_count = ctx->track_accepts ? ctx->d_acc_count : nullptr;
  a.acc_list = ctx->track_accepts ? ctx->d_acc_list : nullptr;
  a.sh_Rin3 = (sh_Rin * sh_Rin) * sh_Rin;
  a.sh_dR3 = (ctx->g.Rins * ctx->g.Rins) * ctx->g.Rins - a.sh_Rin3;
  const bool cb = n_trial > 0;
  // timing: ONE event pair around the 8 launches of the sweep (an event pair per launch costs more than the gaps
  // between the launches it would exclude); hpmc_move_kernel_ms counts 8 launches per pair
  EventPair* ep = nullptr;
  if (ctx->timing) {
    if (ctx->ev_used == ctx->ev.size()) {
      EventPair e;
      CU(cudaEventCreate(&e.a)); CU(cudaEventCreate(&e.b));
      ctx->ev.push_back(e);
    }
    ep = &ctx->ev[ctx->ev_used++];
    CU(cudaEventRecord(ep->a, ctx->stream));
  }
  int nlaunch = 8;
  const bool cb_queue = ctx->cb_kernel == 2 || (ctx->cb_kernel == 0 && (n_trial >= 16 || ctx->N >= 200000));
  if (ctx->use_queue && (!cb || cb_queue)) {
    // item-queue kernel (moveq.cuh): one cooperative launch for the 8 passes (CTAs synchronise with their spatial
    // neighbours only), or one launch per pass
    const bool one = ctx->plan[cb ? 1 : 0].one_launch;
    for (int pass = 0; pass < (one ? 1 : 8); ++pass) {
      a.colour = perm[pass];
      const uint32_t* p8 = one ? perm : nullptr;
      int rc2 = 0;
      switch (ctx->p.shape) {
        case HPMC_SPHERE: rc2 = cb ? launch_moveq<SH_SPHERE, true>(ctx, a, pt, p8) : launch_moveq<SH_SPHERE, false>(ctx, a, pt, p8); break;
        case HPMC_HALFBALL: rc2 = cb ? launch_moveq<SH_HALFBALL, true>(ctx, a, pt, p8) : launch_moveq<SH_HALFBALL, false>(ctx, a, pt, p8); break;
        case HPMC_SPHERODISK: rc2 = cb ? launch_moveq<SH_SPHERODISK, true>(ctx, a, pt, p8) : launch_moveq<SH_SPHERODISK, false>(ctx, a, pt, p8); break;
        case HPMC_ELLIPSOID: rc2 = cb ? launch_moveq<SH_ELLIPSOID, true>(ctx, a, pt, p8) : launch_moveq<SH_ELLIPSOID, false>(ctx, a, pt, p8); break;
        default: rc2 = cb ? launch_moveq<SH_TETRAHEDRON, true>(ctx, a, pt, p8) : launch_moveq<SH_TETRAHEDRON, false>(ctx, a, pt, p8); break;
      }
      if (rc2) { if (ep) --ctx->ev_used; return rc2; }    // no half-recorded event pair for hpmc_move_kernel_ms
    }
    if (one) nlaunch = 1;
  } else {
    // first design (move.cuh, HPMC_MOVE_KERNEL=warp): one warp per active cell, one launch per pass
    for (int pass = 0; pass < 8; ++pass) {
      a.colour = perm[pass];
      switch (ctx->p.shape) {
        case HPMC_SPHERE: launch_move<SH_SPHERE>(ctx, a, cb); break;
        case HPMC_HALFBALL: launch_move<SH_HALFBALL>(ctx, a, cb); break;
        case HPMC_SPHERODISK: launch_move<SH_SPHERODISK>(ctx, a, cb); break;
        case HPMC_ELLIPSOID: launch_move<SH_ELLIPSOID>(ctx, a, cb); break;
        default: launch_move<SH_TETRAHEDRON>(ctx, a, cb); break;
      }
    }
  }
  if (ep) {
    const cudaError_t eb = cudaEventRecord(ep->b, ctx->stream);
    if (eb != cudaSuccess) { --ctx->ev_used; return fail(ctx, HPMC_E_CUDA, std::string("cudaEventRecord: ") + cudaGetErrorString(eb)); }
    ep->n = nlaunch;
  }
  ctx->launches += nlaunch;
  CU(cudaGetLastError());
  ctx->built = false;
  return HPMC_OK;
}

int hpmc_free_volume(hpmc_ctx* ctx, uint32_t seed, uint32_t step, int64_t n_samples, uint64_t* host_free_count) {
  if (!ctx || !host_free_count || n_samples < 0) return HPMC_E_BADARG;
  if (!ctx->built || ctx->b_seed != seed || ctx->b_step != step)
    return fail(ctx, HPMC_E_STATE, "hpmc_free_volume: call hpmc_build_cells(seed, step) first");
  // the tally lives behind the context's counters: no allocation per measurement, and no cudaFree (which waits for the
  // whole device)
  unsigned long long* d_cnt = ctx->d_counters + C_COUNT;
  CU(cudaMemsetAsync(d_cnt, 0, sizeof(unsigned long long), ctx->stream));
  if (n_samples > 0) {
    const Key10 key = make_key(seed, step);
    long long blocks = (n_samples + 255) / 256;
    const long long cap = (long long)ctx->num_sms * 16;
    if (blocks > cap) blocks = cap;
    const dim3 grid((unsigned)blocks);
    switch (ctx->p.shape) {
      case HPMC_SPHERE: k_free_volume<SH_SPHERE><<<grid, 256, 0, ctx->stream>>>(ctx->g, key, ctx->shift[0], ctx->shift[1], ctx->shift[2], n_samples, ctx->d_cpos, ctx->d_caxis, ctx->d_cell_start, d_cnt); break;
      case HPMC_HALFBALL: k_free_volume<SH_HALFBALL><<<grid, 256, 0, ctx->stream>>>(ctx->g, key, ctx->shift[0], ctx->shift[1], ctx->shift[2], n_samples, ctx->d_cpos, ctx->d_caxis, ctx->d_cell_start, d_cnt); break;
      case HPMC_SPHERODISK: k_free_volume<SH_SPHERODISK><<<grid, 256, 0, ctx->stream>>>(ctx->g, key, ctx->shift[0], ctx->shift[1], ctx->shift[2], n_samples, ctx->d_cpos, ctx->d_caxis, ctx->d_cell_start, d_cnt); break;
      case HPMC_ELLIPSOID: k_free_volume<SH_ELLIPSOID><<<grid, 256, 0, ctx->stream>>>(ctx->g, key, ctx->shift[0], ctx->shift[1], ctx->shift[2], n_samples, ctx->d_cpos, ctx->d_caxis, ctx->d_cell_start, d_cnt); break;
      default: k_free_volume<SH_TETRAHEDRON><<<grid, 256, 0, ctx->stream>>>(ctx->g, key, ctx->shift[0], ctx->shift[1], ctx->shift[2], n_samples, ctx->d_cpos, ctx->d_caxis, ctx->d_cell_start, d_cnt); break;
    }
    ctx->launches += 1;
  }
  unsigned long long h = 0;
  CU(cudaMemcpyAsync(&h, d_cnt, sizeof(h), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  CU(cudaGetLastError());
  *host_free_count = (uint64_t)h;
  return HPMC_OK;
}

int hpmc_set_options(hpmc_ctx* ctx, uint32_t options) {
  if (!ctx) return HPMC_E_BADARG;
  if (options & ~(uint32_t)(HPMC_OPT_SHELL | HPMC_OPT_ROSENBLUTH)) return fail(ctx, HPMC_E_BADARG, "hpmc_set_options: unknown option bit");
  ctx->options = options;
  return HPMC_OK;
}

int hpmc_run(hpmc_ctx* ctx, uint32_t seed, uint32_t step0, int64_t n_sweeps, double n_R, float d_max, float a_max,
             int32_t n_trial) {
  for (int64_t s = 0; s < n_sweeps; ++s) {
    int rc = hpmc_build_cells(ctx, seed, step0 + (uint32_t)s);
    if (rc) return rc;
    rc = hpmc_sweep(ctx, seed, step0 + (uint32_t)s, n_R, d_max, a_max, n_trial);
    if (rc) return rc;
  }
  return HPMC_OK;
}

static int check_err_flag(hpmc_ctx* ctx) {
  int e = 0;
  CU(cudaMemcpyAsync(&e, ctx->d_err, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  if (e == 2) {
    CU(cudaMemsetAsync(ctx->d_err, 0, sizeof(int), ctx->stream));
    return fail(ctx, HPMC_E_CUDA, "move kernel: a CTA waited longer than the wall-clock limit (60 s in the default build) for a "
                                  "neighbouring CTA's pass and abandoned the sweep without committing its remaining moves "
                                  "(poses and counters of that sweep are invalid)");
  }
  if (e) {
    CU(cudaMemsetAsync(ctx->d_err, 0, sizeof(int), ctx->stream));
    return fail(ctx, HPMC_E_NEIGHBOR_OVERFLOW, "move kernel: one move has more neighbours inside the list radius than the "
                                               "shared-memory pool (item-queue kernel) or MAXNB = 64 (warp kernel) holds");
  }
  return HPMC_OK;
}

int hpmc_counters(hpmc_ctx* ctx, hpmc_counters_t* host_out) {
  if (!ctx || !host_out) return HPMC_E_BADARG;
  static_assert(sizeof(hpmc_counters_t) == sizeof(unsigned long long) * C_COUNT, "counter layout");
  CU(cudaMemcpyAsync(host_out, ctx->d_counters, sizeof(hpmc_counters_t), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  return check_err_flag(ctx);
}

int hpmc_reset_counters(hpmc_ctx* ctx) {
  if (!ctx) return HPMC_E_BADARG;
  CU(cudaMemsetAsync(ctx->d_counters, 0, sizeof(unsigned long long) * C_COUNT, ctx->stream));
  return HPMC_OK;
}

int hpmc_outcomes(hpmc_ctx* ctx, uint8_t* d_outcome) {
  if (!ctx || !d_outcome) return HPMC_E_BADARG;
  CU(cudaMemcpyAsync(d_outcome, ctx->d_outcome, (size_t)ctx->N, cudaMemcpyDeviceToDevice, ctx->stream));
  return HPMC_OK;
}

int hpmc_grid(hpmc_ctx* ctx, int32_t* n_c, float* w) {
  if (!ctx || !n_c || !w) return HPMC_E_BADARG;
  *n_c = ctx->g.nc; *w = ctx->g.w;
  return HPMC_OK;
}

int hpmc_cells(hpmc_ctx* ctx, uint32_t* d_cell_start, uint32_t* d_cell_pid, float* host_shift3) {
  if (!ctx || !d_cell_start || !d_cell_pid || !host_shift3) return HPMC_E_BADARG;
  CU(cudaMemcpyAsync(d_cell_start, ctx->d_cell_start, sizeof(uint32_t) * ((size_t)ctx->ncell + 1),
                     cudaMemcpyDeviceToDevice, ctx->stream));
  CU(cudaMemcpyAsync(d_cell_pid, ctx->d_cell_pid, sizeof(uint32_t) * (size_t)ctx->N, cudaMemcpyDeviceToDevice,
                     ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  for (int a = 0; a < 3; ++a) host_shift3[a] = ctx->shift[a];
  return HPMC_OK;
}

int hpmc_upload(hpmc_ctx* ctx, const float* host_pos4, const float* host_quat4) {
  if (!ctx || !host_pos4) return HPMC_E_BADARG;
  CU(cudaMemcpyAsync(ctx->d_pos, host_pos4, sizeof(float4) * ctx->N, cudaMemcpyHostToDevice, ctx->stream));
  if (host_quat4 && ctx->d_quat)
    CU(cudaMemcpyAsync(ctx->d_quat, host_quat4, sizeof(float4) * ctx->N, cudaMemcpyHostToDevice, ctx->stream));
  return HPMC_OK;
}

int hpmc_download(hpmc_ctx* ctx, float* host_pos4, float* host_quat4, uint8_t* host_outcome) {
  if (!ctx) return HPMC_E_BADARG;
  if (host_pos4) CU(cudaMemcpyAsync(host_pos4, ctx->d_pos, sizeof(float4) * ctx->N, cudaMemcpyDeviceToHost, ctx->stream));
  if (host_quat4 && ctx->d_quat)
    CU(cudaMemcpyAsync(host_quat4, ctx->d_quat, sizeof(float4) * ctx->N, cudaMemcpyDeviceToHost, ctx->stream));
  if (host_outcome) CU(cudaMemcpyAsync(host_outcome, ctx->d_outcome, (size_t)ctx->N, cudaMemcpyDeviceToHost, ctx->stream));
  return HPMC_OK;
}

int hpmc_step_host(hpmc_ctx* ctx, float* host_pos4, float* host_quat4, uint8_t* host_outcome, uint32_t seed,
                   uint32_t step, double n_R, float d_max, float a_max, int32_t n_trial) {
  if (!ctx || !host_pos4) return HPMC_E_BADARG;
  const int64_t N = ctx->N;
  const bool has_q = host_quat4 && ctx->d_quat;
  const size_t per = sizeof(float4) * (has_q ? 2 : 1);
  if (!ctx->d_acc_list) {
    // sparse download: the device keeps the list of the particles accepted in the sweep; if it is short, only their
    // poses come back and are patched into the host arrays (which hold the uploaded poses of all the others)
    ctx->acc_cap = (size_t)std::max<int64_t>(1, N / 4);
    // all six or none: a failure half-way (the pinned buffers are the likely ones) must not leave d_acc_list set,
    // or the next call would skip this block and use the missing ones
    cudaError_t ea = cudaMalloc(&ctx->d_acc_count, sizeof(uint32_t));
    if (ea == cudaSuccess) ea = cudaMalloc(&ctx->d_acc_pack, sizeof(float4) * 2 * ctx->acc_cap);
    if (ea == cudaSuccess) ea = cudaMallocHost(&ctx->h_acc_list, sizeof(uint32_t) * ctx->acc_cap);
    if (ea == cudaSuccess) ea = cudaMallocHost(&ctx->h_acc_pack, sizeof(float4) * 2 * ctx->acc_cap);
    if (ea == cudaSuccess) ea = cudaMallocHost(&ctx->h_acc_count, sizeof(uint32_t));
    if (ea == cudaSuccess) ea = cudaMalloc(&ctx->d_acc_list, sizeof(uint32_t) * (size_t)N);
    if (ea != cudaSuccess) {
      cudaFree(ctx->d_acc_count); cudaFree(ctx->d_acc_pack); cudaFree(ctx->d_acc_list);
      if (ctx->h_acc_list) cudaFreeHost(ctx->h_acc_list);
      if (ctx->h_acc_pack) cudaFreeHost(ctx->h_acc_pack);
      if (ctx->h_acc_count) cudaFreeHost(ctx->h_acc_count);
      ctx->d_acc_count = ctx->d_acc_list = ctx->h_acc_list = ctx->h_acc_count = nullptr;
      ctx->d_acc_pack = ctx->h_acc_pack = nullptr;
      cudaGetLastError();
      return fail(ctx, HPMC_E_CUDA, std::string("hpmc_step_host: staging buffers: ") + cudaGetErrorString(ea));
    }
  }
  int rc = hpmc_upload(ctx, host_pos4, host_quat4);
  if (rc) return rc;
  CU(cudaMemsetAsync(ctx->d_acc_count, 0, sizeof(uint32_t), ctx->stream));
  rc = hpmc_build_cells(ctx, seed, step);
  if (rc) return rc;
  ctx->track_accepts = true;
  rc = hpmc_sweep(ctx, seed, step, n_R, d_max, a_max, n_trial);
  ctx->track_accepts = false;
  if (rc) return rc;
  ctx->last_h2d = (int64_t)(sizeof(float4) * N * (has_q ? 2 : 1));
  ctx->last_d2h = 0;
  if (host_outcome) {
    CU(cudaMemcpyAsync(host_outcome, ctx->d_outcome, (size_t)N, cudaMemcpyDeviceToHost, ctx->stream));
    ctx->last_d2h += N;
  }
  CU(cudaMemcpyAsync(ctx->h_acc_count, ctx->d_acc_count, sizeof(uint32_t), cudaMemcpyDeviceToHost, ctx->stream));
  CU(cudaStreamSynchronize(ctx->stream));
  const uint32_t n = *ctx->h_acc_count;
  ctx->last_d2h += 4;
  if ((size_t)n <= ctx->acc_cap) {
    if (n > 0) {
      k_gather_accepted<<<(n + 255) / 256, 256, 0, ctx->stream>>>(ctx->d_acc_list, n, ctx->d_pos, has_q ? ctx->d_quat : nullptr,
                                                                  ctx->d_acc_pack);
      ctx->launches += 1;
      CU(cudaMemcpyAsync(ctx->h_acc_list, ctx->d_acc_list, sizeof(uint32_t) * n, cudaMemcpyDeviceToHost, ctx->stream));
      CU(cudaMemcpyAsync(ctx->h_acc_pack, ctx->d_acc_pack, per * n, cudaMemcpyDeviceToHost, ctx->stream));
      CU(cudaStreamSynchronize(ctx->stream));
      float4* hp4 = reinterpret_cast<float4*>(host_pos4);
      float4* hq4 = reinterpret_cast<float4*>(host_quat4);
      for (uint32_t i = 0; i < n; ++i) {
        const uint32_t pid = ctx->h_acc_list[i];
        hp4[pid] = ctx->h_acc_pack[i];
        if (has_q) hq4[pid] = ctx->h_acc_pack[(size_t)n + i];
      }
      ctx->last_d2h += (int64_t)((sizeof(uint32_t) + per) * n);
    }
  } else {
    rc = hpmc_download(ctx, host_pos4, host_quat4, nullptr);
    if (rc) return rc;
    ctx->last_d2h += (int64_t)(per * N);
  }
  return check_err_flag(ctx);
}

int hpmc_step_host_bytes(hpmc_ctx* ctx, int64_t* h2d_bytes, int64_t* d2h_bytes) {
  if (!ctx || !h2d_bytes || !d2h_bytes) return HPMC_E_BADARG;
  *h2d_bytes = ctx->last_h2d; *d2h_bytes = ctx->last_d2h;
  return HPMC_OK;
}

int64_t hpmc_launch_count(hpmc_ctx* ctx) { return ctx ? ctx->launches : 0; }

int hpmc_time_move_kernel(hpmc_ctx* ctx, int32_t enable) {
  if (!ctx) return HPMC_E_BADARG;
  CU(cudaStreamSynchronize(ctx->stream));
  ctx->timing = enable != 0;
  ctx->ev_used = 0; ctx->ev_ms = 0.0; ctx->ev_launches = 0;
  return HPMC_OK;
}

int hpmc_move_kernel_ms(hpmc_ctx* ctx, double* ms_total, int64_t* launches) {
  if (!ctx || !ms_total || !launches) return HPMC_E_BADARG;
  CU(cudaStreamSynchronize(ctx->stream));
  for (size_t i = 0; i < ctx->ev_used; ++i) {
    float ms = 0.0f;
    CU(cudaEventElapsedTime(&ms, ctx->ev[i].a, ctx->ev[i].b));
    ctx->ev_ms += ms;
  }
  for (size_t i = 0; i < ctx->ev_used; ++i) ctx->ev_launches += ctx->ev[i].n;
  ctx->ev_used = 0;
  *ms_total = ctx->ev_ms; *launches = ctx->ev_launches;
  return HPMC_OK;
}

int hpmc_alu_peaks(hpmc_alu_peaks_t* out, void* cuda_stream) {
  hpmc_ctx* ctx = nullptr;
  if (!out) return fail(nullptr, HPMC_E_BADARG, "hpmc_alu_peaks: NULL argument");
  std::memset(out, 0, sizeof(*out));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0, khz = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return fail(nullptr, HPMC_E_CUDA, std::string("hpmc_alu_peaks: no usable CUDA device: ") + cudaGetErrorString(cudaGetLastError()));
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
  out->num_sms = sms; out->sm_clock_khz = khz;
  const int grid = 2 * sms;                       // 2 CTAs x 512 threads = 32 warps per SM, one wave
  unsigned long long* d_cyc = nullptr;
  uint32_t* d_sink = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  struct Release {                                // frees on every return path, the CU() ones included
    unsigned long long*& cyc; uint32_t*& sink; cudaEvent_t &a, &b;
    ~Release() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); cudaFree(cyc); cudaFree(sink); }
  } release{d_cyc, d_sink, e0, e1};
  CU(cudaMalloc(&d_cyc, sizeof(unsigned long long) * grid));
  CU(cudaMalloc(&d_sink, sizeof(uint32_t)));
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  const Key10 key = make_key(1u, 2u);
  std::vector<unsigned long long> cyc((size_t)grid);
  const int iters = 2048;
  double mhz_sum = 0.0;
  for (int kind = 0; kind < AK_COUNT; ++kind) {
    double best = 0.0;
    for (int rep = 0; rep < 3; ++rep) {           // first repetition warms up the instruction cache
      CU(cudaMemsetAsync(d_cyc, 0, sizeof(unsigned long long) * grid, st));
      CU(cudaEventRecord(e0, st));
#define HPMC_AK(K) case K: k_alu_peak<K><<<grid, AK_THREADS, 0, st>>>(iters, 0x9E3779B9u + rep, 0xBB67AE85u, 1.0000001f, 0.99999994f, key, d_cyc, d_sink); break;
      switch (kind) {
        HPMC_AK(AK_FADD) HPMC_AK(AK_FMUL) HPMC_AK(AK_FFMA) HPMC_AK(AK_IMAD) HPMC_AK(AK_IMADW_XOR) HPMC_AK(AK_LOP3) HPMC_AK(AK_MIX)
        HPMC_AK(AK_PHILOX1) HPMC_AK(AK_PHILOX2) HPMC_AK(AK_PHILOX4)
      }
#undef HPMC_AK
      CU(cudaEventRecord(e1, st));
      CU(cudaMemcpyAsync(cyc.data(), d_cyc, sizeof(unsigned long long) * grid, cudaMemcpyDeviceToHost, st));
      CU(cudaStreamSynchronize(st));
      CU(cudaGetLastError());
      unsigned long long cmax = 0;
      for (int i = 0; i < grid; ++i) cmax = cyc[(size_t)i] > cmax ? cyc[(size_t)i] : cmax;
      float ms = 0.0f;
      CU(cudaEventElapsedTime(&ms, e0, e1));
      // thread-instructions per SM per clock: 1024 threads per SM, per thread iters x (32 plain ops | NB Philox blocks)
      const double per_thread = kind >= AK_PHILOX1 ? (double)iters * (kind == AK_PHILOX1 ? 1.0 : kind == AK_PHILOX2 ? 2.0 : 4.0)
                                                   : (double)iters * (kind == AK_IMADW_XOR ? 64.0 : 32.0);
      const double rate = cmax ? 2.0 * AK_THREADS * per_thread / (double)cmax : 0.0;
      if (rep > 0 && rate > best) { best = rate; if (kind == AK_FADD && ms > 0.0f) mhz_sum = (double)cmax / ((double)ms * 1e3); }
    }
    out->rate[kind] = best;
  }
  out->sm_mhz_during = mhz_sum;
  return HPMC_OK;
}

const char* hpmc_last_error(hpmc_ctx* ctx) { return ctx ? ctx->err.c_str() : g_init_error.c_str(); }

}  // extern "C"

// =====================================================================================================================
// hpmc_cells_noalloc: step a2 (cell-list build) for callers that may not allocate device memory.
// Contract and rationale: include/hpmc.h.  Nothing above this line is touched by it; the kernels it shares with
// hpmc_build_cells (k_scan_tiles, k_fill, the device helpers of cells.cuh) are used as they are, through pointers.
//
// The working storage of the build (per-cell counts, scan tile totals, per-particle cell id and arrival rank) lives in
// ONE file-scope device array of fixed size instead of cudaMalloc'ed buffers.  Layout in 32-bit words:
//   [0, NA_MAX_CELLS)                 counts     must be zero when k_na_bin starts: cleared at the top of every call
//   [.., + NA_MAX_TILES)              tile_sums  fully rewritten by k_scan_tiles before it is read
//   [.., + NA_MAX_N)                  cid        rewritten for i < N before it is read
//   [.., + NA_MAX_N)                  rank       likewise
// 3 MiB + 512 B, present on every GPU that loads the library, for the life of the process.
// =====================================================================================================================

namespace {
constexpr int NA_MAX_N = 1 << 18;                         // 262,144 particles
constexpr int NA_MAX_CELLS = 1 << 18;                     // 262,144 cells, i.e. n_c <= 64
constexpr int NA_MAX_TILES = NA_MAX_CELLS / SCAN_TILE;
static_assert(NA_MAX_CELLS % SCAN_TILE == 0, "the counts region is scanned in whole tiles");
constexpr size_t NA_OFF_COUNTS = 0;
constexpr size_t NA_OFF_TILES = NA_OFF_COUNTS + NA_MAX_CELLS;
constexpr size_t NA_OFF_CID = NA_OFF_TILES + NA_MAX_TILES;
constexpr size_t NA_OFF_RANK = NA_OFF_CID + NA_MAX_N;
constexpr size_t NA_WORDS = NA_OFF_RANK + NA_MAX_N;
static_assert(NA_OFF_TILES % 64 == 0 && NA_OFF_CID % 64 == 0 && NA_OFF_RANK % 64 == 0, "sub-arrays stay 256-byte aligned");
}  // namespace

// In host code this name is only a handle for cudaGetSymbolAddress -- it is NOT a device pointer and must never be
// handed to a kernel or to cudaMemset* as one.  na_scratch_of_current_device() below turns it into the real address.
static __device__ __align__(256) uint32_t g_na_scratch[NA_WORDS];

namespace {

// k_bin_count without the outcome-code reset (there is no sweep behind this build) and with the cell index clamped at
// zero, so that a pose outside [0, L) -- a caller error -- lands in an edge cell instead of writing out of bounds.
__global__ void __launch_bounds__(256) k_na_bin(const float4* __restrict__ pos, int N, Geo g, float sx, float sy, float sz,
                                                uint32_t* __restrict__ cid, uint32_t* __restrict__ rank,
                                                uint32_t* __restrict__ counts) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const float4 p = pos[i];
  const int ix = max(cell_axis(g, p.x, sx), 0), iy = max(cell_axis(g, p.y, sy), 0), iz = max(cell_axis(g, p.z, sz), 0);
  const uint32_t c = ((uint32_t)iz * g.nc + iy) * g.nc + ix;
  cid[i] = c;
  rank[i] = atomicAdd(&counts[c], 1u);
}

// k_scan_apply<true> writing into a caller-owned cell_start of exactly n + 1 words (no padding to write into, so the
// stores are guarded scalars) and leaving the counts alone (the next call clears them itself).
__global__ void __launch_bounds__(SCAN_THREADS) k_na_scan_apply(const uint32_t* __restrict__ counts, int n,
                                                                const uint32_t* __restrict__ tile_sums,
                                                                uint32_t* __restrict__ cell_start) {
  __shared__ uint32_t s_warp[32];
  __shared__ uint32_t s_off;
  uint32_t part = 0;
  for (int i = threadIdx.x; i < (int)blockIdx.x; i += SCAN_THREADS) part += tile_sums[i];
  uint32_t tot;
  block_exclusive_scan(part, s_warp, tot);
  if (threadIdx.x == 0) s_off = tot;
  __syncthreads();
  const uint32_t off = s_off;
  const int base = blockIdx.x * SCAN_TILE + threadIdx.x * SCAN_ITEMS;
  uint32_t v[SCAN_ITEMS], s = 0;
  load8(counts + base, v);                         // the words between n and the end of the last tile are zero
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) s += v[k];
  uint32_t total;
  uint32_t run = off + block_exclusive_scan(s, s_warp, total);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    if (base + k <= n) cell_start[base + k] = run;   // index n receives the grand total N
    run += v[k];
  }
  if (base + SCAN_ITEMS == n) cell_start[n] = run;   // n a whole number of tiles: nobody owns index n above
}

// the ordering half of k_sort_write: ascending particle id inside every cell (undoes the atomics' arrival order)
__global__ void __launch_bounds__(256) k_na_sort(const uint32_t* __restrict__ cell_start, int ncell,
                                                 uint32_t* __restrict__ cell_pid) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  const uint32_t b = cell_start[c], e = cell_start[c + 1];
  for (uint32_t s = b + 1; s < e; ++s) {
    const uint32_t v = cell_pid[s];
    uint32_t t = s;
    while (t > b && cell_pid[t - 1] > v) { cell_pid[t] = cell_pid[t - 1]; --t; }
    cell_pid[t] = v;
  }
}

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mutex;
uint32_t* g_na_dev_ptr[NA_MAX_DEVICES] = {};     // device address of g_na_scratch, one per device, filled on first use

// Set-up, once per device, with that device current: ask the runtime where g_na_scratch lives on THIS device.
int na_scratch_of_current_device(uint32_t** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess)
    return fail(nullptr, HPMC_E_CUDA, std::string("hpmc_cells_noalloc: no usable CUDA device: ") + cudaGetErrorString(e));
  if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(nullptr, HPMC_E_CUDA, "hpmc_cells_noalloc: device ordinal beyond 63");
  std::lock_guard<std::mutex> lock(g_na_mutex);
  if (!g_na_dev_ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_na_scratch);
    if (e != cudaSuccess || !p)
      return fail(nullptr, HPMC_E_CUDA, std::string("hpmc_cells_noalloc: cudaGetSymbolAddress(g_na_scratch): ") + cudaGetErrorString(e));
    g_na_dev_ptr[dev] = static_cast<uint32_t*>(p);
  }
  *out = g_na_dev_ptr[dev];
  return HPMC_OK;
}

}  // namespace

extern "C" int hpmc_cells_noalloc(const float* d_pos4, int64_t N, float box_L, int32_t n_c, const float* host_shift3,
                                  uint32_t* d_cell_start, uint32_t* d_cell_pid, void* cuda_stream) {
  hpmc_ctx* ctx = nullptr;                          // CU() reports through hpmc_last_error(NULL)
  if (!d_pos4 || !host_shift3 || !d_cell_start || !d_cell_pid)
    return fail(nullptr, HPMC_E_BADARG, "hpmc_cells_noalloc: NULL argument");
  if (N < 1 || N > NA_MAX_N)
    return fail(nullptr, HPMC_E_BADARG, "hpmc_cells_noalloc: N = " + std::to_string(N) + " is outside 1 .. " +
                                            std::to_string(NA_MAX_N) + " (the fixed scratch array holds no more; use "
                                            "hpmc_init + hpmc_build_cells for larger systems)");
  if (n_c < 1 || (int64_t)n_c * n_c * n_c > NA_MAX_CELLS)
    return fail(nullptr, HPMC_E_BADARG, "hpmc_cells_noalloc: n_c = " + std::to_string(n_c) + " is outside 1 .. 64 (n_c^3 <= " +
                                            std::to_string(NA_MAX_CELLS) + " cells fit the fixed scratch array)");
  if (!(box_L > 0.0f)) return fail(nullptr, HPMC_E_BADARG, "hpmc_cells_noalloc: box_L must be positive");
  for (int a = 0; a < 3; ++a)
    if (!(host_shift3[a] >= 0.0f && host_shift3[a] <= box_L))
      return fail(nullptr, HPMC_E_BADARG, "hpmc_cells_noalloc: grid shift outside [0, box_L]");
  uint32_t* scratch = nullptr;
  const int rc = na_scratch_of_current_device(&scratch);
  if (rc) return rc;
  uint32_t* counts = scratch + NA_OFF_COUNTS;
  uint32_t* tile_sums = scratch + NA_OFF_TILES;
  uint32_t* cid = scratch + NA_OFF_CID;
  uint32_t* rank = scratch + NA_OFF_RANK;

  Geo g{};                                          // the binning reads L, w and nc only; same fp32 expressions as make_geo
  g.L = box_L; g.halfL = 0.5f * box_L; g.nc = n_c; g.w = box_L / (float)n_c;
  const int n = (int)N, ncell = n_c * n_c * n_c;
  const int ntiles = (ncell + SCAN_TILE - 1) / SCAN_TILE, nb = (n + 255) / 256;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // the array keeps whatever the previous call (any stream, any size) left in it: the counts must start at zero
  CU(cudaMemsetAsync(counts, 0, sizeof(uint32_t) * (size_t)ntiles * SCAN_TILE, st));
  k_na_bin<<<nb, 256, 0, st>>>(reinterpret_cast<const float4*>(d_pos4), n, g, host_shift3[0], host_shift3[1],
                               host_shift3[2], cid, rank, counts);
  k_scan_tiles<<<ntiles, SCAN_THREADS, 0, st>>>(counts, ncell, tile_sums);
  k_na_scan_apply<<<ntiles, SCAN_THREADS, 0, st>>>(counts, ncell, tile_sums, d_cell_start);
  k_fill<<<nb, 256, 0, st>>>(cid, rank, d_cell_start, n, d_cell_pid);
  k_na_sort<<<(ncell + 255) / 256, 256, 0, st>>>(d_cell_start, ncell, d_cell_pid);
  CU(cudaGetLastError());
  return HPMC_OK;
}
