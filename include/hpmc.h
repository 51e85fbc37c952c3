/* hpmc.h -- C-ABI boundary of the B200 (sm_100a) implicit-depletant hard-particle Monte Carlo library.
 *
 * The library implements ONE thing: the checkerboard-parallel colloid trial move with implicit
 * (ideal-gas) depletant insertion of arXiv 1508.07077 (Glaser, Karas, Glotzer).  Citations are line
 * numbers of /root/reference/PAPER.md (L<n>) and the readings R-* listed in DESIGN.md.
 *
 *   move rule            Sec. III.B  L64-68, Fig. 2 L72, Eq. 5
 *   insertion volume     Sec. III.C  L117, L156 (circumsphere of diameter d_colloid+d_depletant, new pose)
 *   configurational bias Sec. III.D  L170-174, Eq. 16
 *   checkerboard         Sec. III.E  L180
 *
 * Conventions
 *   - All entry points are extern "C", take plain pointers and sizes, return 0 on success or a negative
 *     hpmc_status; they never throw.  hpmc_last_error() gives the message of the last failure.
 *   - "device" pointers are CUDA device pointers of the current device; "host" pointers are ordinary (or,
 *     better, page-locked) host memory.  Every argument below says which.
 *   - Poses: centre = float4 (x, y, z, unused) with 0 <= x,y,z < box_L; orientation = float4 unit
 *     quaternion (w, x, y, z).  fp32 throughout (paper: "single precision", L232).
 *   - Work is enqueued on the cudaStream_t given to hpmc_init and is asynchronous unless stated.
 *   - There is no CPU fallback: without a CUDA device every call that touches the device fails with
 *     HPMC_E_CUDA.
 */
#ifndef HPMC_H_
#define HPMC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct hpmc_ctx hpmc_ctx; /* opaque, library-owned */

typedef enum {
  HPMC_SPHERE = 0,     /* sphere of diameter sigma_c */
  HPMC_HALFBALL = 1,   /* {x: |x| <= sigma_c/2, x.z_body <= 0}: flat face through the pose centre, outward normal +z_body */
  HPMC_SPHERODISK = 2, /* Minkowski sum of a flat disk (radius disk_a, normal z_body) and a ball (radius disk_s) */
  HPMC_TETRAHEDRON = 4, /* regular tetrahedron with circumradius sigma_c / 2, body-frame vertices (sigma_c / (2 sqrt 3)) x
                          {(1,1,1), (1,-1,-1), (-1,1,-1), (-1,-1,1)} (Fig. 1 L21; NEXT-2, reading R-N2b) */
  HPMC_ELLIPSOID = 3,  /* oblate spheroid, semi-axes (disk_a, disk_a, disk_s), 4 disk_s >= disk_a >= disk_s > 0 (aspect ratio at
                          most 4: what the fixed-length closest-point iteration resolves), short axis z_body: the paper's
                          discoids (reading R-N2); sigma_c must equal 2 disk_a */
  HPMC_SHAPE_COUNT = 5
} hpmc_shape;

typedef enum {
  HPMC_OK = 0,
  HPMC_E_BADARG = -1,            /* NULL pointer, N <= 0, box_L <= 0, negative density, n_trial > 65535 ... */
  HPMC_E_GEOMETRY = -2,          /* fewer than 4 cells per axis: box too small for the interaction range */
  HPMC_E_STATE = -3,             /* hpmc_sweep without hpmc_build_cells for the same (seed, step) */
  HPMC_E_DMAX = -4,              /* d_max > d_max_cap given at init */
  HPMC_E_CUDA = -5,              /* CUDA runtime error (message in hpmc_last_error).  Also: in the one-launch sweep a CTA
                                    waited longer than 60 s of wall clock for a neighbouring CTA's pass -- which the
                                    cooperative launch rules out short of a lost CTA -- and abandoned the sweep without
                                    committing the rest of its moves; reported and cleared like the overflow below,
                                    poses and counters of that sweep are invalid, the context stays usable */
  HPMC_E_NEIGHBOR_OVERFLOW = -6  /* ONE move has more neighbours inside the list radius than the staging buffer holds
                                    (reported and cleared by the next synchronising call; poses of that sweep are
                                    then invalid).  Locally dense tiles do not raise it: the move kernel halves a
                                    tile whose neighbour pool overflows and redoes it; the pool holds >= 768
                                    neighbours, far more than hard particles can place around one move. */
} hpmc_status;

typedef struct {
  int32_t shape;       /* hpmc_shape */
  float sigma_c;       /* circumsphere diameter d_colloid: sphere diameter, 2 R_halfball, 2 (disk_a + disk_s) */
  float disk_a;        /* spherodisk: disk radius a >= 0; ellipsoid: equatorial semi-axis */
  float disk_s;        /* spherodisk: rounding radius s >= 0, sigma_c must equal 2 (a + s); ellipsoid: polar semi-axis,
                          sigma_c must equal 2 disk_a; else HPMC_E_BADARG */
  float sigma_d;       /* depletant diameter d_depletant (>= 0) */
  float box_L;         /* edge of the cubic periodic box */
  float d_max_cap;     /* largest d_max any later sweep will use; fixes the cell width
                          w >= sigma_c + sigma_d + 2 d_max_cap (BASELINE.json north_star; L180) */
} hpmc_params;

/* All counters accumulate since init / hpmc_reset_counters. */
typedef struct {
  uint64_t trials_trans, accept_trans, trials_rot, accept_rot;
  uint64_t rej_boundary;    /* new centre left the cell (L180 "not allowed to move outside their cells") */
  uint64_t rej_hard;        /* overlap with another colloid (Eq. 5) */
  uint64_t rej_depletant;   /* plain rule: a depletant overlapped the new pose only (L68, L72) */
  uint64_t rej_cb;          /* configurational-bias rule: zero weight or u >= product (Eq. 16) */
  uint64_t dep_drawn;       /* sum of N_d over moves that reached the depletant stage (L67) */
  uint64_t dep_needed;      /* sum of (index of the first rejecting depletant + 1), or N_d if none: the
                               sequential algorithm's work; identical in the oracle */
  uint64_t dep_evaluated;   /* depletant positions the kernel actually generated (>= dep_needed).  This one and
                               philox_blocks describe the kernel's own work, not the algorithm's: a tile that is
                               split and redone (neighbour-pool overflow) or a configurational-bias window that is
                               redone (job overflow) is counted again, so both depend on the tiling */
  uint64_t cb_reinsertions; /* 2 n_trial per rejecting depletant handled (Sec. III.D); 2 n_trial - 1 with HPMC_OPT_ROSENBLUTH */
  uint64_t philox_blocks;   /* Philox4x32-10 blocks computed (warp-uniform ones counted once) */
} hpmc_counters_t;

/* Per-particle outcome code of the last sweep (each particle is tried at most once per sweep). */
enum { HPMC_OUT_NONE = 0, HPMC_OUT_ACCEPT = 1, HPMC_OUT_BOUNDARY = 2, HPMC_OUT_HARD = 3,
       HPMC_OUT_DEPLETANT = 4, HPMC_OUT_CB = 5 };

/* Create a context for N colloids.
 *   d_pos4   device, N x float4, caller-owned, borrowed for the context's lifetime, updated IN PLACE by
 *            hpmc_sweep.  NULL: the library allocates its own pose buffers (use hpmc_upload/hpmc_download).
 *   d_quat4  device, N x float4 (w,x,y,z), same ownership; may be NULL for spheres.  Must be NULL iff
 *            d_pos4 is NULL.
 *   cuda_stream  a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream), or NULL for the default.
 * Cell grid (R-1, L180): n_c = largest even integer <= box_L / (sigma_c + sigma_d + 2 d_max_cap) per axis,
 * n_c >= 4 else HPMC_E_GEOMETRY.  Cell arrays, tables, counters are library-owned device memory. */
int hpmc_init(hpmc_ctx** out, const hpmc_params* p, int64_t N, float* d_pos4, float* d_quat4, void* cuda_stream);

/* Free everything the library owns.  Caller-owned pose buffers are left alone.  Synchronises the stream. */
void hpmc_destroy(hpmc_ctx* ctx);

/* Cell-list build, step a2: draws this sweep's grid shift from Philox(seed, step) ("grid lines are randomly
 * shifted", L180), bins the centres, lists the occupants of every cell in ascending particle id and writes the
 * cell-ordered pose copy.  Call once before every hpmc_sweep with the same (seed, step).  Asynchronous. */
int hpmc_build_cells(hpmc_ctx* ctx, uint32_t seed, uint32_t step);

/* One sweep = the 8 checkerboard sub-lattice passes in a Philox-permuted order (L180), steps a3-a10, normally ONE
 * cooperative kernel launch in which a CTA waits between passes only for the CTAs owning neighbouring cells.  In every
 * non-empty active cell one colloid gets a trial move: translation uniform in [-d_max, d_max]^3, or (if
 * a_max > 0, with probability 1/2) a Cayley rotation with parameter vector uniform in the ball of radius a_max.
 *   n_R      depletant reservoir number density (fugacity z_p, L214); 0 = plain hard-particle MC
 *   n_trial  0 = plain rule (L68); > 0 = configurational bias with n_trial reinsertions each way (Eq. 16)
 * Requires hpmc_build_cells(seed, step) before it, else HPMC_E_STATE; d_max <= d_max_cap else HPMC_E_DMAX.
 * Asynchronous; poses are updated in place. */
int hpmc_sweep(hpmc_ctx* ctx, uint32_t seed, uint32_t step, double n_R, float d_max, float a_max, int32_t n_trial);

/* Options of the sweeps that follow (persistent; default 0 = the path exactly as described above).
 *   HPMC_OPT_SHELL       SURVEY 8(f) NEXT-1, PAPER.md L158 ("restricting the sampling to the excluded volume shell of
 *                        the moved colloid"), reading R-N1: depletants are drawn uniformly in the shell
 *                        R_in < |d| <= R about the new centre, R = (sigma_c + sigma_d)/2, R_in = max(0, r_in - sqrt(3) d_max)
 *                        with r_in = R (sphere), sigma_d/2 (half-ball), disk_s + sigma_d/2 (spherodisk): the largest
 *                        concentric ball that lies inside the OLD pose's excluded volume for every move of the sweep,
 *                        which is what Eq. 12 (L136) requires.  N_d ~ Poisson(n_R V_shell).  Same transition rate
 *                        (Eq. 15), fewer insertions: the shell is 42 % of the ball at C3's d_max = 0.05.
 *   HPMC_OPT_ROSENBLUTH  NEXT-4, refs 27, 28, 33 (L288-294), reading R-N4: with n_trial > 0 the weight of a rejecting
 *                        depletant is N'_ins / (N_ins + 1) from n_trial forward and n_trial - 1 fresh reverse
 *                        reinsertions (the exact Rosenbluth form) instead of Eq. 16 as printed / adopted (R-G1).
 * Unknown bits: HPMC_E_BADARG.  Host-side only, takes effect with the next hpmc_sweep. */
enum { HPMC_OPT_SHELL = 1, HPMC_OPT_ROSENBLUTH = 2 };
int hpmc_set_options(hpmc_ctx* ctx, uint32_t options);

/* n_sweeps x (hpmc_build_cells + hpmc_sweep) with step = step0, step0+1, ...  Asynchronous. */
int hpmc_run(hpmc_ctx* ctx, uint32_t seed, uint32_t step0, int64_t n_sweeps, double n_R, float d_max, float a_max,
             int32_t n_trial);

/* Synchronise the stream and copy the counters to host_out (host).  Does not reset them.  Reports a pending
 * HPMC_E_NEIGHBOR_OVERFLOW. */
int hpmc_counters(hpmc_ctx* ctx, hpmc_counters_t* host_out);
int hpmc_reset_counters(hpmc_ctx* ctx);

/* Free-volume measurement (Sec. IV.A, Fig. 4: the depletant density in the system
 * is n_R times the free-volume fraction).  n_samples test depletants at points uniform in the box -- sample s from the
 * Philox block (s mod 2^32, s / 2^32, 0, FREEVOL = 7) of key (seed, step), x_a = unit01(word a) box_L -- are tested with
 * the insertion kernel's own predicate against the 27 cells around the point; *host_free_count = how many overlap no
 * colloid, so free-volume fraction = count / n_samples.  Needs hpmc_build_cells(seed, step) (else HPMC_E_STATE) and may
 * be called before or instead of hpmc_sweep.  Synchronises the stream. */
int hpmc_free_volume(hpmc_ctx* ctx, uint32_t seed, uint32_t step, int64_t n_samples, uint64_t* host_free_count);

/* Copy the outcome codes of the last sweep into d_outcome (device, N bytes, caller-owned).  Asynchronous.
 * hpmc_build_cells resets the codes to HPMC_OUT_NONE for the sweep it prepares. */
int hpmc_outcomes(hpmc_ctx* ctx, uint8_t* d_outcome);

/* Grid geometry chosen at init: cells per axis and cell width. */
int hpmc_grid(hpmc_ctx* ctx, int32_t* n_c, float* w);

/* Debug / parity: copy the cell list of the last hpmc_build_cells into caller-owned DEVICE buffers
 * (cell_start: n_c^3 + 1 uint32; cell_pid: N uint32) and the grid shift into host_shift3 (host, 3 floats).
 * Synchronises the stream. */
int hpmc_cells(hpmc_ctx* ctx, uint32_t* d_cell_start, uint32_t* d_cell_pid, float* host_shift3);

/* Host-buffer path (end-to-end measurements; library-owned pose buffers or borrowed ones alike).
 * hpmc_upload: host -> device copy of N x float4 centres (and orientations unless NULL).
 * hpmc_download: device -> host copy of centres, orientations and outcome codes (any may be NULL).
 * hpmc_step_host: upload, hpmc_build_cells, hpmc_sweep, download, then synchronise: one whole step with the
 * host<->device traffic inside it.  The download is sparse when it pays: the move kernel lists the particles it accepted,
 * the outcome codes (N bytes) and the list length come back first, and if at most N/4 particles moved only their poses
 * are copied (packed by a gather kernel) and patched into host_pos4 / host_quat4 -- which still hold the uploaded poses
 * of everybody else -- otherwise the whole arrays.  The host arrays end up exactly as after a full download.
 * hpmc_step_host_bytes: bytes the last hpmc_step_host moved in each direction. */
int hpmc_upload(hpmc_ctx* ctx, const float* host_pos4, const float* host_quat4);
int hpmc_download(hpmc_ctx* ctx, float* host_pos4, float* host_quat4, uint8_t* host_outcome);
int hpmc_step_host(hpmc_ctx* ctx, float* host_pos4, float* host_quat4, uint8_t* host_outcome, uint32_t seed,
                   uint32_t step, double n_R, float d_max, float a_max, int32_t n_trial);
int hpmc_step_host_bytes(hpmc_ctx* ctx, int64_t* h2d_bytes, int64_t* d2h_bytes);

/* Number of kernel launches the library has enqueued since init (for bench.py's gpu_launches). */
int64_t hpmc_launch_count(hpmc_ctx* ctx);

/* Event timing of the move kernel (the dominant kernel): while enabled, the move-kernel launch(es) of every sweep -- one
 * cooperative launch for the 8 passes, or 8 launches (HPMC_SWEEP_LAUNCHES=8, the warp-per-cell kernel) -- are bracketed
 * by ONE pair of CUDA events on the context's stream (gaps between launches are inside the bracket);
 * hpmc_move_kernel_ms synchronises and returns the accumulated milliseconds and the number of launches since enabling. */
int hpmc_time_move_kernel(hpmc_ctx* ctx, int32_t enable);
int hpmc_move_kernel_ms(hpmc_ctx* ctx, double* ms_total, int64_t* launches);

/* Micro-benchmark of the plain ALU pipes on the current device (the roofline denominator of the move kernel;
 * MEASURED_PEAKS.json holds no ALU figure).  rate[i] = thread-instructions per SM per clock of a
 * dependency-free stream of one kind, 32 resident warps per SM, counted with clock64() (clock-independent):
 *   [0] FADD  [1] FMUL  [2] FFMA (context: the path is compiled without contraction)  [3] IMAD
 *   [4] IMAD.WIDE.U32 + LOP3 pairs (one half of a Philox round; both instructions counted)
 *   [5] LOP3  [6] FADD and LOP3 alternating (both pipes: the issue limit)
 *   [7],[8],[9] Philox4x32-10 BLOCKS per SM per clock with 1, 2, 4 independent blocks per thread.
 * out is host memory; needs no context; synchronises cuda_stream.  Takes a few milliseconds. */
typedef struct {
  int32_t num_sms;         /* cudaDevAttrMultiProcessorCount */
  int32_t sm_clock_khz;    /* cudaDevAttrClockRate (nominal maximum) */
  double sm_mhz_during;    /* SM clock seen during the FADD stream: cycles / event time */
  double rate[10];
} hpmc_alu_peaks_t;
int hpmc_alu_peaks(hpmc_alu_peaks_t* out, void* cuda_stream);

/* Cell-list build without any device allocation (step a2 on its own).
 *
 * Who this is for.  Every other call needs an hpmc_ctx, and hpmc_init / hpmc_free_volume / hpmc_step_host obtain their
 * working buffers with cudaMalloc.  Some programs that want the checkerboard cell list of a configuration cannot afford
 * that: an analysis hook (cluster search, local density, neighbour query) called from inside a running simulation
 * whose framework pool -- PyTorch's caching allocator, a simulation engine's arena -- already owns almost all of HBM, so
 * that a raw cudaMalloc from this library fails although the application has memory to spare; and per-step code for
 * which cudaMalloc / cudaFree are too costly because cudaFree waits for every stream of the device.  For them this one
 * entry point keeps its working storage (cell counts, scan partials, per-particle cell id and rank) in a fixed array
 * that is part of the library image: 3 MiB that every GPU which loads the library holds until the process exits.  It
 * calls no cudaMalloc, cudaFree or other allocating routine, creates no context and needs none.
 *
 *   d_pos4        device, N x float4 centres (x, y, z, unused), 0 <= x,y,z < box_L; read only
 *   N             1 .. 262,144                                  } beyond either limit: HPMC_E_BADARG, nothing is launched;
 *   n_c           cells per axis, 1 .. 64 (n_c^3 <= 262,144)    } hpmc_last_error(NULL) names the limit
 *   box_L         edge of the cubic periodic box; cell width w = box_L / n_c in fp32, as hpmc_init computes it
 *   host_shift3   host, 3 floats in [0, box_L]: the grid shift (hpmc_build_cells draws it from Philox(seed, step) and
 *                 hpmc_cells reports it; pass zeros for an unshifted grid)
 *   d_cell_start  device, n_c^3 + 1 uint32, caller-owned, written: first slot of every cell, cells in ascending linear
 *                 index (ix fastest); d_cell_start[n_c^3] = N
 *   d_cell_pid    device, N uint32, caller-owned, written: particle ids, ascending inside each cell
 *   cuda_stream   a cudaStream_t or NULL; the work is enqueued there and the call returns without synchronising
 * The result equals, bit for bit, what hpmc_build_cells + hpmc_cells give for the same poses, grid and shift.
 *
 * Rules that follow from the shared array:
 *   - One array per GPU serves every call, whatever the stream or thread.  Two calls whose kernels can overlap on the
 *     GPU (different streams, no event between them) race on it and both results are garbage; calls on one stream, or
 *     ordered by events, are fine.  The array keeps the previous call's contents; the part that must start at zero is
 *     cleared (cudaMemsetAsync on the same stream) at the start of every call, so nothing carries over.
 *   - The first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *     current) and remembers it; later calls on that device skip this.  Make that first call before any stream
 *     capture is begun.  Call with the device current that owns d_pos4 and the outputs.
 * Errors: HPMC_E_BADARG (NULL pointer, sizes beyond the limits above, box_L <= 0, shift outside [0, box_L]),
 * HPMC_E_CUDA (no device, address look-up or launch failure); message in hpmc_last_error(NULL). */
int hpmc_cells_noalloc(const float* d_pos4, int64_t N, float box_L, int32_t n_c, const float* host_shift3,
                       uint32_t* d_cell_start, uint32_t* d_cell_pid, void* cuda_stream);

/* Message of the last error on this context (or, if ctx is NULL, of the last failed call that takes no context --
 * hpmc_init, hpmc_alu_peaks, hpmc_cells_noalloc -- on the calling thread). */
const char* hpmc_last_error(hpmc_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* HPMC_H_ */
