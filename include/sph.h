/* include/sph.h — C ABI of libsph, the B200 (sm_100a) implementation of the per-time-step
 * particle pipeline of arXiv 2110.02621 (Rezavand, Zhang, Hu: "Generalised and efficient wall
 * boundary condition treatment in GPU-accelerated SPH").
 *
 * Citations are PAPER.md:<line> (+ equation).  "Reading Axx" refers to DESIGN.md §3.
 *
 * Conventions
 *  - No torch types, no C++ types, no exceptions cross this boundary.
 *  - Every function returns 0 (SPH_OK) or a negative sph_error; sph_last_error() gives text.
 *  - Pointers named *_dev are DEVICE pointers owned by the caller (e.g. torch tensors);
 *    pointers named *_host are HOST pointers owned by the caller.  The library copies in
 *    at sph_set_particles* and out at sph_get_fields*; it never keeps a caller pointer.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls are
 *    asynchronous on that stream unless stated; the *_host variants and the calls that
 *    return values to the host synchronise the stream before returning.
 *  - Particle arrays are in the CALLER'S ORDER: pos[n*3], vel[n*3] (xyz interleaved, z ignored
 *    in 2-D), rho[n], tag[n].  tag = phase id 0..n_phases-1 for fluid (phase 0 the heaviest),
 *    SPH_TAG_WALL for wall dummy particles.  Results come back in the same
 *    order; the internal cell-sorted order is visible only through sph_debug_*.
 *  - Pair arithmetic is float32 on the device ("fully developed on single precision");
 *    density is held as the deviation rho - rho0 of the particle's phase, positions as 42-bit fixed
 *    point (units of Q/1024, Q = 2^-k m about 1 nm for metre-sized domains; the pair kernels read it modulo
 *    2^32 units of Q / 2^m) so that float32 inputs are held exactly and sph_get_fields returns the float32
 *    rounding of the held position; the number density sigma_i is summed in float64 (DESIGN.md §4 says why).
 *  - There is no CPU fallback: every call fails with SPH_ECUDA if no CUDA device is usable.
 *  - No global state (one exception, stated there: the device scratch array of sph_cell_sort_static).  sph_create reads six environment variables that exist only so that the experiments of
 *    profiles/r02_README.md can be repeated from the committed build (SPH_SKIN: largest skin; SPH_SUB_BITS: sub-cell
 *    Morton bits in the sort key; SPH_REACH=2: cell edge h with a 125-cell walk; SPH_MBITS: cap on m above;
 *    SPH_FORCE_SUBQ / SPH_NO_SUBQ: the low position bits in sigma on / off).  None is needed for normal use.
 */
#ifndef SPH_H_
#define SPH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sph_ctx sph_ctx; /* opaque; owned by the library; one per simulation */

enum { SPH_MAX_PHASES = 4, SPH_TAG_WALL = -1 };

enum sph_flags {
  SPH_FLAG_REINIT = 1,          /* density reinitialisation each step, Eq. 2.17/2.18 */
  SPH_FLAG_WALL_VEL_MIRROR = 2, /* v_w = 2 v_wall - <v_f> (Adami-style mirror; reading A6), else v_w = v_wall */
  SPH_FLAG_NO_GRAPH = 4,        /* sph_step issues every kernel itself instead of replaying one captured step
                                   as a CUDA graph (same kernels, same results) */
  SPH_FLAG_WALL_ADAMI_ONLY = 8  /* NEXT-4 ablation, PAPER.md:99, :250 ("compare the results with the method of Adami et
                                   al. (2012)"): the wall model without the paper's extensions: Eq. 2.12 in its
                                   single-phase form for every phase (no division by rho_f) and no
                                   penalty force F_p (Eq. 2.13), whatever penalty_phase_mask says */
};

enum sph_error {
  SPH_OK = 0,
  SPH_EINVAL = -1,      /* bad argument / tag out of range / called before sph_set_particles */
  SPH_ENOMEM = -2,      /* device or host allocation failed */
  SPH_ECUDA = -3,       /* CUDA runtime error (no device, launch failure, ...) */
  SPH_ENONFINITE = -4,  /* a non-finite position or velocity was seen (reported by sph_get_stats) */
  SPH_EDTUNDERFLOW = -5, /* the time step fell below 1e-12 (reported by sph_get_stats) */
  SPH_ENEIGHBOURS = -6   /* a particle had more neighbours than max_neighbours (reported by sph_get_stats);
                            the step results are then incomplete */
};

/* Physical and numerical parameters: the paper's statement of the problem. */
typedef struct {
  int32_t dim;                   /* 2 or 3   */
  int32_t n_phases;              /* 1..SPH_MAX_PHASES  */
  double dp;                     /* initial particle spacing dx */
  double h;                      /* smoothing length (paper: 1.3 dx; support 2h) */
  double rho0[SPH_MAX_PHASES];   /* reference density per phase  */
  double c0[SPH_MAX_PHASES];     /* speed of sound per phase, Eq. 2.3 (reading A2, A3) */
  double g[3];                   /* body acceleration */
  double g_osc_amp[3];           /* g(t) = g + g_osc_amp * sin(2 pi t / g_osc_period)   (config 3)   */
  double g_osc_period;           /* 0 = constant gravity                                             */
  double cfl;                    /* 0.25 in Eq. 2.23 and 2.24 */
  double penalty_strength;       /* gamma_p (paper: 1) */
  uint32_t penalty_phase_mask;   /* bit k: phase k receives F_p, Eq. 2.13 (reading A11) PAPER.md:120 */
  uint32_t free_surface_mask;    /* bit k: phase k uses continuity Eq. 2.9/2.21 + reinit Eq. 2.17, and in a multi-phase
                                    run its number density sigma_i counts its own phase and the walls only (reading
                                    A13b, "free-surface-like flow"); otherwise summation Eq. 2.4 + reinit
                                    Eq. 2.18 with sigma_i over every neighbour (reading A13, A15) */
  uint32_t flags;                /* sph_flags */
  uint32_t max_neighbours;       /* capacity of the per-particle fluid-fluid neighbour lists; 0 = default (160 in 3-D,
                                    64 in 2-D); the fluid-wall lists hold 3/4 of it */
  double domain_min[3];          /* box of the cell grid; particles outside are binned in the edge */
  double domain_max[3];          /* cells and counted as escaped (reading A23)                      */
  double wall_osc_amp[3];        /* NEXT-1: all walls translate rigidly, x_w(t) = x_w(0) + wall_osc_amp *   */
  double wall_osc_freq;          /* sin(2 pi wall_osc_freq t); a_w enters Eq. 2.12,
                                    v_wall the mirror of reading A6; 0 = static walls.  The wall cell list is
                                    then rebuilt with the lists; the domain box must contain the whole excursion */
  double list_skin;              /* Verlet skin s: the cell list and the per-particle neighbour lists are built with radius
                                    2h(1 + s) (cell edge 2h(1 + s)) and kept over the following steps until a pair
                                    further apart than that could have come within 2h, i.e. until 2 sum_n max_i |dx_i^n|
                                    (or that of fluid + walls) exceeds 2 h s; entries beyond 2h add exactly 0.  The value
                                    given is the LARGEST skin (it fixes the cell edge); every build takes the skin in
                                    [0.002, list_skin] that minimises pass cost + build cost / steps between builds for
                                    the displacement per step seen then (a fluid at rest keeps thin lists for long, a
                                    violent flow thicker ones for a few steps).  0 = rebuild every step; < 0 = library
                                    default (0.1); at most 0.5.  Results do not depend on it beyond the order of
                                    floating-point sums */
} sph_params;

typedef struct {
  double t;          /* simulated time                                  */
  double dt;         /* last time step used                             */
  int64_t steps;     /* steps taken since sph_set_particles             */
  int64_t n_fluid;
  int64_t n_wall;
  int64_t n_pairs;   /* directed pairs (i fluid, j any tag, j != i, r < 2h) at the current positions */
  double e_kin;      /* sum 1/2 m |v|^2 over fluid                      */
  double mass;       /* sum m over fluid (m = rho0_phase dp^dim, reading A19) */
  double x_front;    /* max x over phase-0 particles within 3 dp of the floor (floor = domain_min[dim-1] + 3 dp) */
  int64_t escaped;   /* fluid particles outside [domain_min, domain_max) at the last cell build */
  int64_t nonfinite; /* non-finite positions/velocities seen so far     */
  int64_t rebuilds;  /* cell-list / neighbour-list builds since sph_set_particles (its own included) */
  double list_skin;  /* skin of the lists in use (adaptive, within [0.002, sph_params.list_skin]) */
} sph_stats;

/* Stages timed by sph_set_profiling (indices into sph_get_timings' array). */
enum sph_stage {
  SPH_STAGE_PREDICT = 0,   /* dt reduction + reinit (Eq. 2.17/2.18) + half kick + drift (Eq. 2.19-2.20) + cell hash */
  SPH_STAGE_SORT = 1,      /* device radix sort of (cell id, index); only on steps that rebuild the lists */
  SPH_STAGE_REORDER = 2,   /* gather into sorted SoA float4 + cell ranges; only on steps that rebuild */
  SPH_STAGE_WALL = 3,      /* wall extrapolation Eq. 2.12 (both calls of a step) */
  SPH_STAGE_PASS_A = 4,    /* sigma + continuity Eq. 2.9 + density update Eq. 2.21 / 2.4 + EOS */
  SPH_STAGE_PASS_B = 5,    /* momentum Eq. 2.10/2.11 + penalty Eq. 2.13 + second kick Eq. 2.22 */
  SPH_STAGE_BUILD = 6,     /* neighbour-list build: the 27 / 9-cell candidate walks (fluid and wall rows), on the
                              steps that rebuild (every step when list_skin = 0) */
  SPH_STAGE_COUNT = 7
};

/* Create a context.  Validates the parameters (SPH_EINVAL), selects the current CUDA device. */
int sph_create(const sph_params* params, sph_ctx** out);

/* Free everything the context owns.  NULL is allowed. */
void sph_destroy(sph_ctx* ctx);

/* Load n particles (fluid + wall).  One-off set-up work happens here (PAPER.md:101, :139-143,
 * SURVEY §8(c) O-0): masses, the static wall cell list, wall normals Eq. 2.16 (in float64,
 * reading A10), the first fluid cell list, sigma_i, wall extrapolation and (dv/dt)^0 (reading
 * A18).  Resets t = 0.  May be called again to restart from a checkpoint.
 * Synchronises the stream (it sizes allocations from the tag counts). */
int sph_set_particles(sph_ctx* ctx, int64_t n, const float* pos_dev, const float* vel_dev,
                      const float* rho_dev, const int32_t* tag_dev, void* stream);
int sph_set_particles_host(sph_ctx* ctx, int64_t n, const float* pos_host, const float* vel_host,
                           const float* rho_host, const int32_t* tag_host, void* stream);

/* Advance n_steps kick-drift-kick steps (Eq. 2.19-2.24); dt is computed on
 * the device each step from Eq. 2.23-2.24 (reading A17).  Asynchronous; no host sync per step.
 * The first call after sph_set_particles captures one step as a CUDA graph (it synchronises the
 * stream once to do so); later steps replay it on `stream` (SPH_FLAG_NO_GRAPH: plain launches). */
int sph_step(sph_ctx* ctx, int32_t n_steps, void* stream);

/* Same, with a caller-given dt sequence (host array of n_steps doubles) so that the oracle and
 * the device can be driven by identical time steps in parity runs. */
int sph_step_dt(sph_ctx* ctx, int32_t n_steps, const double* dt_host, void* stream);

/* Copy fields out in the caller's particle order.  Any pointer may be NULL.
 * pos, vel, acc: n*3; rho, p: n.  Wall entries: vel = extrapolated v_w, p = p_w (Eq. 2.12),
 * rho = rho0[0] + p_w / c0[0]^2, acc = 0.  The _host variant synchronises. */
int sph_get_fields(sph_ctx* ctx, float* pos_dev, float* vel_dev, float* rho_dev, float* p_dev,
                   float* acc_dev, void* stream);
int sph_get_fields_host(sph_ctx* ctx, float* pos_host, float* vel_host, float* rho_host,
                        float* p_host, float* acc_host, void* stream);

/* Integral quantities; runs small reduction kernels and synchronises.  Returns SPH_ENONFINITE /
 * SPH_EDTUNDERFLOW (with *out filled) if the run has gone bad. */
int sph_get_stats(sph_ctx* ctx, sph_stats* out, void* stream);
/* Same; with_pairs = 0 skips the contract-exact pair count (a full stencil walk, as expensive as a
 * pair pass) and returns n_pairs = -1: the per-step monitoring call (t, dt, E_k, mass, x_front). */
int sph_get_stats_ex(sph_ctx* ctx, sph_stats* out, int32_t with_pairs, void* stream);

/* Per-stage device times.  With profiling on, sph_step brackets every stage with CUDA events
 * on the caller's stream; sph_get_timings synchronises and returns the accumulated milliseconds
 * per stage since the last call (ms_host[SPH_STAGE_COUNT]) and the number of steps they cover.  With profiling
 * on the steps are issued as plain launches and the host reads the rebuild decision once per step. */
int sph_set_profiling(sph_ctx* ctx, int32_t on);
int sph_get_timings(sph_ctx* ctx, float* ms_host, int32_t* n_steps_host, int32_t* n_rebuilds_host /* may be NULL:
                    how many of those steps rebuilt the lists */);

/* Number of cells of the grid (cell edge 2h(1+2^-10), reading A24). */
int64_t sph_num_cells(const sph_ctx* ctx);

/* Integer contract, all HOST pointers, synchronises:
 * cell_id[n]: cell of every particle, caller order; perm[n]: fluid ids in cell-sorted order
 * followed by wall ids in cell-sorted order; cell_start/cell_end[2*ncell]: ranges in the fluid
 * block then in the wall block (both 0 for an empty cell).  Any pointer may be NULL. */
int sph_debug_cells(sph_ctx* ctx, int32_t* cell_id_host, int32_t* perm_host,
                    int32_t* cell_start_host, int32_t* cell_end_host, void* stream);

/* Neighbour lists in CSR form, caller ids, ascending within a row: fluid i -> all j != i with
 * r2 < 4h^2 (float32 rule of reading A24); wall i -> fluid j only.  offsets_host[n+1];
 * ids_host may be NULL (count only) and holds at most cap entries.  *total_host = number of
 * entries needed. */
int sph_debug_neighbours(sph_ctx* ctx, int64_t* offsets_host, int32_t* ids_host, int64_t cap,
                         int64_t* total_host, void* stream);

/* On-device probes (SURVEY.md section 8(f) NEXT-3; PAPER.md:296 pressure sensors, :304 water-level
 * probes; the paper prints neither formula: readings A29 / A30 of DESIGN.md section 3).  m probes,
 * xyz_host = m*3 floats (z ignored in 2-D); all pointers HOST, each call synchronises the stream; the
 * state probed is the one sph_get_fields would return.
 * sph_probe_pressure: p_host[k] = sum_f p_f W(|x_k - r_f|) / sum_f W over the fluid particles within
 *   2h of x_k (Wendland C2, reading A1), 0 where there is none; wsum_host[k] = sum_f W (1/m^d).
 * sph_probe_gauge: eta_host[k] = max { z_f + dp/2 : phase 0, horizontal distance to (x_k[, y_k]) < h }
 *   ("z" is y in 2-D), NaN where there is no such particle.
 * Errors: SPH_EINVAL (NULL pointers, m < 0, no particles), SPH_ECUDA. */
int sph_probe_pressure(sph_ctx* ctx, int32_t m, const float* xyz_host, float* p_host, float* wsum_host,
                       void* stream);
int sph_probe_gauge(sph_ctx* ctx, int32_t m, const float* xyz_host, float* eta_host, void* stream);

/* Checks the step's fluid-fluid neighbour lists (built once per step by the candidate filter,
 * DESIGN.md section 5) against the float32 contract of reading A24 on the current positions:
 * out3_host[0] = contract neighbours missing from a list (must be 0: the filter is conservative),
 * out3_host[1] = list entries that are not contract neighbours (filter margin; they add exactly 0,
 * reading B2), out3_host[2] = list entries in total (self entries included).  HOST pointer to 3
 * values; synchronises the stream.  Errors: SPH_EINVAL without particles, SPH_ECUDA. */
int sph_debug_list_check(sph_ctx* ctx, int64_t* out3_host, void* stream);

/* The neighbour lists the pair passes (pass A, pass B) and the second wall pass of a step actually READ, in CSR
 * form with caller ids: row of a fluid particle = its fluid-fluid list (the self entry included) followed by its
 * fluid-wall list; row of a wall particle = its wall-fluid list.  Entries are in list order (not sorted) and
 * include the false positives of the conservative candidate filter (reading B2: they add exactly 0).  Same
 * argument meaning as sph_debug_neighbours; all pointers HOST; synchronises.  A host-side test compares them
 * with the oracle's float32 contract lists (superset, every extra entry within the documented margin). */
int sph_debug_step_lists(sph_ctx* ctx, int64_t* offsets_host, int32_t* ids_host, int64_t cap,
                         int64_t* total_host, void* stream);

/* BASELINE.json config 4 asks for the density-reinitialisation kernel and the integrator to be timed on their own;
 * the step runs them fused with the cell hash in one predictor launch (note under the step
 * table).  This call times, on scratch outputs (the state is not changed), ms_host[0] = the stand-alone reinitialisation
 * kernel (Eq. 2.17 / 2.18 from the stored sigma_i), ms_host[1] = the stand-alone integrator (first kick Eq. 2.19, drift
 * Eq. 2.20, cell hash), ms_host[2] = the fused predictor; each the mean of 5 launches after one warm-up launch.
 * HOST pointer to 3 floats; synchronises. */
int sph_debug_time_pointwise(sph_ctx* ctx, float* ms_host, void* stream);

/* Measured non-tensor FP32 peak of the current device: a register-resident FMA loop (8 independent chains per
 * thread, 2048 threads per SM, no memory traffic), best of 4 timed launches after 2 warm-up launches, in
 * TFLOP/s (fma = 2 flop).  SURVEY.md section 8(d) "Peaks"; bench.py's roofline denominator.  Needs no context. */
int sph_debug_fma_peak(double* tflops_host, void* stream);

/* Measured roofline of the gather form: the list walk of the pair passes ("one thread per particle"
 * reading its neighbours from global memory; DESIGN.md section 5 "list walk": one coalesced 16-byte list load, four
 * 256-bit record gathers per lane) over the context's CURRENT fluid-fluid neighbour lists and records, with an empty
 * pair body, in the passes' launch configuration.  State and lists are read, never written.
 *   body_fma    0: empty pair body (every word of the record enters one XOR / ADD); > 0: a synthetic body of that many
 *               FFMAs per pair in four dependent chains on top of it, to see how a pass with as much arithmetic as the
 *               real ones (66-82 instructions per pair) would follow a cheaper walk; at most 4096;
 *   ms_host[0]  every lane gathers its own list entries: exactly the memory requests of pass A / pass B;
 *   ms_host[1]  both lanes of a lane pair gather the even lane's entry (a list merged per lane pair);
 *   ms_host[2]  the four lanes of a quad gather the first lane's entry (a list merged per quad);
 *   ms_host[3]  32 consecutive records per request (the coalesced optimum: 1 KiB from 8 cache lines);
 *   ms_host[4]  as [0], but the chunks (128 consecutive particles, one block's work) are taken in an SM-affine order:
 *               sorted by blobs of cells, every SM works through a contiguous part of that order with persistent
 *               blocks (what the plain block order costs in L1 misses; 0 if the blob key does not fit 32 bits);
 *   each the best of 3 launches after one warm-up launch, in ms.  Modes 1-3 run every lane to the warp's largest count.
 *   *requests_host (may be NULL) = warp-wide gather requests of one walk (sum over warps of the largest count).
 * HOST pointers (5 floats, one int64); synchronises; allocates and frees its own scratch.
 * Errors: SPH_EINVAL without particles or body_fma out of range, SPH_ENOMEM, SPH_ECUDA. */
int sph_debug_gather_floor(sph_ctx* ctx, int32_t body_fma, float* ms_host, int64_t* requests_host, void* stream);

/* What a warp-wide gather of 32-byte records (one 256-bit load per lane, the pair passes' request) costs in the L1 of
 * the current device as a function of the address pattern, records resident in L1; SM cycles (at the device's maximum
 * clock) per request, best of 3 launches:
 *   cycles_host[0]  32 random records of a 16 KiB window          [4]  8 records, each read by 4 adjacent lanes
 *   cycles_host[1]  32 consecutive records (8 cache lines)        [5]  one record for all 32 lanes
 *   cycles_host[2]  16 random lines, adjacent lane pairs share one [6]  32 different lines, one record of each
 *   cycles_host[3]  8 random lines, each read by 4 adjacent lanes  [7]  32 random records of a 64-record window (16 lines)
 * The L1 model of DESIGN.md section 7 rests on this table.  HOST pointer to 8 doubles; needs no context; synchronises.
 * Errors: SPH_EINVAL, SPH_ENOMEM, SPH_ECUDA. */
int sph_debug_gather_patterns(double* cycles_host, void* stream);

/* Wall normals Eq. 2.16 in caller order (n*3, zero for fluid entries); HOST pointer. */
int sph_debug_normals(sph_ctx* ctx, float* normals_host, void* stream);

/* Per-particle number density sigma_i (first n floats) and d rho/dt (next n floats) of the last
 * pass A, caller order, zero for wall entries; sigma_drho_host holds 2*n floats (HOST). */
int sph_debug_sigma(sph_ctx* ctx, float* sigma_drho_host, void* stream);

/* The cell-list sort for callers that must not allocate (code under CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the stable device radix sort of (cell id, index) that the step and the set-up
 * run (SPH_STAGE_SORT; PAPER.md:200 names the step, BASELINE.json north_star "cell hash, device radix sort"; the same
 * kernels, sph_sort.cuh), with its scratch (digit totals, tile histograms, one ping-pong pair of key / value
 * buffers) in a file-scope `static __device__` array of the library instead of buffers owned by a context.
 *
 *   keys_dev[n]      in:  keys with key_bits significant bits (1..32); not modified
 *   vals_dev[n]      in:  values carried with the keys; NULL = the indices 0..n-1 (the cell list's use); not modified
 *   keys_out_dev[n]  out: the keys in ascending order
 *   vals_out_dev[n]  out: the values in that order; equal keys keep their input order (stable)
 * All four are DEVICE pointers owned by the caller; the outputs must not overlap the inputs or each other.
 *
 * Needs no context.  Calls no cudaMalloc / cudaFree and no allocating library routine: kernel launches and one
 * cudaMemsetAsync on `stream` only; asynchronous, does not synchronise.  The first call on a device looks the array's
 * device address up (cudaGetSymbolAddress; it loads the library's module if CUDA has not done so yet).
 * Limit: n <= SPH_STATIC_SORT_MAX_KEYS = 2^20 keys (BASELINE.json configs 0-2 and config 4 at 1 M); the array is
 * 10 MiB + 2 KiB (2 KiB digit totals, 2 MiB tile histograms, 2 x 4 MiB ping-pong buffers) and every GPU that loads
 * the library holds it until the process exits.  A larger n is rejected with SPH_EINVAL and nothing is launched.
 * Every call on a device shares the one array, which keeps the previous call's contents: the call clears the
 * digit totals itself (the only part that must start at zero) and overwrites the rest before reading it.  Calls that
 * OVERLAP on the GPU (two streams, or two host threads on two streams) race on the array: order them (same
 * stream, or events).
 * Errors: SPH_EINVAL (n < 0, n > SPH_STATIC_SORT_MAX_KEYS, key_bits outside 1..32, a NULL keys / output pointer with
 * n > 0), SPH_ECUDA (no device, launch failure); sph_cell_sort_static_error() returns the text of the last failure
 * of this entry point (a static buffer: read it before another thread fails). */
enum { SPH_STATIC_SORT_MAX_KEYS = 1 << 20 };
int sph_cell_sort_static(int32_t n, const uint32_t* keys_dev, const uint32_t* vals_dev, int32_t key_bits,
                         uint32_t* keys_out_dev, uint32_t* vals_out_dev, void* stream);
const char* sph_cell_sort_static_error(void);

/* Number of kernel launches issued by the library since sph_create (bench.py's gpu_launches). */
int64_t sph_launch_count(const sph_ctx* ctx);

const char* sph_last_error(const sph_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* SPH_H_ */
