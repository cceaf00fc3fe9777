/*
 * bm.h -- C ABI of the B200-native ensemble Langevin integrator for Brownian motors
 *         (hot path of arXiv 1409.4923, Spiechowicz, Kostur, Machura).
 *
 * What one call computes: "multiple realizations of [eq. 24] have to be simulated and then
 * according to (18) an ensemble average must be performed", for many parameter values in one call
 * (PAPER.md:397).  Each realization is integrated with the jump-adapted weak-order-2.0 predictor-corrector
 * scheme (Alg. 1; jump adaptation :301) driven by Gaussian white noise (eq. 9), white
 * Poissonian noise (eq. 3-8) and dichotomous noise (eq. 13-17); the observable is eq. (30).
 * DESIGN.md section 3 lists every reading (R1..R12) taken where the paper is silent or garbled.
 *
 * Conventions
 *   - Unless a function says HOST, every data pointer is a DEVICE pointer owned by the caller (e.g. the
 *     storage of a torch tensor); the library never frees or retains it.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device-pointer
 *     calls are asynchronous on `stream`, never synchronise and keep no global mutable state.
 *   - Every call returns a bm_status; nothing throws.  There is no CPU fallback of any kind: without a
 *     CUDA device the compute calls return BM_ERR_CUDA.
 *   - Determinism: identical arguments give bit-identical outputs, independent of stream or of earlier
 *     calls.  Path g = point*n_paths + p sees the same random words whatever the grid shape is.  The default block
 *     size and the register class of the fp32 kernel (which fix the reduction tree of out_stats) are functions of the
 *     arguments only, computed for the 148 SMs of the B200 the library is built for -- on a device with another SM
 *     count the statistics are still the same bits, the choice is just no longer the tuned one.
 */
#ifndef BM_H
#define BM_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BM_VERSION 210 /* 0.2.1: bm_config.event_mode */

#if defined(__GNUC__)
#define BM_API __attribute__((visibility("default")))
#else
#define BM_API
#endif

typedef enum {
  BM_OK = 0,
  BM_ERR_INVALID_ARG = 1, /* null pointer, n <= 0, dt <= 0, n_discard >= n_steps, bad enum, ... */
  BM_ERR_UNSUPPORTED = 2, /* combination not compiled (see bm_simulate) */
  BM_ERR_WORKSPACE = 3,   /* workspace too small or misaligned */
  BM_ERR_CUDA = 4         /* a CUDA runtime call failed (no device, launch error, ...) */
} bm_status;

typedef enum { BM_OVERDAMPED = 0, BM_INERTIAL = 1 } bm_model;
typedef enum { BM_F32 = 0, BM_F64 = 1 } bm_prec;
/* fp32 only: where sin/cos/log/sqrt are evaluated.  SFU = MUFU approximations, FMA = polynomial
 * evaluation of the force cosines on the FMA pipe.  AUTO = the variant measured faster. */
typedef enum { BM_SINCOS_AUTO = 0, BM_SINCOS_SFU = 1, BM_SINCOS_FMA = 2 } bm_sincos;
/* SINE2: V = A1 sin(2 pi x) + A2 sin(4 pi x), L = 1 (BASELINE.json configs).
 * PWL:   eq. (2), scaled by A1, L = 2.      QUAD: V = A1 x^2/2 (no folding; OU pin). */
typedef enum { BM_POT_SINE2 = 0, BM_POT_PWL = 1, BM_POT_QUAD = 2 } bm_potential;
/* JUMP_ADAPTED: exact kick/flip times, Box-Muller Gaussians (the hot path).
 * PAPER_LITERAL: Alg. 2/3/4 exactly as printed (three-point increments, grid-quantised countdowns,
 * constant forces in the corrector line only); over-damped only.
 * ADAPTIVE: the jump-adapted scheme with dynamic step size control from chi = xbar_{n+1} - x_{n+1}, the difference of
 * Alg. 1's predictor and corrector (reading R14): a grid step dt is
 * covered by aligned intervals dt 2^-k, k = 0..adapt_levels; no step is rejected; the largest |chi| of an interval
 * halves the next one if above adapt_tol and doubles it if below adapt_tol/8.  BM_F64, over-damped only (else
 * BM_ERR_UNSUPPORTED); no chunked runs. */
typedef enum { BM_SCHEME_JUMP_ADAPTED = 0, BM_SCHEME_PAPER_LITERAL = 1, BM_SCHEME_ADAPTIVE = 2 } bm_scheme;
/* fp32 only: how Philox words of the Gaussian stream become Box-Muller pairs (R3, R13).
 * W32: one word per uniform (radius from w0, angle from w1, ...): four normals per call -- the oracle's assignment,
 *      so a jump-free fp32 path follows the fp64 oracle's path (common random numbers).
 * W16: radius from the top 23 bits and angle from the low 16 bits of ONE word: eight normals per call, half the
 *      integer work; the angle's sine and cosine on the SFU (MUFU.SIN, MUFU.COS).
 * W16P: the W16 assignment with the angle's sine and cosine evaluated by polynomials on the FMA pipe (two MUFU per
 *      Box-Muller pair instead of four).  AUTO = W16 (the variant measured fastest).
 * Ignored for BM_F64. */
typedef enum { BM_GAUSS_AUTO = 0, BM_GAUSS_W32 = 1, BM_GAUSS_W16 = 2, BM_GAUSS_W16P = 3 } bm_gauss;
/* BM_F32 over-damped jump-adapted kernels: how a warp steps onto the kick and flip times of its 32 paths (
 * the divergence PAPER.md:412 leaves open).  CELLS: all lanes stay in the same grid cell; a cell in which some lane has
 * an event is taken in two phases (event lanes integrate up to their events, then every lane finishes the cell).
 * LANES: per-lane clocks -- every lane advances from its own (cell, offset) to its own next event or cell boundary, one
 * sub-step per lane and pass; the warp only agrees on a sliding window of two blocks of 8 grid cells (a lane that is
 * a block ahead of the slowest one waits), so a pass costs the same however the events are spread over the lanes.
 * AUTO: per PARAMETER POINT, LANES where the expected number of events per path and grid cell exceeds 0.02 (there
 * about every second cell of a warp holds an event), else CELLS -- the measured break-even.
 * The two forms perform the same operations per path: results are bit-identical whatever the mode.  With a jump
 * source on, bm_simulate launches both forms on the same grid (each block is taken by exactly one of them). */
typedef enum { BM_EVENTS_AUTO = 0, BM_EVENTS_CELLS = 1, BM_EVENTS_LANES = 2 } bm_event_mode;
/* noise sources that are switched on; a source that is off ignores its parameters */
enum { BM_NOISE_GAUSS = 1, BM_NOISE_POISSON = 2, BM_NOISE_DICH = 4 };

/* One parameter point: 16 doubles = 128 B. */
typedef struct {
  double A1, A2;            /* potential amplitudes (see bm_potential) */
  double F;                 /* static load (f of the inertial model) */
  double D;                 /* Gaussian intensity: overdamped sqrt(2D) dW (eq. 9-10); inertial D := gamma*Q */
  double lambda, zeta;      /* Poisson rate (eq. 4) and mean amplitude (eq. 5); bias -lambda*zeta (eq. 3, 6);
                               lambda <= 0 switches the source off at this point */
  double Fa, Fb;            /* dichotomous values -Fa, +Fb (eq. 13), both > 0 */
  double mu_a, mu_b;        /* rate of leaving -Fa, rate of leaving +Fb (eq. 14).  mu_a <= 0 switches the source off at
                               this point (Gamma = 0); mu_b <= 0 with mu_a > 0 makes +Fb absorbing */
  double gamma, amp, omega; /* inertial: friction, drive amplitude, drive angular frequency.  BM_F64: the drive cosine is
                               the kernel's own, accurate for |omega * t_final| < 2^20 (1.3e4 at the end of C3); beyond
                               that its argument reduction loses bits (not checked) */
  double x0_fixed;          /* >= 0: x0 = x0_fixed; < 0: x0 ~ U[0,L) */
  double v0_lo, v0_hi;      /* inertial: v0 ~ U[v0_lo, v0_hi] */
} bm_params;

/* Per-point result: 8 doubles = 64 B.  Variances are unbiased (divide by n-1). */
typedef struct {
  double n;             /* paths averaged */
  double mean_v, var_v; /* vbar_p = (x_p(t_f) - x_p(t_i))/(t_f - t_i), eq. (30); t_i = n_discard*dt */
  double mean_xT, var_xT; /* unfolded x_p(t_f) */
  double mean_jumps;    /* kicks + flips per path */
  double mean_substeps; /* predictor-corrector sub-steps per path (= n_steps + events inside grid cells) */
  double rsv;
} bm_stats;

typedef struct {
  int32_t model;       /* bm_model */
  int32_t prec;        /* bm_prec */
  int32_t sincos;      /* bm_sincos */
  int32_t potential;   /* bm_potential */
  int32_t scheme;      /* bm_scheme */
  int32_t noise;       /* OR of BM_NOISE_* */
  int32_t block_threads; /* 0 = library default (a function of the arguments only, see bm_kernel_info); else a
                            multiple of 32 in [32,256], up to 512 for the BM_F32 over-damped jump-adapted kernel.  Part
                            of the determinism contract (it fixes the reduction tree). */
  int32_t gauss;       /* bm_gauss (BM_F32 only) */
  int64_t n_discard;   /* grid steps before t_i, 0 <= n_discard < n_steps (PAPER.md:423 uses n_steps/10) */
  int64_t trace_steps; /* with out_trace: record the first trace_steps grid steps ... */
  int64_t trace_paths; /* ... of global paths 0..trace_paths-1 (BM_F64 only) */
  int32_t paths_per_thread; /* BM_F64 jump-adapted kernels: realizations carried by one thread.  0 = library default
                            (1: the measured-faster form); 1; 2
                            (BM_POT_SINE2 only, else BM_ERR_UNSUPPORTED; two independent chains per thread measured
                            slower at the BASELINE ensemble sizes and ships for ensembles below one warp per scheduler,
                            where it is the only way to fill the FP64 pipe).  A path's result does not depend on it; it
                            enters the determinism contract through the reduction tree of out_stats only.  Must be 0
                            for BM_F32, the paper-literal and the adaptive scheme (else BM_ERR_UNSUPPORTED). */
  int32_t adapt_levels; /* BM_SCHEME_ADAPTIVE: how often dt may be halved, 0..20 */
  double adapt_tol;    /* BM_SCHEME_ADAPTIVE: tolerance on |chi| (in units of x), >= 0; +inf = never refine */
  int32_t event_mode;  /* bm_event_mode; must be AUTO unless BM_F32, BM_OVERDAMPED, JUMP_ADAPTED with a jump source in
                          `noise` (else BM_ERR_UNSUPPORTED) */
  int32_t rsv;         /* must be 0 (else BM_ERR_INVALID_ARG) */
} bm_config;

/* per-path record written to out_paths: 6 doubles */
enum { BM_OUT_XT = 0, BM_OUT_VT = 1, BM_OUT_VBAR = 2, BM_OUT_JUMPS = 3, BM_OUT_SUBSTEPS = 4, BM_OUT_XTI = 5,
       BM_OUT_STRIDE = 6 };

/* Bytes of device scratch bm_simulate needs (per-block partial sums of the two-level reduction).
 * Returns 0 on invalid arguments. */
BM_API size_t bm_workspace_bytes(const bm_config *cfg, int32_t n_points, int64_t n_paths);

/*
 * Simulate n_points x n_paths realizations for n_steps grid steps of length dt and reduce them.
 *   params     [n_points]               device, read only
 *   out_stats  [n_points]               device, written
 *   out_paths  [n_points*n_paths][6]    device, optional (NULL to skip): BM_OUT_* per path, index g
 *   out_trace  [trace_paths][trace_steps][2] device, optional: (x unfolded, v) after each grid step
 *   workspace  device scratch of >= bm_workspace_bytes(...) bytes, 16-byte aligned
 * Kernels launched on `stream`: the path kernel (a1-a10 of DESIGN.md section 2) and the grid pass of the
 * reduction (a11).  n_steps <= 2^31 - 16 for BM_F32 (32-bit cell counters), <= 2^33 for BM_F64 (the Gaussian stream is
 * indexed by a 32-bit counter word that advances once per four sub-steps: grid steps + events must stay below 2^34);
 * BM_SCHEME_ADAPTIVE: n_steps * 2^adapt_levels <= 2^33 (every grid step may be refined to the last level).  Parameter VALUES are not checked here (params is a device pointer; see
 * bm_simulate_host).  Errors: BM_ERR_INVALID_ARG as listed above; BM_ERR_UNSUPPORTED for
 * PAPER_LITERAL with BM_INERTIAL, BM_INERTIAL with a potential other than SINE2, out_trace with BM_F32;
 * BM_ERR_WORKSPACE; BM_ERR_CUDA.
 */
BM_API bm_status bm_simulate(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                      int64_t n_steps, double dt, uint64_t seed, bm_stats *out_stats, double *out_paths,
                      double *out_trace, void *workspace, size_t workspace_bytes, void *stream);

/*
 * bm_simulate with one step length per parameter point ("per-point dt"; the paper fixes the step
 * as a number of steps per characteristic time, dt = tau_char / spp, so a sweep over the noise parameters
 * is a sweep over dt).  dt_points [n_points] device, read only, each > 0 (not checked on the device: a non-positive
 * entry gives NaN statistics for that point).  Everything else as bm_simulate; no trace output.
 */
BM_API bm_status bm_simulate_dt(const bm_config *cfg, const bm_params *params, const double *dt_points, int32_t n_points,
                         int64_t n_paths, int64_t n_steps, uint64_t seed, bm_stats *out_stats, double *out_paths,
                         void *workspace, size_t workspace_bytes, void *stream);

/*
 * Chunked runs and checkpoint / resume (Alg. 5 steps 2 and 6: "load the state
 * ... advance `samples` steps ... save the state").  bm_simulate_chunk performs grid steps
 * [step_begin, step_begin + step_count) of a run of n_steps steps.  step_begin == 0 initialises the paths (the
 * contents of `state` are ignored); any other chunk continues from `state` as the previous chunk left it.  Every chunk
 * rewrites `state`; the chunk that reaches n_steps also writes out_stats (and out_paths, if given) -- for the other
 * chunks they are not touched.  A run cut into chunks gives bit-identical results to the single bm_simulate call
 * with the same arguments.  The Philox generator is stateless, so the state of a path is its position, clocks,
 * counters and snapshot: BM_STATE_SLOTS 8-byte words per path, slot-major ([slot][n_points*n_paths], coalesced).
 *   state      device, >= bm_state_bytes(...) bytes, 16-byte aligned; owned by the caller, may be copied to the host
 *              and back between chunks (that is the checkpoint)
 * step_begin, and step_begin + step_count unless it equals n_steps, must be multiples of BM_CHUNK_ALIGN.  All other
 * arguments as bm_simulate and the same in every chunk of a run (not checked).  No trace output in chunked runs.
 * Errors: as bm_simulate; BM_ERR_INVALID_ARG for a misaligned or out-of-range chunk or a null / misaligned state;
 * BM_ERR_WORKSPACE for a state buffer that is too small.
 */
enum { BM_STATE_SLOTS = 16, BM_CHUNK_ALIGN = 8 };
BM_API size_t bm_state_bytes(const bm_config *cfg, int32_t n_points, int64_t n_paths);
BM_API bm_status bm_simulate_chunk(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                            int64_t n_steps, double dt, uint64_t seed, int64_t step_begin, int64_t step_count,
                            void *state, size_t state_bytes, bm_stats *out_stats, double *out_paths, void *workspace,
                            size_t workspace_bytes, void *stream);

/*
 * More observables from the same pass: the stationary density p(x mod L) of eq. (19),
 * PAPER.md:183, as a histogram.  Adds, for every path of the checkpoint `state` (as bm_simulate_chunk left it), one
 * count to counts[point][bin], bin = floor(n_bins * frac(x / L)): called after every chunk of a chunked run it
 * accumulates the occupation of the reduced coordinate at the chunk boundaries t = k * chunk * dt.  Integer counts
 * (device, uint64 [n_points][n_bins], zeroed by the caller): independent of the order of accumulation.
 * Errors: BM_ERR_INVALID_ARG (null / misaligned pointers, n_bins outside [1, 4096]); BM_ERR_UNSUPPORTED for
 * BM_POT_QUAD (no period); BM_ERR_WORKSPACE for a state buffer smaller than bm_state_bytes(...).
 */
BM_API bm_status bm_state_histogram(const bm_config *cfg, int32_t n_points, int64_t n_paths, const void *state,
                             size_t state_bytes, int32_t n_bins, uint64_t *counts, void *stream);

/*
 * Effective diffusion and velocity autocorrelation (the stationary state of eq. 18-19,
 * PAPER.md:176-183): per-point ensemble moments of the checkpoint `state` (as bm_simulate_chunk left it at time t),
 * optionally against `ref_state`, a copy of the checkpoint of the SAME run at an earlier time t0 (NULL: the entries
 * that need it are 0).  out [n_points][BM_MOM_STRIDE] doubles, device:
 *   N, MEAN_X, VAR_X (unfolded x(t)), MEAN_V, VAR_V (v(t); 0 for the over-damped model),
 *   MEAN_DX, VAR_DX of x(t) - x(t0):  D_eff(t - t0) = VAR_DX / (2 (t - t0)),
 *   COV_V0V = <v(t0) v(t)> - <v(t0)><v(t)>,  VAR_V0 = Var v(t0).            Variances divide by n-1.
 * One block per point, two passes in a fixed order: bit-reproducible.  Called between the chunks of a chunked run it
 * gives D_eff(t) and the velocity autocorrelation function without touching the path kernels (whose state stays in
 * registers); DESIGN.md section 6 has the measured cost of a chunk boundary.
 * Errors: BM_ERR_INVALID_ARG (null / misaligned pointers), BM_ERR_WORKSPACE (state smaller than bm_state_bytes(...)).
 */
enum { BM_MOM_N = 0, BM_MOM_MEAN_X = 1, BM_MOM_VAR_X = 2, BM_MOM_MEAN_V = 3, BM_MOM_VAR_V = 4, BM_MOM_MEAN_DX = 5,
       BM_MOM_VAR_DX = 6, BM_MOM_COV_V0V = 7, BM_MOM_VAR_V0 = 8, BM_MOM_STRIDE = 10 };
BM_API bm_status bm_state_moments(const bm_config *cfg, int32_t n_points, int64_t n_paths, const void *state, size_t state_bytes,
                           const void *ref_state, double *out, void *stream);

/*
 * HOST-pointer convenience entry (the end-to-end path): params, out_stats and out_paths (optional) are HOST
 * buffers.  Takes device scratch from a private stream-ordered pool (one per device, kept between calls: an
 * allocation cache with no influence on results), copies params in, runs bm_simulate on `stream`, copies the
 * results out, returns the scratch to the pool and synchronises the stream.  With the parameter values in view it also
 * resolves BM_EVENTS_AUTO to one form when all points fall on the same side of the break-even (one launch less; the
 * results do not depend on the form).  May be called from several host threads
 * (the pool table is guarded by a mutex; calls on the same stream serialise on that stream as usual).
 * Having the values on the host, it also checks them: BM_ERR_INVALID_ARG for a non-finite entry, a negative D, lambda,
 * mu_a, mu_b or gamma, zeta <= 0 where lambda > 0, Fa <= 0 or Fb <= 0 where mu_a > 0, v0_hi < v0_lo -- for the sources
 * cfg->noise switches on and the model cfg->model selects.
 */
BM_API bm_status bm_simulate_host(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                           int64_t n_steps, double dt, uint64_t seed, bm_stats *out_stats, double *out_paths,
                           void *stream);

/*
 * bm_simulate for callers that cannot allocate device memory.  bm_simulate asks the caller for `workspace`; this entry
 * takes none.  It is meant for code that has no allocator to call: a plug-in inside an application that owns the GPU
 * heap, a real-time loop where cudaMalloc (which may synchronise the device and has no time bound) is off limits, a
 * process whose device memory is already fully committed.  The scratch is a fixed array of BM_STATIC_SCRATCH_BYTES
 * inside the library's device image: every GPU on which libbm.so is loaded holds those 4 MiB from module load until the
 * process exits, used or not.  The call performs no cudaMalloc, cudaFree, pool or other allocating routine.
 *   Arguments, outputs, errors and results: exactly bm_simulate's (same kernels, same reduction tree, bit-identical
 *   out_stats / out_paths / out_trace); params, out_* are DEVICE pointers the caller owns, as there.
 *   Limit: bm_workspace_bytes(cfg, n_points, n_paths) <= BM_STATIC_SCRATCH_BYTES, i.e. at most 65 536 thread blocks
 *   (n_points x ceil(n_paths / block size)); beyond it the call returns BM_ERR_WORKSPACE and launches nothing.
 *   First call on a device: looks up the array's device address (cudaGetSymbolAddress, with the calling thread's current
 *   device) and keeps it; make that first call outside any stream capture.  Later calls on that device skip the look-up.
 *   Sharing: all calls on one device use the same array, and it keeps whatever the last call wrote.  Nothing in it needs
 *   clearing (each call overwrites every slot it later reads), but two calls that may run on the GPU at the same time --
 *   different streams, or different host threads without ordering between their streams -- race on it and corrupt each
 *   other's statistics.  Keep calls on one device in one stream, or order them with events.  bm_simulate with
 *   caller-owned workspaces has no such restriction.
 */
enum { BM_STATIC_SCRATCH_BYTES = 4 * 1024 * 1024 };
BM_API bm_status bm_simulate_static(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                             int64_t n_steps, double dt, uint64_t seed, bm_stats *out_stats, double *out_paths,
                             double *out_trace, void *stream);

/* Raw Philox4x32-10 words (R1, R2): out[p][j][0..3] = call (seed, g = path0+p, stream_id, idx = idx0+j). */
BM_API bm_status bm_philox_fill(uint64_t seed, uint64_t path0, int32_t n_paths, uint32_t stream_id, uint32_t idx0,
                         int32_t n_idx, uint32_t *out, void *stream);

/* Standard normals of the Gaussian stream (R3): out[p][j] = Gaussian number m0+j of path path0+p, produced by
 * exactly the device code the path kernels use.  prec BM_F64: out is double*; BM_F32: out is float* and `gauss`
 * (bm_gauss; AUTO = W16) selects the assignment.  m0 must be a multiple of 8. */
BM_API bm_status bm_gauss_fill(int32_t prec, int32_t gauss, uint64_t seed, uint64_t path0, int32_t n_paths, uint64_t m0,
                        int32_t n_m, void *out, void *stream);

/* The variate transform alone (a4; eq. 27, reading R3) on GIVEN words, for its edge cases (u next to 0 and
 * to 1, angles on the quadrant boundaries), which the Philox stream only reaches by chance: out[2i], out[2i+1] = the
 * Box-Muller pair of (words[2i], words[2i+1]) -- radius from the first word, angle from the second -- by the device code
 * of the path kernels.  prec BM_F64: out is double*; BM_F32: float*, the W32 assignment.  words, out: device, 8- and
 * 16-byte aligned.  Errors: BM_ERR_INVALID_ARG. */
BM_API bm_status bm_box_muller_words(int32_t prec, const uint32_t *words, int32_t n_pairs, void *out, void *stream);

/* The normal of a sub-step that ENDS ON AN EVENT in the BM_F32 kernels (reading R13; the jump adaptation of
 * PAPER.md:301 cuts a grid step at a kick or flip, and the piece before it needs its own Gaussian increment, eq. 9): it
 * comes from word 2 of the event's own Philox call (call k of the Poisson or dichotomous stream: bm_philox_fill with
 * stream_id 2 or 3), radius from the word's top 23 bits, angle from its low 16.  No Gaussian-stream fill reaches that
 * code, so this call applies it to GIVEN words: out[i] = the normal of words[i].  words, out: device, n > 0.
 * Errors: BM_ERR_INVALID_ARG. */
BM_API bm_status bm_event_normal_words(const uint32_t *words, int32_t n, float *out, void *stream);

/* Registers per thread, threads per block, resident blocks per SM, SM count and the Gaussian assignment selected
 * (bm_gauss, never AUTO; 0 for BM_F64), for the path kernel bm_simulate would launch for (cfg, n_points, n_paths)
 * (measurement aid; HOST outputs, each may be NULL).  Where bm_simulate launches both event forms (BM_EVENTS_AUTO with
 * a jump source on), the figures are those of the CELLS form; set cfg->event_mode = BM_EVENTS_LANES to get the
 * per-lane-clock form's. */
BM_API bm_status bm_kernel_info(const bm_config *cfg, int32_t n_points, int64_t n_paths, int32_t *regs_per_thread,
                         int32_t *launch_threads, int32_t *blocks_per_sm, int32_t *sm_count, int32_t *gauss);

/* Pipe-throughput probes used by bench.py for the "alu" roofline: launches a kernel
 * of `blocks` x `threads` threads each issuing iters x 64 dependent-chain-free operations of kind `op`
 * (BM_PROBE_*); `sink` is a device buffer of >= blocks*threads floats.  The caller times it with CUDA events. */
enum { BM_PROBE_FFMA = 0, BM_PROBE_MUFU_COS = 1, BM_PROBE_MUFU_LG2 = 2, BM_PROBE_MUFU_SQRT = 3, BM_PROBE_IMAD_WIDE = 4,
       BM_PROBE_LOP3 = 5, BM_PROBE_DFMA = 6, BM_PROBE_I2F = 7, BM_PROBE_FADD = 8, BM_PROBE_MIX = 9,
       BM_PROBE_COUNT = 10 };
BM_API bm_status bm_pipe_probe(int32_t op, int32_t iters, int32_t blocks, int32_t threads, float *sink, void *stream);

BM_API const char *bm_status_string(bm_status s);
BM_API int bm_version(void);

#ifdef __cplusplus
}
#endif
#endif
