// api.cu -- the C ABI of include/bm.h: argument validation, kernel selection, launches.  No compute here.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "dispatch.cuh"

using namespace bm;

namespace {

constexpr int DEFAULT_BLOCK_F32 = 128;

PhiloxKeys make_keys(uint64_t seed) {
  PhiloxKeys K;
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) {
    K.k0[r] = k0;
    K.k1[r] = k1;
    k0 += PHILOX_W0;
    k1 += PHILOX_W1;
  }
  return K;
}

bool valid_cfg(const bm_config *c) {
  if (!c) return false;
  if (c->model != BM_OVERDAMPED && c->model != BM_INERTIAL) return false;
  if (c->prec != BM_F32 && c->prec != BM_F64) return false;
  if (c->sincos < BM_SINCOS_AUTO || c->sincos > BM_SINCOS_FMA) return false;
  if (c->potential < BM_POT_SINE2 || c->potential > BM_POT_QUAD) return false;
  if (c->scheme != BM_SCHEME_JUMP_ADAPTED && c->scheme != BM_SCHEME_PAPER_LITERAL && c->scheme != BM_SCHEME_ADAPTIVE) return false;
  if (c->scheme == BM_SCHEME_ADAPTIVE && (c->adapt_levels < 0 || c->adapt_levels > 20 || !(c->adapt_tol >= 0.0))) return false;
  if (c->noise < 0 || c->noise > 7) return false;
  if (c->block_threads != 0 && (c->block_threads < 32 || c->block_threads > 512 || (c->block_threads & 31))) return false;
  if (c->block_threads > 256 && !(c->prec == BM_F32 && c->model == BM_OVERDAMPED && c->scheme == BM_SCHEME_JUMP_ADAPTED)) return false;
  if (c->gauss < BM_GAUSS_AUTO || c->gauss > BM_GAUSS_W16P) return false;
  if (c->paths_per_thread < 0 || c->paths_per_thread > 2) return false;
  if (c->rsv != 0) return false;  // bm.h: reserved, must be 0
  if (c->n_discard < 0 || c->trace_steps < 0 || c->trace_paths < 0) return false;
  if (c->event_mode < BM_EVENTS_AUTO || c->event_mode > BM_EVENTS_LANES) return false;
  return true;
}

// Default block size: a function of the arguments only (the block size fixes the reduction tree, so it must not
// depend on the device the call happens to run on; the library is built for the 148-SM B200).  Among 128, 256
// and 512 threads (512: fp32 over-damped jump-adapted kernel only) the size that leaves the busiest SM scheduler with the
// fewest warps, ties to the larger block: the warps of one block run in phase and share the instruction stream
// (C1: 2.91 / 2.80 / 2.65 ms per 20 000 steps at 128 / 256 / 512).  Beyond 8 warps per scheduler
// the block size stops mattering and 128 is kept.
constexpr int DESIGN_SMS = 148;
int max_block_threads(const bm_config *c) {
  return (c->prec == BM_F32 && c->model == BM_OVERDAMPED && c->scheme == BM_SCHEME_JUMP_ADAPTED) ? 512 : 256;
}
int paths_per_thread_of(const bm_config *c, int32_t n_points, int64_t n_paths);
int block_threads_of(const bm_config *c, int32_t n_points, int64_t n_paths) {
  if (c->block_threads) return c->block_threads;
  int best = DEFAULT_BLOCK_F32;
  long long best_cost = -1;
  const int ppt = paths_per_thread_of(c, n_points, n_paths);
  for (int bt = 128; bt <= max_block_threads(c); bt *= 2) {
    const long long blocks = (long long)n_points * ((n_paths + (long long)bt * ppt - 1) / ((long long)bt * ppt));
    const long long cost = ((blocks + DESIGN_SMS - 1) / DESIGN_SMS) * (bt / 128);  // warps on the busiest scheduler
    if (best_cost < 0 || cost <= best_cost) { best = bt; best_cost = cost; }
  }
  return best_cost > 8 ? DEFAULT_BLOCK_F32 : best;
}

// Realizations per thread of the fp64 jump-adapted kernels (sim_f64.cuh).  Two per thread exist for the smooth
// potential as a measured choice; AUTO is one: with a fixed ensemble two chains per thread only trade warps for
// chains (C1 131.8 ms against 103.5, C2 404.8 against 283.9).
bool has_two_paths(const bm_config *c) {
  return c->prec == BM_F64 && c->scheme == BM_SCHEME_JUMP_ADAPTED && c->potential == BM_POT_SINE2;
}
int paths_per_thread_of(const bm_config *c, int32_t n_points, int64_t n_paths) {
  if (!has_two_paths(c)) return 1;
  (void)n_points; (void)n_paths;
  return c->paths_per_thread ? c->paths_per_thread : 1;
}

int resolve_sincos(const bm_config *c) {
  // AUTO: the SFU variant measured faster on B200 for every config
  return c->sincos == BM_SINCOS_FMA ? BM_SINCOS_FMA : BM_SINCOS_SFU;
}

int resolve_gauss(const bm_config *c) {
  // AUTO: eight normals per Philox call with the Box-Muller angle on the SFU: W16 and W16P measure within 1 % of
  // each other on the over-damped configs, W16 is 3-4 % faster on the inertial ones
  return c->gauss == BM_GAUSS_AUTO ? BM_GAUSS_W16 : c->gauss;
}

struct Launch {
  KernelFn fn = nullptr;
  int threads = 0;  // threads per block
  int gauss = 0;    // bm_gauss selected (fp32), 0 for fp64
  int ppt = 1;      // realizations per thread (fp64 jump-adapted kernels)
  size_t smem = 0;  // dynamic shared memory per block (event rings of the fp32 jump-adapted kernel)
  // fp32 over-damped kernels with a jump source: the per-lane-clock form, launched on the same grid (every block is
  // taken by exactly one of the two, by the event mode of its parameter point); fn is null when LANES is forced
  KernelFn fn_lanes = nullptr;
  size_t smem_lanes = 0;
};

bool has_event_modes(const bm_config *c) {
  return c->prec == BM_F32 && c->model == BM_OVERDAMPED && c->scheme == BM_SCHEME_JUMP_ADAPTED &&
         (c->noise & (BM_NOISE_POISSON | BM_NOISE_DICH));
}

bm_status opt_in_smem(KernelFn fn, size_t smem) {
  // beyond the 48 KB default a kernel has to opt in (per function and device; repeating the call is harmless)
  if (smem > 44 * 1024 &&  /* the kernels also hold 1792 B of static shared memory (block reduction) */
      cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
    cudaGetLastError();
    return BM_ERR_CUDA;
  }
  return BM_OK;
}

bm_status pick_kernel(const bm_config *c, int32_t n_points, int64_t n_paths, Launch *L, bool chunked = false) {
  *L = Launch();
  if (c->scheme == BM_SCHEME_PAPER_LITERAL && c->model != BM_OVERDAMPED) return BM_ERR_UNSUPPORTED;
  if (c->scheme == BM_SCHEME_ADAPTIVE && (c->model != BM_OVERDAMPED || c->prec != BM_F64 || chunked)) return BM_ERR_UNSUPPORTED;
  if (c->model == BM_INERTIAL && c->potential != BM_POT_SINE2) return BM_ERR_UNSUPPORTED;
  if (c->paths_per_thread == 2 && !has_two_paths(c)) return BM_ERR_UNSUPPORTED;
  // bm.h: a knob of the BM_F64 jump-adapted kernels only; it must be 0 everywhere else
  if (c->paths_per_thread != 0 && !(c->prec == BM_F64 && c->scheme == BM_SCHEME_JUMP_ADAPTED)) return BM_ERR_UNSUPPORTED;
  if (c->event_mode != BM_EVENTS_AUTO && !has_event_modes(c)) return BM_ERR_UNSUPPORTED;
  L->threads = block_threads_of(c, n_points, n_paths);
  L->ppt = paths_per_thread_of(c, n_points, n_paths);
  if (c->scheme == BM_SCHEME_PAPER_LITERAL) {
    L->fn = pick_literal(c->prec, c->potential, c->noise);
  } else if (c->scheme == BM_SCHEME_ADAPTIVE) {
    L->fn = pick_adaptive_f64(c->potential, c->noise);
  } else if (c->prec == BM_F64) {
    L->fn = c->model == BM_OVERDAMPED ? pick_f64_overdamped(c->potential, c->noise, chunked, L->ppt)
                                      : pick_f64_inertial(c->potential, c->noise, chunked, L->ppt);
  } else {
    typedef KernelFn (*Picker)(int, int, int, int);
    static const Picker table[2][2][3] = {  // [model][sincos fma][gauss - 1]
        {{pick_f32_od_sfu_w32, pick_f32_od_sfu_w16, pick_f32_od_sfu_w16p},
         {pick_f32_od_fma_w32, pick_f32_od_fma_w16, pick_f32_od_fma_w16p}},
        {{pick_f32_in_sfu_w32, pick_f32_in_sfu_w16, pick_f32_in_sfu_w16p},
         {pick_f32_in_fma_w32, pick_f32_in_fma_w16, pick_f32_in_fma_w16p}}};
    L->gauss = resolve_gauss(c);
    // register class of the over-damped kernel: 64 registers once the grid is more than the ~95-register form can
    // keep resident (5 blocks of 128 threads per SM); a function of the arguments only
    const long long threads_total = (long long)n_points * ((n_paths + L->threads - 1) / L->threads) * L->threads;
    const int occ = threads_total > (long long)DESIGN_SMS * 640 ? 1 : 0;
    const Picker pick = table[c->model == BM_INERTIAL][resolve_sincos(c) == BM_SINCOS_FMA][L->gauss - 1];
    if (!has_event_modes(c) || c->event_mode != BM_EVENTS_LANES) {
      L->fn = pick(c->potential, c->noise, occ, 0);
      L->smem = (size_t)L->threads * sizeof(uint32_t) * (size_t)f32_smem_words_per_thread(c->noise, L->gauss);
      if (!L->fn) return BM_ERR_UNSUPPORTED;
    }
    if (has_event_modes(c) && c->event_mode != BM_EVENTS_CELLS) {
      L->fn_lanes = pick(c->potential, c->noise, occ, 1);
      L->smem_lanes = (size_t)L->threads * sizeof(uint32_t) * (size_t)f32_smem_words_per_thread(c->noise, L->gauss, 1);
      if (!L->fn_lanes) return BM_ERR_UNSUPPORTED;
    }
  }
  if (!L->fn && !L->fn_lanes) return BM_ERR_UNSUPPORTED;
  if (L->fn && opt_in_smem(L->fn, L->smem) != BM_OK) return BM_ERR_CUDA;
  if (L->fn_lanes && opt_in_smem(L->fn_lanes, L->smem_lanes) != BM_OK) return BM_ERR_CUDA;
  return BM_OK;
}

// Scratch pool of the HOST-pointer entry: one private stream-ordered pool per device that keeps its blocks between
// calls (release threshold = never), so that only the first call pays for device allocations.  A cache only: it has
// no influence on any result.
cudaMemPool_t host_entry_pool() {
  static cudaMemPool_t pools[64] = {};
  static std::mutex guard;  // the HOST entry may be called from several host threads at once
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return nullptr;
  std::lock_guard<std::mutex> lock(guard);
  if (!pools[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t pool = nullptr;
    if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    unsigned long long keep = ~0ULL;
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    pools[dev] = pool;
  }
  return pools[dev];
}

// Parameter values as SURVEY.md s.8(b) lists them for BM_ERR_INVALID_ARG.  Only the HOST entry can check them (the
// device-pointer calls never read `params` on the host): finite numbers, no negative rate or intensity, positive
// amplitudes of a source that is switched on.
bool valid_params_host(const bm_config *c, const bm_params *p, int32_t n_points) {
  for (int32_t i = 0; i < n_points; ++i) {
    const bm_params &q = p[i];
    const double all[16] = {q.A1, q.A2, q.F, q.D, q.lambda, q.zeta, q.Fa, q.Fb, q.mu_a, q.mu_b, q.gamma, q.amp, q.omega,
                            q.x0_fixed, q.v0_lo, q.v0_hi};
    for (double v : all)
      if (!std::isfinite(v)) return false;
    if ((c->noise & BM_NOISE_GAUSS) && q.D < 0.0) return false;
    if ((c->noise & BM_NOISE_POISSON) && (q.lambda < 0.0 || (q.lambda > 0.0 && !(q.zeta > 0.0)))) return false;
    if ((c->noise & BM_NOISE_DICH) && (q.mu_a < 0.0 || q.mu_b < 0.0 || (q.mu_a > 0.0 && (!(q.Fa > 0.0) || !(q.Fb > 0.0))))) return false;
    if (c->model == BM_INERTIAL && (q.gamma < 0.0 || q.v0_hi < q.v0_lo)) return false;
  }
  return true;
}

// BM_EVENTS_AUTO with the parameter values on the host: when every point of the table falls on the same side of the
// break-even (the expression of lane_clock_point, common.cuh), the other form's launch would find no block to take --
// name the form and save the launch.  Results do not depend on the mode (bit-identical by construction and by test).
int resolve_event_mode_host(const bm_config *c, const bm_params *p, int32_t n_points, double dt) {
  if (!has_event_modes(c) || c->event_mode != BM_EVENTS_AUTO) return c->event_mode;
  bool any_lanes = false, any_cells = false;
  for (int32_t i = 0; i < n_points; ++i) {
    double rate = 0.0;
    if ((c->noise & BM_NOISE_POISSON) && p[i].lambda > 0.0) rate += p[i].lambda;
    if ((c->noise & BM_NOISE_DICH) && p[i].mu_a > 0.0) rate += 0.5 * (p[i].mu_a + (p[i].mu_b > 0.0 ? p[i].mu_b : 0.0));
    (rate * dt > LCLK_EVENTS_PER_CELL ? any_lanes : any_cells) = true;
  }
  return any_lanes == any_cells ? BM_EVENTS_AUTO : (any_lanes ? BM_EVENTS_LANES : BM_EVENTS_CELLS);
}

long long blocks_per_point_of(const bm_config *c, int32_t n_points, int64_t n_paths) {
  const long long per_block = (long long)block_threads_of(c, n_points, n_paths) * paths_per_thread_of(c, n_points, n_paths);
  return (n_paths + per_block - 1) / per_block;
}

}  // namespace

extern "C" {

BM_API int bm_version(void) { return BM_VERSION; }

BM_API const char *bm_status_string(bm_status s) {
  switch (s) {
    case BM_OK: return "BM_OK";
    case BM_ERR_INVALID_ARG: return "BM_ERR_INVALID_ARG";
    case BM_ERR_UNSUPPORTED: return "BM_ERR_UNSUPPORTED";
    case BM_ERR_WORKSPACE: return "BM_ERR_WORKSPACE";
    case BM_ERR_CUDA: return "BM_ERR_CUDA";
    default: return "BM_ERR_UNKNOWN";
  }
}

BM_API size_t bm_workspace_bytes(const bm_config *cfg, int32_t n_points, int64_t n_paths) {
  if (!valid_cfg(cfg) || n_points <= 0 || n_paths <= 0) return 0;
  const long long bpp = blocks_per_point_of(cfg, n_points, n_paths);
  const long long grid = bpp * (long long)n_points;
  if (grid > 0x7FFFFFFFLL) return 0;
  return (size_t)grid * PARTIAL_STRIDE * sizeof(double);
}

// the launch behind bm_simulate (state == nullptr: the whole run) and bm_simulate_chunk
static bm_status simulate_range(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                                int64_t n_steps, double dt, const double *dt_points, uint64_t seed, int64_t step_begin,
                                int64_t step_end,
                                void *state, bm_stats *out_stats, double *out_paths, double *out_trace, void *workspace,
                                size_t workspace_bytes, void *stream) {
  if (!valid_cfg(cfg) || !params || !out_stats || n_points <= 0 || n_paths <= 0 || n_steps <= 0) return BM_ERR_INVALID_ARG;
  if (!(dt > 0.0) || !(dt < 1e300)) return BM_ERR_INVALID_ARG;
  if (cfg->n_discard >= n_steps) return BM_ERR_INVALID_ARG;
  // step and draw counters: the fp32 kernels count grid cells in 32 bits; the fp64 kernels index the Gaussian stream
  // by (sub-step count)/4 in a 32-bit counter word (sub-steps = grid steps + events < 2^34)
  const bool narrow = cfg->prec == BM_F32;
  if (n_steps > (narrow ? 0x7FFFFFF0LL : (1LL << 33))) return BM_ERR_INVALID_ARG;
  // the adaptive scheme may take 2^adapt_levels sub-steps per grid step: the same counter bounds the refined count
  if (cfg->scheme == BM_SCHEME_ADAPTIVE && n_steps > ((1LL << 33) >> cfg->adapt_levels)) return BM_ERR_INVALID_ARG;
  if (out_trace && (cfg->trace_steps <= 0 || cfg->trace_paths <= 0)) return BM_ERR_INVALID_ARG;
  if (out_trace && cfg->prec != BM_F64) return BM_ERR_UNSUPPORTED;
  Launch L;
  const bm_status ps = pick_kernel(cfg, n_points, n_paths, &L, state != nullptr);
  if (ps != BM_OK) return ps;
  const size_t need = bm_workspace_bytes(cfg, n_points, n_paths);
  if (need == 0) return BM_ERR_INVALID_ARG;
  if (!workspace || workspace_bytes < need || ((uintptr_t)workspace & 15)) return BM_ERR_WORKSPACE;

  SimArgs a;
  memset(&a, 0, sizeof(a));
  a.params = params;
  a.partials = reinterpret_cast<double *>(workspace);
  a.out_paths = out_paths;
  a.out_trace = out_trace;
  a.n_paths = n_paths;
  a.n_steps = n_steps;
  a.n_discard = cfg->n_discard;
  a.trace_steps = out_trace ? cfg->trace_steps : 0;
  a.trace_paths = out_trace ? cfg->trace_paths : 0;
  a.dt = dt;
  a.dt_points = dt_points;
  a.n_points = n_points;
  a.blocks_per_point = (int)blocks_per_point_of(cfg, n_points, n_paths);
  a.state = reinterpret_cast<unsigned long long *>(state);
  a.step_begin = step_begin;
  a.step_end = step_end;
  a.adapt_tol = cfg->adapt_tol;
  a.adapt_levels = cfg->adapt_levels;
  a.event_mode = cfg->event_mode;
  a.keys = make_keys(seed);

  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const unsigned grid = (unsigned)((long long)a.blocks_per_point * n_points);
  if (L.fn) L.fn<<<grid, L.threads, L.smem, st>>>(a);  // a1: (point x path) -> grid
  if (L.fn_lanes) L.fn_lanes<<<grid, L.threads, L.smem_lanes, st>>>(a);
  if (cudaGetLastError() != cudaSuccess) return BM_ERR_CUDA;
  if (step_end < n_steps) return BM_OK;  // the ensemble reduction belongs to the last chunk
  if (launch_grid_reduce(a.partials, n_points, a.blocks_per_point, out_stats, st) != cudaSuccess) return BM_ERR_CUDA;
  return BM_OK;
}

BM_API bm_status bm_simulate(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                      int64_t n_steps, double dt, uint64_t seed, bm_stats *out_stats, double *out_paths,
                      double *out_trace, void *workspace, size_t workspace_bytes, void *stream) {
  return simulate_range(cfg, params, n_points, n_paths, n_steps, dt, nullptr, seed, 0, n_steps, nullptr, out_stats,
                        out_paths, out_trace, workspace, workspace_bytes, stream);
}

BM_API bm_status bm_simulate_dt(const bm_config *cfg, const bm_params *params, const double *dt_points, int32_t n_points,
                         int64_t n_paths, int64_t n_steps, uint64_t seed, bm_stats *out_stats, double *out_paths,
                         void *workspace, size_t workspace_bytes, void *stream) {
  if (!dt_points || ((uintptr_t)dt_points & 7)) return BM_ERR_INVALID_ARG;
  // dt = 1 passes the scalar checks; every kernel reads its step length from dt_points[point]
  return simulate_range(cfg, params, n_points, n_paths, n_steps, 1.0, dt_points, seed, 0, n_steps, nullptr, out_stats,
                        out_paths, nullptr, workspace, workspace_bytes, stream);
}

BM_API size_t bm_state_bytes(const bm_config *cfg, int32_t n_points, int64_t n_paths) {
  if (!valid_cfg(cfg) || n_points <= 0 || n_paths <= 0) return 0;
  return (size_t)STATE_SLOTS * sizeof(unsigned long long) * (size_t)n_points * (size_t)n_paths;
}

BM_API bm_status bm_simulate_chunk(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                            int64_t n_steps, double dt, uint64_t seed, int64_t step_begin, int64_t step_count,
                            void *state, size_t state_bytes, bm_stats *out_stats, double *out_paths, void *workspace,
                            size_t workspace_bytes, void *stream) {
  if (step_begin < 0 || step_count <= 0 || n_steps <= 0 || step_begin > n_steps - step_count) return BM_ERR_INVALID_ARG;
  const int64_t step_end = step_begin + step_count;
  // chunk boundaries inside a run sit on multiples of BM_CHUNK_ALIGN grid steps (one Gaussian call of the fp32 kernel)
  if ((step_begin % BM_CHUNK_ALIGN) != 0 || (step_end != n_steps && (step_end % BM_CHUNK_ALIGN) != 0)) return BM_ERR_INVALID_ARG;
  if (!state || ((uintptr_t)state & 15)) return BM_ERR_INVALID_ARG;
  const size_t need = bm_state_bytes(cfg, n_points, n_paths);
  if (need == 0 || state_bytes < need) return BM_ERR_WORKSPACE;
  return simulate_range(cfg, params, n_points, n_paths, n_steps, dt, nullptr, seed, step_begin, step_end, state, out_stats,
                        out_paths, nullptr, workspace, workspace_bytes, stream);
}

BM_API bm_status bm_state_histogram(const bm_config *cfg, int32_t n_points, int64_t n_paths, const void *state,
                             size_t state_bytes, int32_t n_bins, uint64_t *counts, void *stream) {
  if (!valid_cfg(cfg) || n_points <= 0 || n_paths <= 0 || !state || !counts || n_bins <= 0 || n_bins > 4096) return BM_ERR_INVALID_ARG;
  if (((uintptr_t)state & 15) || ((uintptr_t)counts & 7)) return BM_ERR_INVALID_ARG;
  if (cfg->potential == BM_POT_QUAD) return BM_ERR_UNSUPPORTED;  // no period to fold into
  const size_t need = bm_state_bytes(cfg, n_points, n_paths);
  if (need == 0 || state_bytes < need) return BM_ERR_WORKSPACE;
  const double period = cfg->potential == BM_POT_SINE2 ? 1.0 : 2.0;
  const bool theta = cfg->prec == BM_F32 && cfg->scheme == BM_SCHEME_JUMP_ADAPTED;   // position kept as scale * x
  const double scale = (theta && cfg->potential == BM_POT_SINE2) ? 6.283185307179586 : 1.0;
  return launch_state_hist(reinterpret_cast<const unsigned long long *>(state), n_points, n_paths, theta ? 0 : 1,
                           1.0 / (period * scale), n_bins, reinterpret_cast<unsigned long long *>(counts),
                           reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

BM_API bm_status bm_state_moments(const bm_config *cfg, int32_t n_points, int64_t n_paths, const void *state, size_t state_bytes,
                           const void *ref_state, double *out, void *stream) {
  if (!valid_cfg(cfg) || n_points <= 0 || n_paths <= 0 || !state || !out) return BM_ERR_INVALID_ARG;
  if (((uintptr_t)state & 15) || ((uintptr_t)ref_state & 15) || ((uintptr_t)out & 7)) return BM_ERR_INVALID_ARG;
  const size_t need = bm_state_bytes(cfg, n_points, n_paths);
  if (need == 0 || state_bytes < need) return BM_ERR_WORKSPACE;
  const double period = cfg->potential == BM_POT_SINE2 ? 1.0 : (cfg->potential == BM_POT_PWL ? 2.0 : 0.0);
  const bool literal = cfg->scheme == BM_SCHEME_PAPER_LITERAL;
  const bool theta = cfg->prec == BM_F32 && !literal;  // position and velocity kept as scale * x
  const double scale = (theta && cfg->potential == BM_POT_SINE2) ? 6.283185307179586 : 1.0;
  return launch_state_moments(reinterpret_cast<const unsigned long long *>(state),
                              reinterpret_cast<const unsigned long long *>(ref_state), n_points, n_paths,
                              theta ? 0 : (literal ? 2 : 1), period, 1.0 / scale, out,
                              reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

BM_API bm_status bm_simulate_host(const bm_config *cfg, const bm_params *params, int32_t n_points, int64_t n_paths,
                           int64_t n_steps, double dt, uint64_t seed, bm_stats *out_stats, double *out_paths,
                           void *stream) {
  if (!valid_cfg(cfg) || !params || !out_stats || n_points <= 0 || n_paths <= 0) return BM_ERR_INVALID_ARG;
  if (!valid_params_host(cfg, params, n_points)) return BM_ERR_INVALID_ARG;
  const size_t ws = bm_workspace_bytes(cfg, n_points, n_paths);
  if (ws == 0) return BM_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const size_t pb = (size_t)n_points * sizeof(bm_params), sb = (size_t)n_points * sizeof(bm_stats);
  const size_t ob = out_paths ? (size_t)n_points * (size_t)n_paths * BM_OUT_STRIDE * sizeof(double) : 0;
  void *d_params = nullptr, *d_stats = nullptr, *d_ws = nullptr, *d_paths = nullptr;
  bm_status rc = BM_ERR_CUDA;
  cudaMemPool_t pool = host_entry_pool();
  if (!pool) return BM_ERR_CUDA;
  do {  // stream-ordered allocation: after the first call the blocks come from the library's pool
    if (cudaMallocFromPoolAsync(&d_params, pb, pool, st) != cudaSuccess) break;
    if (cudaMallocFromPoolAsync(&d_stats, sb, pool, st) != cudaSuccess) break;
    if (cudaMallocFromPoolAsync(&d_ws, ws, pool, st) != cudaSuccess) break;
    if (ob && cudaMallocFromPoolAsync(&d_paths, ob, pool, st) != cudaSuccess) break;
    if (cudaMemcpyAsync(d_params, params, pb, cudaMemcpyHostToDevice, st) != cudaSuccess) break;
    bm_config run = *cfg;
    run.event_mode = resolve_event_mode_host(cfg, params, n_points, dt);
    rc = bm_simulate(&run, (const bm_params *)d_params, n_points, n_paths, n_steps, dt, seed, (bm_stats *)d_stats,
                     (double *)d_paths, nullptr, d_ws, ws, stream);
    if (rc != BM_OK) break;
    rc = BM_ERR_CUDA;
    if (cudaMemcpyAsync(out_stats, d_stats, sb, cudaMemcpyDeviceToHost, st) != cudaSuccess) break;
    if (ob && cudaMemcpyAsync(out_paths, d_paths, ob, cudaMemcpyDeviceToHost, st) != cudaSuccess) break;
    rc = BM_OK;
  } while (0);
  if (d_params) cudaFreeAsync(d_params, st);
  if (d_stats) cudaFreeAsync(d_stats, st);
  if (d_ws) cudaFreeAsync(d_ws, st);
  if (d_paths) cudaFreeAsync(d_paths, st);
  if (cudaStreamSynchronize(st) != cudaSuccess && rc == BM_OK) rc = BM_ERR_CUDA;
  if (rc == BM_ERR_CUDA) cudaGetLastError();
  return rc;
}

BM_API bm_status bm_philox_fill(uint64_t seed, uint64_t path0, int32_t n_paths, uint32_t stream_id, uint32_t idx0,
                         int32_t n_idx, uint32_t *out, void *stream) {
  if (!out || n_paths <= 0 || n_idx <= 0 || ((uintptr_t)out & 15)) return BM_ERR_INVALID_ARG;
  if ((long long)n_paths * n_idx > (1LL << 36)) return BM_ERR_INVALID_ARG;
  const PhiloxKeys K = make_keys(seed);
  return launch_philox_fill(K, path0, n_paths, stream_id, idx0, n_idx, out, reinterpret_cast<cudaStream_t>(stream)) ==
                 cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

BM_API bm_status bm_gauss_fill(int32_t prec, int32_t gauss, uint64_t seed, uint64_t path0, int32_t n_paths, uint64_t m0,
                        int32_t n_m, void *out, void *stream) {
  if (!out || n_paths <= 0 || n_m <= 0 || (m0 & 7)) return BM_ERR_INVALID_ARG;
  if (gauss < BM_GAUSS_AUTO || gauss > BM_GAUSS_W16P) return BM_ERR_INVALID_ARG;
  if (prec != BM_F32 && prec != BM_F64) return BM_ERR_INVALID_ARG;
  const PhiloxKeys K = make_keys(seed);
  return launch_gauss_fill(prec, gauss, K, path0, n_paths, m0, n_m, out, reinterpret_cast<cudaStream_t>(stream)) ==
                 cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

BM_API bm_status bm_box_muller_words(int32_t prec, const uint32_t *words, int32_t n_pairs, void *out, void *stream) {
  if (!words || !out || n_pairs <= 0 || (prec != BM_F32 && prec != BM_F64)) return BM_ERR_INVALID_ARG;
  if (((uintptr_t)words & 7) || ((uintptr_t)out & 15)) return BM_ERR_INVALID_ARG;
  return launch_box_muller_words(prec, words, n_pairs, out, reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

BM_API bm_status bm_event_normal_words(const uint32_t *words, int32_t n, float *out, void *stream) {
  if (!words || !out || n <= 0 || ((uintptr_t)words & 3) || ((uintptr_t)out & 3)) return BM_ERR_INVALID_ARG;
  return launch_event_normal_words(words, n, out, reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

BM_API bm_status bm_kernel_info(const bm_config *cfg, int32_t n_points, int64_t n_paths, int32_t *regs_per_thread,
                         int32_t *launch_threads, int32_t *blocks_per_sm, int32_t *sm_count, int32_t *gauss) {
  if (!valid_cfg(cfg) || n_points <= 0 || n_paths <= 0) return BM_ERR_INVALID_ARG;
  Launch L;
  const bm_status ps = pick_kernel(cfg, n_points, n_paths, &L);
  if (ps != BM_OK) return ps;
  cudaFuncAttributes attr;
  const KernelFn fn = L.fn ? L.fn : L.fn_lanes;  // the per-lane-clock form when cfg forces it
  const size_t smem = L.fn ? L.smem : L.smem_lanes;
  if (cudaFuncGetAttributes(&attr, (const void *)fn) != cudaSuccess) { cudaGetLastError(); return BM_ERR_CUDA; }
  int nb = 0, dev = 0, sms = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, (const void *)fn, L.threads, smem) != cudaSuccess) { cudaGetLastError(); return BM_ERR_CUDA; }
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    cudaGetLastError();
    return BM_ERR_CUDA;
  }
  if (regs_per_thread) *regs_per_thread = attr.numRegs;
  if (launch_threads) *launch_threads = L.threads;
  if (blocks_per_sm) *blocks_per_sm = nb;
  if (sm_count) *sm_count = sms;
  if (gauss) *gauss = L.gauss;
  return BM_OK;
}

BM_API bm_status bm_pipe_probe(int32_t op, int32_t iters, int32_t blocks, int32_t threads, float *sink, void *stream) {
  if (op < 0 || op >= BM_PROBE_COUNT || iters <= 0 || blocks <= 0 || threads <= 0 || threads > 1024 || !sink) return BM_ERR_INVALID_ARG;
  return launch_probe(op, iters, blocks, threads, sink, reinterpret_cast<cudaStream_t>(stream)) == cudaSuccess ? BM_OK : BM_ERR_CUDA;
}

}  // extern "C"
