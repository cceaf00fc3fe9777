// dispatch.cuh -- kernel selection tables (one translation unit per family keeps nvcc parallel).
#pragma once
#include "common.cuh"

namespace bm {

typedef void (*KernelFn)(const SimArgs);

KernelFn pick_f64_overdamped(int potential, int noise, bool chunked, int paths_per_thread);
KernelFn pick_f64_inertial(int potential, int noise, bool chunked, int paths_per_thread);
// fp32: one family per (model, sincos, gauss) triple (BM_SINCOS_AUTO / BM_GAUSS_AUTO are resolved by the caller)
KernelFn pick_f32_od_sfu_w16(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_od_sfu_w32(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_od_fma_w16(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_od_fma_w32(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_in_sfu_w16(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_in_sfu_w32(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_in_fma_w16(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_in_fma_w32(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_od_sfu_w16p(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_od_fma_w16p(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_in_sfu_w16p(int potential, int noise, int occ, int lclk);
KernelFn pick_f32_in_fma_w16p(int potential, int noise, int occ, int lclk);

// the paper's own scheme as printed (sim_literal.cu); over-damped only
KernelFn pick_literal(int prec, int potential, int noise);
// dynamic step size control from chi (sim_adaptive.cu); fp64, over-damped only
KernelFn pick_adaptive_f64(int potential, int noise);

// fills (fill.cu)
cudaError_t launch_philox_fill(const PhiloxKeys &K, unsigned long long path0, int n_paths, uint32_t stream_id,
                               uint32_t idx0, int n_idx, uint32_t *out, cudaStream_t st);
cudaError_t launch_gauss_fill(int prec, int gauss, const PhiloxKeys &K, unsigned long long path0, int n_paths,
                              unsigned long long m0, int n_m, void *out, cudaStream_t st);
cudaError_t launch_box_muller_words(int prec, const uint32_t *words, int n_pairs, void *out, cudaStream_t st);
cudaError_t launch_event_normal_words(const uint32_t *words, int n, float *out, cudaStream_t st);
cudaError_t launch_grid_reduce(const double *partials, int n_points, int blocks_per_point, bm_stats *out,
                               cudaStream_t st);
cudaError_t launch_state_hist(const unsigned long long *state, int n_points, long long n_paths, int kind, double inv_period,
                              int n_bins, unsigned long long *counts, cudaStream_t st);
cudaError_t launch_state_moments(const unsigned long long *state, const unsigned long long *ref, int n_points, long long n_paths,
                                 int kind, double period, double inv_scale, double *out, cudaStream_t st);
cudaError_t launch_probe(int op, int iters, int blocks, int threads, float *sink, cudaStream_t st);

}  // namespace bm
