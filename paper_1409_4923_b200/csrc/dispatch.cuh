// dispatch.cuh -- kernel selection tables (one translation unit per family keeps nvcc parallel).
#pragma once
#include "common.cuh"

namespace bm {

typedef void (*KernelFn)(const SimArgs);

KernelFn pick_f64_overdamped(int potential, int noise);
KernelFn pick_f64_inertial(int potential, int noise);
// fp32: one family per sincos variant (BM_SINCOS_AUTO is resolved by the caller)
KernelFn pick_f32_overdamped_sfu(int potential, int noise);
KernelFn pick_f32_overdamped_fma(int potential, int noise);
KernelFn pick_f32_inertial_sfu(int potential, int noise);
KernelFn pick_f32_inertial_fma(int potential, int noise);
// warp-specialised variants (Gaussian producer warps; launched with 2 x block_threads threads and
// ws_ring_bytes(block_threads) of dynamic shared memory); nullptr when the combination has none
KernelFn pick_f32_overdamped_ws(int sincos, int potential, int noise);
KernelFn pick_f32_inertial_ws(int sincos, int potential, int noise);
size_t ws_ring_bytes(int path_threads);

// fills (fill.cu)
cudaError_t launch_philox_fill(const PhiloxKeys &K, unsigned long long path0, int n_paths, uint32_t stream_id,
                               uint32_t idx0, int n_idx, uint32_t *out, cudaStream_t st);
cudaError_t launch_gauss_fill(int prec, int sincos, const PhiloxKeys &K, unsigned long long path0, int n_paths,
                              unsigned long long m0, int n_m, void *out, cudaStream_t st);
cudaError_t launch_grid_reduce(const double *partials, int n_points, int blocks_per_point, bm_stats *out,
                               cudaStream_t st);
cudaError_t launch_probe(int op, int iters, int blocks, int threads, float *sink, cudaStream_t st);

}  // namespace bm
