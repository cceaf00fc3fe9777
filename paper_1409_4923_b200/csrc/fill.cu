// fill.cu -- small kernels around the path kernels: raw Philox words (a3), Gaussian-stream normals (a4),
// the grid pass of the ensemble reduction (a11).
#include "dispatch.cuh"
#include "sim_f32.cuh"
#include "sim_f64.cuh"

namespace bm {

__global__ void philox_fill_kernel(const __grid_constant__ PhiloxKeys K, unsigned long long path0, int n_paths,
                                   uint32_t stream_id, uint32_t idx0, int n_idx, uint32_t *out) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)n_paths * n_idx) return;
  const int p = (int)(i / n_idx), j = (int)(i - (long long)p * n_idx);
  const uint4 w = philox_call(K, path0 + (unsigned long long)p, stream_id, idx0 + (uint32_t)j);
  reinterpret_cast<uint4 *>(out)[i] = w;
}

cudaError_t launch_philox_fill(const PhiloxKeys &K, unsigned long long path0, int n_paths, uint32_t stream_id,
                               uint32_t idx0, int n_idx, uint32_t *out, cudaStream_t st) {
  const long long total = (long long)n_paths * n_idx;
  const int threads = 256;
  const long long blocks = (total + threads - 1) / threads;
  philox_fill_kernel<<<(unsigned)blocks, threads, 0, st>>>(K, path0, n_paths, stream_id, idx0, n_idx, out);
  return cudaGetLastError();
}

// one thread = one Gaussian call of one path: NB = 4 normals (fp64, fp32 W32) or 8 (fp32 W16)
template <int PREC, int GW>
__global__ void gauss_fill_kernel(const __grid_constant__ PhiloxKeys K, unsigned long long path0, int n_paths,
                                  unsigned long long m0, int n_blocks, int n_m, void *out) {
  constexpr int NB = (PREC == BM_F32 && GW != BM_GAUSS_W32) ? 8 : 4;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)n_paths * n_blocks) return;
  const int p = (int)(i / n_blocks), b = (int)(i - (long long)p * n_blocks);
  const unsigned long long g = path0 + (unsigned long long)p;
  const uint32_t call = (uint32_t)(m0 / NB + b);
  if (PREC == BM_F64) {
    const uint4 w = philox_call(K, g, STREAM_GAUSS, call);
    double q[4];
    box_muller_f64(w.x, w.y, q[0], q[1]);
    box_muller_f64(w.z, w.w, q[2], q[3]);
    double *o = reinterpret_cast<double *>(out) + (long long)p * n_m;
    for (int j = 0; j < 4; ++j)
      if (4 * b + j < n_m) o[4 * b + j] = q[j];
  } else {
    float q[NB];
    gauss_block_standard_f32<GW>(K, g, call, q);
    float *o = reinterpret_cast<float *>(out) + (long long)p * n_m;
    for (int j = 0; j < NB; ++j)
      if (NB * b + j < n_m) o[NB * b + j] = q[j];
  }
}

cudaError_t launch_gauss_fill(int prec, int gauss, const PhiloxKeys &K, unsigned long long path0, int n_paths,
                              unsigned long long m0, int n_m, void *out, cudaStream_t st) {
  const int nb = (prec == BM_F32 && gauss != BM_GAUSS_W32) ? 8 : 4;
  const int n_blocks = (n_m + nb - 1) / nb;
  const long long total = (long long)n_paths * n_blocks;
  const int threads = 256;
  const unsigned blocks = (unsigned)((total + threads - 1) / threads);
  if (prec == BM_F64)
    gauss_fill_kernel<BM_F64, BM_GAUSS_W32><<<blocks, threads, 0, st>>>(K, path0, n_paths, m0, n_blocks, n_m, out);
  else if (gauss == BM_GAUSS_W32)
    gauss_fill_kernel<BM_F32, BM_GAUSS_W32><<<blocks, threads, 0, st>>>(K, path0, n_paths, m0, n_blocks, n_m, out);
  else if (gauss == BM_GAUSS_W16P)
    gauss_fill_kernel<BM_F32, BM_GAUSS_W16P><<<blocks, threads, 0, st>>>(K, path0, n_paths, m0, n_blocks, n_m, out);
  else  // W16, and AUTO (which resolves to it)
    gauss_fill_kernel<BM_F32, BM_GAUSS_W16><<<blocks, threads, 0, st>>>(K, path0, n_paths, m0, n_blocks, n_m, out);
  return cudaGetLastError();
}

// The variate transforms on GIVEN words (a4; bm_box_muller_words): pair i of `words` -> two standard normals, by the
// device code of the path kernels (fp64: the own ln / sqrt / sincospi of sim_f64.cuh; fp32: box_muller_f32, W32).
__global__ void box_muller_words_kernel(int prec, const uint32_t *__restrict__ words, int n_pairs, void *out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_pairs) return;
  const uint32_t wa = words[2 * i], wb = words[2 * i + 1];
  if (prec == BM_F64) {
    double g0, g1;
    box_muller_f64(wa, wb, g0, g1);
    reinterpret_cast<double *>(out)[2 * i] = g0;
    reinterpret_cast<double *>(out)[2 * i + 1] = g1;
  } else {
    float g0, g1;
    box_muller_f32(wa, wb, g0, g1);
    reinterpret_cast<float *>(out)[2 * i] = g0;
    reinterpret_cast<float *>(out)[2 * i + 1] = g1;
  }
}

// The normal of a sub-step that ends on an event (R13) on GIVEN words: the device code the fp32 path kernels apply to
// word 2 of the event's Philox call (bm_event_normal_words).
__global__ void event_normal_words_kernel(const uint32_t *__restrict__ words, int n, float *__restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = event_normal_f32(words[i]);
}

cudaError_t launch_event_normal_words(const uint32_t *words, int n, float *out, cudaStream_t st) {
  event_normal_words_kernel<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(words, n, out);
  return cudaGetLastError();
}

cudaError_t launch_box_muller_words(int prec, const uint32_t *words, int n_pairs, void *out, cudaStream_t st) {
  box_muller_words_kernel<<<(unsigned)((n_pairs + 127) / 128), 128, 0, st>>>(prec, words, n_pairs, out);
  return cudaGetLastError();
}

// Grid pass (a11): one warp per parameter point merges that point's per-block partials.  Lane l takes partials
// l, l+32, ... in order, then the warp tree merges the 32 lane results: a fixed order for a given
// (n_paths, block size), hence bit-reproducible.
__global__ void grid_reduce_kernel(const double *__restrict__ partials, int n_points, int blocks_per_point,
                                   bm_stats *__restrict__ out) {
  const int warp = (int)(((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5);
  const int lane = threadIdx.x & 31;
  if (warp >= n_points) return;
  const double *src = partials + (long long)warp * blocks_per_point * PARTIAL_STRIDE;
  Partial acc = partial_zero();
  for (int b = lane; b < blocks_per_point; b += 32) {
    const double *q = src + (long long)b * PARTIAL_STRIDE;
    acc = merge(acc, Partial{q[0], q[1], q[2], q[3], q[4], q[5], q[6]});
  }
  acc = warp_reduce(acc);
  if (lane == 0) {
    bm_stats s;
    s.n = acc.n;
    s.mean_v = acc.mv;
    s.var_v = acc.n > 1.0 ? acc.qv / (acc.n - 1.0) : 0.0;
    s.mean_xT = acc.mx;
    s.var_xT = acc.n > 1.0 ? acc.qx / (acc.n - 1.0) : 0.0;
    s.mean_jumps = acc.n > 0.0 ? acc.sj / acc.n : 0.0;
    s.mean_substeps = acc.n > 0.0 ? acc.ss / acc.n : 0.0;
    s.rsv = 0.0;
    out[warp] = s;
  }
}

// Row f3: histogram of the folded positions held in a checkpoint (the state of bm_simulate_chunk), one block-private
// histogram in shared memory, integer atomics only (the counts do not depend on the order of the additions).
// kind 0: fp32 jump-adapted kernel (slot 0 low word = theta as float, theta = scale * x);  kind 1: fp64 kernel and
// both literal kernels (slot 0 = position as double).  u = position / period, reduced to [0, 1).
__global__ void state_hist_kernel(const unsigned long long *__restrict__ state, long long n_paths, int blocks_per_point,
                                  int kind, double inv_period, int n_bins, unsigned long long *__restrict__ counts) {
  extern __shared__ unsigned int sh[];
  for (int i = threadIdx.x; i < n_bins; i += blockDim.x) sh[i] = 0u;
  __syncthreads();
  const int point = blockIdx.x / blocks_per_point;
  const long long p = (long long)(blockIdx.x - point * blocks_per_point) * blockDim.x + threadIdx.x;
  if (p < n_paths) {
    const unsigned long long v = __ldcg(state + (long long)point * n_paths + p);  // slot 0
    const double pos = kind == 0 ? (double)__uint_as_float((uint32_t)v) : __longlong_as_double((long long)v);
    double u = pos * inv_period;
    u -= floor(u);
    int b = (int)(u * (double)n_bins);
    b = b < 0 ? 0 : (b >= n_bins ? n_bins - 1 : b);
    atomicAdd(&sh[b], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < n_bins; i += blockDim.x)
    if (sh[i]) atomicAdd(counts + (long long)point * n_bins + i, (unsigned long long)sh[i]);
}

cudaError_t launch_state_hist(const unsigned long long *state, int n_points, long long n_paths, int kind, double inv_period,
                              int n_bins, unsigned long long *counts, cudaStream_t st) {
  const int threads = 256;
  const long long bpp = (n_paths + threads - 1) / threads;
  if (bpp * n_points > 0x7FFFFFFFLL) return cudaErrorInvalidValue;
  state_hist_kernel<<<(unsigned)(bpp * n_points), threads, (size_t)n_bins * sizeof(unsigned int), st>>>(
      state, n_paths, (int)bpp, kind, inv_period, n_bins, counts);
  return cudaGetLastError();
}

// Row f3: ensemble moments of a checkpoint, per parameter point, optionally against a reference checkpoint of the same
// run taken at an earlier time t0: D_eff(t) = Var[x(t) - x(t0)] / (2 (t - t0)) and the velocity autocovariance
// <v(t0) v(t)> - <v(t0)><v(t)> (the stationary state).  One block per point; thread t
// takes paths t, t + T, ... in order, then a fixed shuffle / shared-memory tree: bit-reproducible.  Two passes (means,
// then central moments), fp64 throughout.  kind 0: fp32 jump-adapted kernel (slot 0 = (theta, wraps), slot 1 low word
// = velocity in theta units, theta = scale * x);  kind 1: fp64 jump-adapted kernel (slots 0, 1, 2 = xi, wraps, v);
// kind 2: paper-literal kernels (slots 0, 1 = x, wraps; no velocity).
struct PathXV { double x, v; };
__device__ __forceinline__ PathXV load_xv(const unsigned long long *st, long long stride, long long i, int kind, double period,
                                          double inv_scale) {
  PathXV r;
  if (kind == 0) {
    const unsigned long long a = __ldcg(st + i), b = __ldcg(st + stride + i);
    r.x = (double)(int)(uint32_t)(a >> 32) * period + (double)__uint_as_float((uint32_t)a) * inv_scale;
    r.v = (double)__uint_as_float((uint32_t)b) * inv_scale;
  } else {
    r.x = (double)(long long)__ldcg(st + stride + i) * period + __longlong_as_double((long long)__ldcg(st + i));
    r.v = kind == 1 ? __longlong_as_double((long long)__ldcg(st + 2 * stride + i)) : 0.0;
  }
  return r;
}

template <int K>
__device__ __forceinline__ void block_sum(double (&acc)[K], double (*sm)[K]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
#pragma unroll
  for (int k = 0; k < K; ++k)
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) acc[k] += __shfl_down_sync(0xffffffffu, acc[k], d);
  __syncthreads();
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < K; ++k) sm[warp][k] = acc[k];
  __syncthreads();
#pragma unroll
  for (int k = 0; k < K; ++k) {
    double t = 0.0;
    for (int w = 0; w < nwarps; ++w) t += sm[w][k];  // every thread adds the warps' sums in the same order
    acc[k] = t;
  }
}

__global__ void __launch_bounds__(1024) state_moments_kernel(const unsigned long long *__restrict__ state,
                                                           const unsigned long long *__restrict__ ref, long long n_paths,
                                                           long long stride, int kind, double period, double inv_scale,
                                                           double *__restrict__ out) {
  __shared__ double sm[32][6];
  const int point = blockIdx.x;
  const long long base = (long long)point * n_paths;
  double a1[6] = {0, 0, 0, 0, 0, 0};  // sums of x, v, dx, v0 (and two spare)
  for (long long p = threadIdx.x; p < n_paths; p += blockDim.x) {
    const PathXV c = load_xv(state, stride, base + p, kind, period, inv_scale);
    a1[0] += c.x; a1[1] += c.v;
    if (ref) {
      const PathXV r = load_xv(ref, stride, base + p, kind, period, inv_scale);
      a1[2] += c.x - r.x; a1[3] += r.v;
    }
  }
  block_sum<6>(a1, sm);
  const double n = (double)n_paths;
  const double mx = a1[0] / n, mv = a1[1] / n, md = a1[2] / n, mv0 = a1[3] / n;
  double a2[6] = {0, 0, 0, 0, 0, 0};  // sums of (x-mx)^2, (v-mv)^2, (dx-md)^2, (v0-mv0)(v-mv), (v0-mv0)^2
  for (long long p = threadIdx.x; p < n_paths; p += blockDim.x) {
    const PathXV c = load_xv(state, stride, base + p, kind, period, inv_scale);
    a2[0] += (c.x - mx) * (c.x - mx); a2[1] += (c.v - mv) * (c.v - mv);
    if (ref) {
      const PathXV r = load_xv(ref, stride, base + p, kind, period, inv_scale);
      const double dx = c.x - r.x;
      a2[2] += (dx - md) * (dx - md); a2[3] += (r.v - mv0) * (c.v - mv); a2[4] += (r.v - mv0) * (r.v - mv0);
    }
  }
  block_sum<6>(a2, sm);
  if (threadIdx.x == 0) {
    const double nm1 = n > 1.0 ? n - 1.0 : 1.0;
    double *o = out + (long long)point * BM_MOM_STRIDE;
    o[BM_MOM_N] = n; o[BM_MOM_MEAN_X] = mx; o[BM_MOM_VAR_X] = a2[0] / nm1; o[BM_MOM_MEAN_V] = mv; o[BM_MOM_VAR_V] = a2[1] / nm1;
    o[BM_MOM_MEAN_DX] = ref ? md : 0.0; o[BM_MOM_VAR_DX] = ref ? a2[2] / nm1 : 0.0; o[BM_MOM_COV_V0V] = ref ? a2[3] / nm1 : 0.0;
    o[BM_MOM_VAR_V0] = ref ? a2[4] / nm1 : 0.0; o[9] = 0.0;
  }
}

cudaError_t launch_state_moments(const unsigned long long *state, const unsigned long long *ref, int n_points, long long n_paths,
                                 int kind, double period, double inv_scale, double *out, cudaStream_t st) {
  // one block per point: 1024 threads for the large single-point ensembles, 256 for sweeps of many points
  state_moments_kernel<<<(unsigned)n_points, n_paths >= 8192 ? 1024 : 256, 0, st>>>(state, ref, n_paths, (long long)n_points * n_paths, kind, period,
                                                          inv_scale, out);
  return cudaGetLastError();
}

cudaError_t launch_grid_reduce(const double *partials, int n_points, int blocks_per_point, bm_stats *out,
                               cudaStream_t st) {
  const int threads = 128;  // 4 points per block
  const unsigned blocks = (unsigned)((n_points + 3) / 4);
  grid_reduce_kernel<<<blocks, threads, 0, st>>>(partials, n_points, blocks_per_point, out);
  return cudaGetLastError();
}

}  // namespace bm
