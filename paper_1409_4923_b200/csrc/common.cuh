// common.cuh -- pieces shared by every kernel of the CUDA path: launch arguments, Philox4x32-10 (a3),
// the (n, mean, M2) merge of the deterministic ensemble reduction (a11).  sm_100a only.
// Nothing here is shared with oracle/ (which has its own Philox, Box-Muller and stepper).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/bm.h"

namespace bm {

constexpr int STREAM_INIT = 0, STREAM_GAUSS = 1, STREAM_POISSON = 2, STREAM_DICH = 3;

// Round keys of Philox4x32-10 (R1): k0 + i*W0, k1 + i*W1.  They depend on the seed only, so the host
// computes them once and they reach the kernels through the parameter constant bank (no registers).
struct PhiloxKeys {
  uint32_t k0[10];
  uint32_t k1[10];
};

struct SimArgs {
  const bm_params *params;
  double *partials;   // [grid][PARTIAL_STRIDE]
  double *out_paths;  // optional [n_points*n_paths][6]
  double *out_trace;  // optional [trace_paths][trace_steps][2]
  long long n_paths;  // per point
  long long n_steps;
  long long n_discard;
  long long trace_steps;
  long long trace_paths;
  double dt;
  const double *dt_points;  // optional [n_points]: per-point step length (overrides dt); nullptr = one dt for all
  int n_points;
  int blocks_per_point;
  // chunked runs (row f2): this launch does grid steps [step_begin, step_end) of a run of n_steps.  state == nullptr:
  // a whole run in one launch (step_begin = 0, step_end = n_steps).
  unsigned long long *state;  // [STATE_SLOTS][n_points * n_paths], 8-byte slots, slot-major (coalesced)
  long long step_begin, step_end;
  double adapt_tol;  // BM_SCHEME_ADAPTIVE (row f4): tolerance on |chi| and number of halvings of dt
  int adapt_levels;
  int event_mode;    // bm_event_mode (fp32 over-damped jump-adapted kernels)
  PhiloxKeys keys;
};

// The resumable state of a path (Alg. 5 steps 2 and 6, without the RNG state: Philox is stateless,
// so the draw counters are the RNG state).  Every kernel uses at most STATE_SLOTS 8-byte slots per path.
constexpr int STATE_SLOTS = 16;
struct StateIO {
  unsigned long long *base;
  long long stride;  // paths in the launch
  __device__ __forceinline__ void put(int slot, unsigned long long v) const { base[(long long)slot * stride] = v; }
  __device__ __forceinline__ unsigned long long get(int slot) const { return base[(long long)slot * stride]; }
  __device__ __forceinline__ void put2(int slot, uint32_t lo, uint32_t hi) const { put(slot, (unsigned long long)lo | ((unsigned long long)hi << 32)); }
  __device__ __forceinline__ void get2(int slot, uint32_t &lo, uint32_t &hi) const { const unsigned long long v = get(slot); lo = (uint32_t)v; hi = (uint32_t)(v >> 32); }
  __device__ __forceinline__ void putd(int slot, double v) const { put(slot, (unsigned long long)__double_as_longlong(v)); }
  __device__ __forceinline__ double getd(int slot) const { return __longlong_as_double((long long)get(slot)); }
};
// step length of a parameter point
__device__ __forceinline__ double step_length(const SimArgs &a, int point) {
  const double *src = a.dt_points ? a.dt_points + point : &a.dt;  // &a.dt: the kernel parameter itself
  return *src;
}
__device__ __forceinline__ StateIO state_io(const SimArgs &a, unsigned long long g) {
  return StateIO{a.state + g, (long long)a.n_points * a.n_paths};
}

// fp32 path kernel: event rings in dynamic shared memory (sim_f32.cuh, "event queues"); the host sizes the launch with
// the same function the kernel lays its arrays out with.
constexpr int EVQ = 8;  // ring capacity per path and stream (a power of two, <= 16)
constexpr int EVK = 4;  // refill passes per episode
constexpr int EV_FIELDS_P = 4, EV_FIELDS_D = 3;  // (cell, off, amplitude, normal), (cell, off, normal)

// 32-bit words of dynamic shared memory per thread of the fp32 path kernel (host and device agree through this): one
// record per thread, padded to an odd number of words; lclk: the per-lane-clock form also keeps the normals of two
// Gaussian calls in it
__host__ __device__ constexpr int f32_smem_words_per_thread(int noise, int gauss, int lclk = 0) {
  const int rings = ((noise & BM_NOISE_POISSON) ? EVQ * EV_FIELDS_P : 0) + ((noise & BM_NOISE_DICH) ? EVQ * EV_FIELDS_D : 0) + 4;
  // LANES form: one record per thread, with the normals of two Gaussian calls, padded to an odd number of words
  const int extra = !(noise & BM_NOISE_GAUSS) ? 0 : lclk ? (gauss == BM_GAUSS_W32 ? 16 : 32) : (gauss == BM_GAUSS_W32 ? 0 : 4);
  return (rings + extra) | 1;  // CELLS form, W16 / W16P: four words for the pairs of the rolled paths
}

// Event mode of a parameter point (fp32 over-damped jump-adapted kernels; sim_f32.cuh, "per-lane clocks"): expected
// kicks + flips per path and grid cell above LCLK_EVENTS_PER_CELL.  A function of the point's parameters and step
// length only (in double), evaluated alike by both forms of the kernel, so every block is taken by exactly one.
#ifndef BM_LCLK_EVENTS_PER_CELL
#define BM_LCLK_EVENTS_PER_CELL 0.02
#endif
constexpr double LCLK_EVENTS_PER_CELL = BM_LCLK_EVENTS_PER_CELL;
__device__ __forceinline__ bool lane_clock_point(const SimArgs &a, const bm_params &bp, double dt, int noise) {
  if (a.event_mode != BM_EVENTS_AUTO) return a.event_mode == BM_EVENTS_LANES;
  double rate = 0.0;
  if ((noise & BM_NOISE_POISSON) && bp.lambda > 0.0) rate += bp.lambda;
  if ((noise & BM_NOISE_DICH) && bp.mu_a > 0.0) rate += 0.5 * (bp.mu_a + (bp.mu_b > 0.0 ? bp.mu_b : 0.0));
  return rate * dt > LCLK_EVENTS_PER_CELL;
}

constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

// PAPER.md:40 uses cuRAND with per-thread state in global memory (Alg. 5 steps 2, 6); here the generator is
// stateless: (seed, path, stream, index) -> four words, recomputed in registers (reading R1, R2).
// Counter = (idx, stream, g lo, g hi); one round: (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2,
// c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0).
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKeys &K) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0;  // IMAD.WIDE.U32
    const unsigned long long p1 = (unsigned long long)PHILOX_M1 * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    c0 = hi1 ^ c1 ^ K.k0[r];  // LOP3
    c1 = lo1;
    c2 = hi0 ^ c3 ^ K.k1[r];
    c3 = lo0;
  }
  return make_uint4(c0, c1, c2, c3);
}

// Rounds R0 .. R1-1 of the same function on a counter held in c (the path kernel spreads the ten rounds of the next
// Gaussian call over a block of grid cells).
template <int R0, int R1>
__device__ __forceinline__ void philox_rounds(uint4 &c, const PhiloxKeys &K) {
#pragma unroll
  for (int r = R0; r < R1; ++r) {
    const unsigned long long p0 = (unsigned long long)PHILOX_M0 * c.x;
    const unsigned long long p1 = (unsigned long long)PHILOX_M1 * c.z;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    c = make_uint4(hi1 ^ c.y ^ K.k0[r], lo1, hi0 ^ c.w ^ K.k1[r], lo0);
  }
}

__device__ __forceinline__ uint4 philox_call(const PhiloxKeys &K, unsigned long long g, uint32_t stream,
                                             uint32_t idx) {
  return philox4x32_10(idx, stream, (uint32_t)g, (uint32_t)(g >> 32), K);
}

// ---- deterministic ensemble reduction (a11) -----------------------------------------------------------
// A leaf/partial carries n, mean and M2 (sum of squared deviations) of vbar and of x(T), plus plain sums of
// the event and sub-step counts.  Two partials merge with Chan's pairwise update, which is exact up to
// rounding whatever the split; the merge ORDER is fixed by (path index, block size) only, so results are
// bit-reproducible from run to run (PAPER.md:412 names the parallel reduction as the optimisation not taken).
constexpr int PARTIAL_STRIDE = 8;  // doubles
struct Partial {
  double n, mv, qv, mx, qx, sj, ss;
};

__device__ __forceinline__ Partial partial_zero() { return Partial{0, 0, 0, 0, 0, 0, 0}; }

__device__ __forceinline__ Partial merge(const Partial &a, const Partial &b) {
  Partial r;
  r.n = a.n + b.n;
  if (r.n == 0.0) return partial_zero();
  const double fb = b.n / r.n;            // weight of b
  const double w = a.n * fb;              // na*nb/n
  const double dv = b.mv - a.mv, dx = b.mx - a.mx;
  r.mv = a.mv + dv * fb;
  r.mx = a.mx + dx * fb;
  r.qv = a.qv + b.qv + dv * dv * w;
  r.qx = a.qx + b.qx + dx * dx * w;
  r.sj = a.sj + b.sj;
  r.ss = a.ss + b.ss;
  return r;
}

__device__ __forceinline__ Partial shfl_down(const Partial &p, int delta) {
  Partial r;
  r.n = __shfl_down_sync(0xffffffffu, p.n, delta);
  r.mv = __shfl_down_sync(0xffffffffu, p.mv, delta);
  r.qv = __shfl_down_sync(0xffffffffu, p.qv, delta);
  r.mx = __shfl_down_sync(0xffffffffu, p.mx, delta);
  r.qx = __shfl_down_sync(0xffffffffu, p.qx, delta);
  r.sj = __shfl_down_sync(0xffffffffu, p.sj, delta);
  r.ss = __shfl_down_sync(0xffffffffu, p.ss, delta);
  return r;
}

// lane 0 ends with the merge of lanes 0..31 in the fixed order ((0,1),(2,3)),... (tree by lane index)
__device__ __forceinline__ Partial warp_reduce(Partial p) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const Partial o = shfl_down(p, d);
    p = merge(p, o);  // lanes whose partner is out of range merge garbage, but their value is never used
  }
  return p;
}

// Whole block -> one partial, written by thread 0 to dst[PARTIAL_STRIDE].  smem: 32 * 7 doubles.
__device__ __forceinline__ void block_reduce_store(Partial p, double *dst) {
  __shared__ double sm[32][7];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
  p = warp_reduce(p);
  if (lane == 0) {
    sm[warp][0] = p.n; sm[warp][1] = p.mv; sm[warp][2] = p.qv; sm[warp][3] = p.mx; sm[warp][4] = p.qx;
    sm[warp][5] = p.sj; sm[warp][6] = p.ss;
  }
  __syncthreads();
  if (warp == 0) {
    Partial q = partial_zero();
    if (lane < nwarps) q = Partial{sm[lane][0], sm[lane][1], sm[lane][2], sm[lane][3], sm[lane][4], sm[lane][5], sm[lane][6]};
    q = warp_reduce(q);
    if (lane == 0) {
      dst[0] = q.n; dst[1] = q.mv; dst[2] = q.qv; dst[3] = q.mx; dst[4] = q.qx; dst[5] = q.sj; dst[6] = q.ss;
      dst[7] = 0.0;
    }
  }
}

__device__ __forceinline__ Partial leaf(double vbar, double xT, double jumps, double substeps) {
  return Partial{1.0, vbar, 0.0, xT, 0.0, jumps, substeps};
}

// launchers implemented per precision (sim_f64.cu / sim_f32_*.cu); return cudaError_t of the launch
struct KernelInfo { int regs; int smem; int blocks_per_sm; };

}  // namespace bm
