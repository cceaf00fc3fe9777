// sim_f64.cuh -- fp64 path kernel: one thread = one realization, state in registers for the whole run
// (Alg. 5 :367-374 without the per-launch load/store of steps 2 and 6).
// It follows DESIGN.md readings R3-R9 operation by operation, so that per-path results track the fp64
// oracle to ~1e-13 (only libm-vs-CUDA transcendental rounding and FMA contraction differ).
#pragma once
#include "common.cuh"

namespace bm {

template <int POT>
__device__ __forceinline__ double period_f64() { return POT == BM_POT_SINE2 ? 1.0 : (POT == BM_POT_PWL ? 2.0 : 0.0); }

// u(w) = (w + 1/2) 2^-32  (R3)
__device__ __forceinline__ double u01_f64(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

// Box-Muller pair from two words (R3): r = sqrt(-2 ln u(wa)); (r cos 2 pi u(wb), r sin 2 pi u(wb))
__device__ __forceinline__ void box_muller_f64(uint32_t wa, uint32_t wb, double &g0, double &g1) {
  const double r = sqrt(-2.0 * log(u01_f64(wa)));
  double s, c;
  sincospi(2.0 * u01_f64(wb), &s, &c);
  g0 = r * c;
  g1 = r * s;
}

// the Gaussian call in progress at a checkpoint is recomputed, not stored (kept out of line: it runs once per launch)
static __device__ __noinline__ void regen_gauss_block_f64(const PhiloxKeys &K, unsigned long long g, uint32_t call, double *gq) {
  const uint4 w = philox_call(K, g, STREAM_GAUSS, call);
  box_muller_f64(w.x, w.y, gq[0], gq[1]);
  box_muller_f64(w.z, w.w, gq[2], gq[3]);
}

// Checkpoint record of the fp64 kernel (row f2).  Loading and storing stay out of line so that the code of the time
// loop is the same whether or not a launch is a chunk (inlined, they cost the whole kernel 6 % on C1).
struct CkptF64 {
  double xi, v, rP, rD, z, jumps, sxi, sv;
  long long wraps, swraps;
  unsigned long long m;
  uint32_t kP, kD;
  int d;
};
static __device__ __noinline__ void ckpt_load_f64(const SimArgs &a, unsigned long long g, CkptF64 &c) {
  const StateIO io = state_io(a, g);
  uint32_t lo, hi;
  c.xi = io.getd(0); c.wraps = (long long)io.get(1); c.v = io.getd(2);
  c.rP = io.getd(3); c.rD = io.getd(4); c.z = io.getd(5);
  io.get2(6, c.kP, c.kD);
  io.get2(7, lo, hi); c.d = (int)lo;
  c.m = io.get(8); c.jumps = io.getd(9);
  c.sxi = io.getd(10); c.swraps = (long long)io.get(11); c.sv = io.getd(12);
}
static __device__ __noinline__ void ckpt_store_f64(const SimArgs &a, unsigned long long g, const CkptF64 &c) {
  const StateIO io = state_io(a, g);
  io.putd(0, c.xi); io.put(1, (unsigned long long)c.wraps); io.putd(2, c.v);
  io.putd(3, c.rP); io.putd(4, c.rD); io.putd(5, c.z);
  io.put2(6, c.kP, c.kD);
  io.put2(7, (uint32_t)c.d, 0u);
  io.put(8, c.m); io.putd(9, c.jumps);
  io.putd(10, c.sxi); io.put(11, (unsigned long long)c.swraps); io.putd(12, c.sv);
}

struct PointF64 {
  double A1, A2, c0, D, lambda, zeta, Fa, Fb, mu_a, mu_b, gamma, amp, omega;
};

// -V'(x) on the (nearly) folded coordinate
template <int POT>
__device__ __forceinline__ double minus_dV_f64(const PointF64 &P, double x) {
  if (POT == BM_POT_SINE2) {
    const double c = cospi(2.0 * x);
    const double c2 = fma(2.0 * c, c, -1.0);  // cos 4 pi x = 2 cos^2 2 pi x - 1: one cosine per force evaluation
    return -(2.0 * M_PI * P.A1 * c + 4.0 * M_PI * P.A2 * c2);
  } else if (POT == BM_POT_PWL) {
    const double y = x - 2.0 * floor(x * 0.5);
    return (y < 1.0) ? P.A1 : -P.A1;
  } else {
    return -P.A1 * x;
  }
}

struct StateF64 {
  double xi;
  long long wraps;
  double v;
};

template <int POT>
__device__ __forceinline__ void fold_f64(StateF64 &s) {
  if (POT == BM_POT_QUAD) return;
  const double L = period_f64<POT>();
  const double k = floor(s.xi / L);
  if (k != 0.0) {
    s.xi -= k * L;
    s.wraps += (long long)k;
    if (s.xi < 0.0) { s.xi += L; s.wraps -= 1; }
    if (s.xi >= L) { s.xi -= L; s.wraps += 1; }
  }
}

template <int POT>
__device__ __forceinline__ double unfolded_f64(const StateF64 &s) {
  return (double)s.wraps * period_f64<POT>() + s.xi;
}

// CHUNKED: the launch may be one chunk of a run (row f2).  A separate instantiation, because the checkpoint code in
// the same kernel changes the register allocation of the time loop (111 -> 102 registers, 6 % slower on C1).
template <int MODEL, int POT, int NOISE, bool CHUNKED>
__global__ void __launch_bounds__(256) bm_paths_f64(const __grid_constant__ SimArgs a) {
  constexpr bool HAS_G = NOISE & BM_NOISE_GAUSS, HAS_P = NOISE & BM_NOISE_POISSON, HAS_D = NOISE & BM_NOISE_DICH;
  constexpr bool INERTIAL = MODEL == BM_INERTIAL;
  const int point = blockIdx.x / a.blocks_per_point;
  const int chunk = blockIdx.x - point * a.blocks_per_point;
  const long long p = (long long)chunk * blockDim.x + threadIdx.x;
  Partial mine = partial_zero();

  if (p < a.n_paths) {
    const unsigned long long g = (unsigned long long)point * (unsigned long long)a.n_paths + (unsigned long long)p;
    const bm_params bp = a.params[point];
    PointF64 P;
    P.A1 = bp.A1; P.A2 = bp.A2; P.D = HAS_G ? bp.D : 0.0;
    P.lambda = HAS_P ? bp.lambda : 0.0; P.zeta = HAS_P ? bp.zeta : 0.0;
    P.Fa = bp.Fa; P.Fb = bp.Fb; P.mu_a = bp.mu_a; P.mu_b = bp.mu_b;
    P.gamma = bp.gamma; P.amp = bp.amp; P.omega = bp.omega;
    P.c0 = bp.F - P.lambda * P.zeta;  // constant part of the drift a(x), all three stages (R6)
    const double dt = step_length(a, point);
    const double L0 = (POT == BM_POT_QUAD) ? 1.0 : period_f64<POT>();

    // R4: initial condition from init-stream call 0
    const uint4 wi = philox_call(a.keys, g, STREAM_INIT, 0);
    StateF64 s;
    s.xi = (bp.x0_fixed >= 0.0) ? bp.x0_fixed : L0 * ((double)wi.x * (1.0 / 4294967296.0));
    s.wraps = 0;
    s.v = INERTIAL ? bp.v0_lo + (bp.v0_hi - bp.v0_lo) * u01_f64(wi.y) : 0.0;
    fold_f64<POT>(s);
    // a non-positive rate of leaving -Fa switches the dichotomous source off at this point (Gamma = 0, as the oracle)
    const bool onD = HAS_D && P.mu_a > 0.0;
    int d = onD ? ((u01_f64(wi.z) < P.mu_a / (P.mu_a + P.mu_b)) ? 1 : 0) : -1;

    uint32_t kP = 0, kD = 0;
    double rP = 0.0, rD = 0.0, z = 0.0;
    bool onP = false;
    if (HAS_P) {
      onP = P.lambda > 0.0;  // lambda == 0 at a point of a sweep: the clock never fires
      if (onP) {
        const uint4 w = philox_call(a.keys, g, STREAM_POISSON, 0);
        rP = -log(u01_f64(w.x)) / P.lambda;
        z = -P.zeta * log(u01_f64(w.y));
      }
    }
    if (HAS_D && onD) {
      const uint4 w = philox_call(a.keys, g, STREAM_DICH, 0);
      rD = -log(u01_f64(w.x)) / (d ? P.mu_b : P.mu_a);
    }

    const bool tracing = a.out_trace != nullptr && (long long)g < a.trace_paths;
    double *trace = tracing ? a.out_trace + (long long)g * a.trace_steps * 2 : nullptr;

    long long n = CHUNKED ? a.step_begin : 0;
    unsigned long long m = 0;
    double rem = dt, jumps = 0.0;
    double gq[4] = {0.0, 0.0, 0.0, 0.0};
    StateF64 snap = s;
    if (CHUNKED && a.state != nullptr && a.step_begin > 0) {  // row f2: continue a run from its checkpoint
      CkptF64 c;
      ckpt_load_f64(a, g, c);
      s.xi = c.xi; s.wraps = c.wraps; s.v = c.v; rP = c.rP; rD = c.rD; z = c.z; kP = c.kP; kD = c.kD; d = c.d;
      m = c.m; jumps = c.jumps; snap.xi = c.sxi; snap.wraps = c.swraps; snap.v = c.sv;
      if (HAS_G && (m & 3ull) != 0) {
        double t[4];
        regen_gauss_block_f64(a.keys, g, (uint32_t)(m >> 2), t);
        gq[0] = t[0]; gq[1] = t[1]; gq[2] = t[2]; gq[3] = t[3];
      }
    }
    const long long n_end = CHUNKED ? a.step_end : a.n_steps;
    while (n < n_end) {
      double h = rem;
      if (HAS_P && onP && rP < h) h = rP;
      if (HAS_D && onD && rD < h) h = rD;
      double gn = 0.0;
      if (HAS_G) {
        if ((m & 3ull) == 0) {
          const uint4 w = philox_call(a.keys, g, STREAM_GAUSS, (uint32_t)(m >> 2));
          box_muller_f64(w.x, w.y, gq[0], gq[1]);
          box_muller_f64(w.z, w.w, gq[2], gq[3]);
        }
        const int j = (int)(m & 3ull);
        gn = (j == 0) ? gq[0] : (j == 1) ? gq[1] : (j == 2) ? gq[2] : gq[3];
      }
      m++;
      const double Gd = (HAS_D && onD) ? (d ? P.Fb : -P.Fa) : 0.0;
      const double cst = P.c0 + Gd;
      const double dxi = HAS_G ? sqrt(2.0 * P.D * h) * gn : 0.0;
      if (!INERTIAL) {
        // Alg. 1
        const double x = s.xi;
        const double F1 = minus_dV_f64<POT>(P, x) + cst;
        double xb = x + F1 * h + dxi;
        double F2 = minus_dV_f64<POT>(P, xb) + cst;
        xb = x + 0.5 * (F1 + F2) * h + dxi;
        F2 = minus_dV_f64<POT>(P, xb) + cst;
        s.xi = x + 0.5 * (F1 + F2) * h + dxi;
      } else {
        // R7: two-component version, additive noise in v only, drive evaluated at t and t+h
        const double t = __dadd_rn(__dmul_rn((double)n, dt), __dsub_rn(dt, rem));
        const double x = s.xi, v = s.v;
        const double A1x = v;
        const double A1v = -P.gamma * v + minus_dV_f64<POT>(P, x) + P.amp * cos(P.omega * t) + cst;
        double xb = x + A1x * h, vb = v + A1v * h + dxi;
        const double drive = P.amp * cos(P.omega * __dadd_rn(t, h));
        double A2x = vb;
        double A2v = -P.gamma * vb + minus_dV_f64<POT>(P, xb) + drive + cst;
        xb = x + 0.5 * (A1x + A2x) * h;
        vb = v + 0.5 * (A1v + A2v) * h + dxi;
        A2x = vb;
        A2v = -P.gamma * vb + minus_dV_f64<POT>(P, xb) + drive + cst;
        s.xi = x + 0.5 * (A1x + A2x) * h;
        s.v = v + 0.5 * (A1v + A2v) * h + dxi;
      }
      rem -= h;
      if (HAS_P && onP) {
        rP -= h;
        if (rP <= 0.0) {  // kick kP (a8)
          if (!INERTIAL) s.xi += z; else s.v += z;
          jumps += 1.0;
          kP++;
          const uint4 w = philox_call(a.keys, g, STREAM_POISSON, kP);
          rP = -log(u01_f64(w.x)) / P.lambda;
          z = -P.zeta * log(u01_f64(w.y));
        }
      }
      if (HAS_D && onD) {
        rD -= h;
        if (rD <= 0.0) {  // flip
          d = 1 - d;
          jumps += 1.0;
          kD++;
          const uint4 w = philox_call(a.keys, g, STREAM_DICH, kD);
          rD = -log(u01_f64(w.x)) / (d ? P.mu_b : P.mu_a);
        }
      }
      fold_f64<POT>(s);
      if (rem <= 0.0) {
        n++;
        rem = dt;
        if (tracing && n <= a.trace_steps) {
          trace[2 * (n - 1)] = unfolded_f64<POT>(s);
          trace[2 * (n - 1) + 1] = s.v;
        }
        if (n == a.n_discard) snap = s;
      }
    }
    if (CHUNKED && a.state != nullptr) {  // row f2: checkpoint (chunks end on completed grid steps, so rem = dt)
      CkptF64 c;
      c.xi = s.xi; c.wraps = s.wraps; c.v = s.v; c.rP = rP; c.rD = rD; c.z = z; c.kP = kP; c.kD = kD; c.d = d;
      c.m = m; c.jumps = jumps; c.sxi = snap.xi; c.swraps = snap.wraps; c.sv = snap.v;
      ckpt_store_f64(a, g, c);
    }
    // a10: eq. (30)
    const double span = (double)(a.n_steps - a.n_discard) * dt;
    const double xT = unfolded_f64<POT>(s);
    const double vbar = ((double)(s.wraps - snap.wraps) * period_f64<POT>() + (s.xi - snap.xi)) / span;
    if (a.out_paths && (!CHUNKED || a.step_end >= a.n_steps)) {
      double *o = a.out_paths + g * BM_OUT_STRIDE;
      o[BM_OUT_XT] = xT; o[BM_OUT_VT] = s.v; o[BM_OUT_VBAR] = vbar; o[BM_OUT_JUMPS] = jumps;
      o[BM_OUT_SUBSTEPS] = (double)m; o[BM_OUT_XTI] = unfolded_f64<POT>(snap);
    }
    mine = leaf(vbar, xT, jumps, (double)m);
  }
  if (CHUNKED && a.step_end < a.n_steps) return;  // not the last chunk: the partials are not used (uniform over the grid)
  block_reduce_store(mine, a.partials + (long long)blockIdx.x * PARTIAL_STRIDE);
}

}  // namespace bm
