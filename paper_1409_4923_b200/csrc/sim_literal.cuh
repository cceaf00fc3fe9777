// sim_literal.cuh -- the paper's own scheme, as printed (R11): constant step dt,
// Alg. 2 three-point increment for the Gaussian noise (eq. 25), Alg. 3 grid-quantised Poisson
// countdown (:270-291), Alg. 4 dichotomous countdown (:305-343), and Alg. 1 (:221-235) with the increments d eta and
// d Gamma entering line 6 only.  Over-damped only (the paper has no inertial model).  One thread = one realization,
// state in registers for the whole run (:389); the ensemble reduction is the one of the jump-adapted kernels.
//
// Readings (R11): [.] in Alg. 3/4 is floor; the first countdowns are drawn before step 0; uniform number n of the
// Gaussian stream is word n mod 4 of call n / 4; exponential variates are -ln(1 - phi) as printed; Poisson call k:
// w0 -> countdown before kick k, w1 -> amplitude of kick k; dichotomous call k: w0 -> countdown of sojourn k.
// The three-way decision of Alg. 2 (phi <= 1/6, 1/6 < phi <= 1/3, else) is taken on the 32-bit word itself
// (w <= 715827882, w <= 1431655764: the same sets as the comparisons of u(w) = (w + 1/2) 2^-32 with 1/6 and 1/3),
// so both precisions and the oracle decide identically.
#pragma once
#include <type_traits>

#include "sim_f32.cuh"
#include "sim_f64.cuh"

namespace bm {

template <typename T> struct LitMath;
template <> struct LitMath<double> {
  static __device__ __forceinline__ double u01(uint32_t w) { return u01_f64(w); }
  static __device__ __forceinline__ double exp_variate(uint32_t w, double scale) { return -scale * log(1.0 - u01_f64(w)); }
  static __device__ __forceinline__ double floor_(double x) { return floor(x); }
  static __device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
};
template <> struct LitMath<float> {
  // 1 - phi on a 2^-23 grid in (0, 1]: the complement of the top 23 bits (never 0, so the logarithm is finite)
  static __device__ __forceinline__ float exp_variate(uint32_t w, float scale) { return scale * neg_log_u_f32(~w); }
  static __device__ __forceinline__ float floor_(float x) { return floorf(x); }
  static __device__ __forceinline__ float sqrt_(float x) { return sqrtf(x); }
};

// -V'(x) + F for x within one period of the folded range
template <typename T, int POT>
__device__ __forceinline__ T lit_force(T x, T A1, T A2, T F) {
  if (POT == BM_POT_SINE2) {
    if (sizeof(T) == 8) {
      const double c = cospi(2.0 * (double)x);  // cos 4 pi x = 2 c^2 - 1
      return (T)(-(2.0 * M_PI * (double)A1 * c + 4.0 * M_PI * (double)A2 * fma(2.0 * c, c, -1.0)) + (double)F);
    } else {
      const float c = cos_approx(TWO_PI_F * (float)x);  // -V' = -2 pi A1 c - 4 pi A2 (2 c^2 - 1)
      return (T)fmaf(c, fmaf(-8.0f * 3.14159265358979f * (float)A2, c, -TWO_PI_F * (float)A1),
                     (float)F + 4.0f * 3.14159265358979f * (float)A2);
    }
  } else if (POT == BM_POT_PWL) {
    if (sizeof(T) == 8) {
      const double y = (double)x - 2.0 * floor((double)x * 0.5);  // eq. (2)
      return (T)(((y < 1.0) ? (double)A1 : -(double)A1) + (double)F);
    } else {  // x in [-1, 1) up to a stage excursion: [0, 1) rising branch, [-1, 0) = [1, 2) falling branch
      float y = (float)x;
      y = (y >= 1.0f) ? y - 2.0f : y;
      y = (y < -1.0f) ? y + 2.0f : y;
      return (T)(((y >= 0.0f) ? (float)A1 : -(float)A1) + (float)F);
    }
  } else {
    return -A1 * x + F;
  }
}

template <typename T, int POT, int NOISE>
__global__ void __launch_bounds__(256) bm_paths_literal(const __grid_constant__ SimArgs a) {
  constexpr bool HAS_G = NOISE & BM_NOISE_GAUSS, HAS_P = NOISE & BM_NOISE_POISSON, HAS_D = NOISE & BM_NOISE_DICH;
  constexpr bool F64 = sizeof(T) == 8;
  typedef LitMath<T> M;
  // step counters, countdowns and wrap counts: 32-bit in the fp32 kernel (n_steps < 2^31 there; a countdown beyond the
  // run saturates, which is the same as never firing), 64-bit in the fp64 kernel
  typedef typename std::conditional<F64, long long, int>::type Count;
  constexpr Count COUNT_MAX = F64 ? (Count)0x7FFFFFFFFFFFFFFFLL : (Count)0x7FFFFFFF;
  const int point = blockIdx.x / a.blocks_per_point;
  const int chunk = blockIdx.x - point * a.blocks_per_point;
  const long long p = (long long)chunk * blockDim.x + threadIdx.x;
  Partial mine = partial_zero();

  if (p < a.n_paths) {
    const unsigned long long g = (unsigned long long)point * (unsigned long long)a.n_paths + (unsigned long long)p;
    const bm_params bp = a.params[point];
    const double Ld = POT == BM_POT_SINE2 ? 1.0 : (POT == BM_POT_PWL ? 2.0 : 0.0);
    const double L0 = (POT == BM_POT_QUAD) ? 1.0 : Ld;
    const double dtd = step_length(a, point);
    const T A1 = (T)bp.A1, A2 = (T)bp.A2, F = (T)bp.F, dt = (T)dtd;
    const T inv_dt = (T)(1.0 / dtd);
    const double lam = HAS_P ? bp.lambda : 0.0, zet = HAS_P ? bp.zeta : 0.0;
    const bool onP = HAS_P && lam > 0.0;
    const T a_dt = (T)(lam * zet * dtd);  // a dt, eq. (6): the bias -lambda zeta of the shot noise over one step
    const T step3 = HAS_G ? (T)(sqrt(2.0 * bp.D) * sqrt(3.0 * dtd)) : (T)0;  // G sqrt(3 dt), Alg. 2

    // R4: initial condition (same init-stream call as the jump-adapted kernels)
    const uint4 wi = philox_call(a.keys, g, STREAM_INIT, 0);
    double x0 = (bp.x0_fixed >= 0.0) ? bp.x0_fixed : L0 * ((double)wi.x * (1.0 / 4294967296.0));
    Count wraps = 0;
    if (POT != BM_POT_QUAD) {  // fp64: [0, L) as the oracle; fp32: [-L/2, L/2) (round-to-nearest fold)
      const double k = F64 ? floor(x0 / L0) : rint(x0 / L0);
      x0 -= k * Ld;
      wraps = (Count)k;
    }
    T x = (T)x0;
    // a non-positive rate of leaving -Fa switches the dichotomous source off at this point (as the oracle); a
    // non-positive rate of leaving +Fb makes that state absorbing (infinite sojourn)
    const bool onD = HAS_D && bp.mu_a > 0.0;
    int d = onD ? ((u01_f64(wi.z) < bp.mu_a / (bp.mu_a + (bp.mu_b > 0.0 ? bp.mu_b : 0.0))) ? 1 : 0) : 0;

    // countdowns in grid steps (integers: exact in both precisions)
    Count sP = 0, sD = 0;
    T z = (T)0;
    uint32_t kP = 0, kD = 0;
    const T inv_lam = onP ? (T)(1.0 / lam) : (T)0, zeta = (T)zet;
    const T inv_mua = onD ? (T)(1.0 / bp.mu_a) : (T)0;
    const T inv_mub = (onD && bp.mu_b > 0.0) ? (T)(1.0 / bp.mu_b) : (T)HUGE_VAL;
    auto to_steps = [&](T wait) -> Count {  // [wait / dt], Alg. 3 line 5 / Alg. 4
      const T q = M::floor_(F64 ? wait / dt : wait * inv_dt);
      return q < (F64 ? (T)9.0e18 : (T)2.0e9) ? (Count)q : COUNT_MAX;
    };
    if (onP) {
      const uint4 w = philox_call(a.keys, g, STREAM_POISSON, 0);
      sP = to_steps(M::exp_variate(w.x, inv_lam));
      z = M::exp_variate(w.y, zeta);
    }
    if (HAS_D && onD) {
      const uint4 w = philox_call(a.keys, g, STREAM_DICH, 0);
      sD = to_steps(M::exp_variate(w.x, d ? inv_mub : inv_mua));
    }

    const bool tracing = F64 && a.out_trace != nullptr && (long long)g < a.trace_paths;
    double *trace = tracing ? a.out_trace + (long long)g * a.trace_steps * 2 : nullptr;

    auto fold = [&]() {
      if (POT == BM_POT_QUAD) return;
      if (F64) {
        const double k = floor((double)x / L0);
        if (k != 0.0) {
          double xx = (double)x - k * Ld;
          wraps += (Count)k;
          if (xx < 0.0) { xx += Ld; wraps -= 1; }
          if (xx >= Ld) { xx -= Ld; wraps += 1; }
          x = (T)xx;
        }
      } else {
        const float t = fmaf((float)x, (float)(1.0 / L0), MAGIC_F);
        x = (T)fmaf(t - MAGIC_F, -(float)L0, (float)x);
        wraps += __float_as_int(t) - MAGIC_BITS;
      }
    };

    Count jumps = 0;
    T snap_x = x;
    Count snap_w = wraps;
    uint4 wg = make_uint4(0u, 0u, 0u, 0u);
    if (a.state != nullptr && a.step_begin > 0) {  // row f2: continue a run from its checkpoint
      const StateIO io = state_io(a, g);
      uint32_t lo, hi;
      x = (T)io.getd(0); wraps = (Count)(long long)io.get(1);
      sP = (Count)(long long)io.get(2); sD = (Count)(long long)io.get(3);
      z = (T)io.getd(4);
      io.get2(5, kP, kD);
      io.get2(6, lo, hi); d = (int)lo;
      jumps = (Count)io.getd(7);
      snap_x = (T)io.getd(8); snap_w = (Count)(long long)io.get(9);
      if (HAS_G && (a.step_begin & 3) != 0) wg = philox_call(a.keys, g, STREAM_GAUSS, (uint32_t)(a.step_begin >> 2));
    }
    const Count n_end = (Count)a.step_end, n_snap = (Count)a.n_discard, n_trace = tracing ? (Count)a.trace_steps : 0;
    for (Count n = (Count)a.step_begin; n < n_end; ++n) {
      // Alg. 2: three-point increment with the first moments of a Gaussian of variance 2 D dt
      T dxi = (T)0;
      if (HAS_G) {
        if ((n & 3) == 0) wg = philox_call(a.keys, g, STREAM_GAUSS, (uint32_t)(n >> 2));
        const int j = (int)(n & 3);
        const uint32_t ww = j == 0 ? wg.x : j == 1 ? wg.y : j == 2 ? wg.z : wg.w;
        dxi = ww <= 715827882u ? -step3 : (ww <= 1431655764u ? step3 : (T)0);
      }
      // Alg. 3: kick when the countdown has run out, else count down; the bias -a dt every step
      T deta = (T)0;
      if (HAS_P && onP) {
        if (sP <= 0) {
          deta = z - a_dt;
          jumps += 1;
          kP++;
          const uint4 w = philox_call(a.keys, g, STREAM_POISSON, kP);
          sP = to_steps(M::exp_variate(w.x, inv_lam));
          z = M::exp_variate(w.y, zeta);
        } else {
          sP -= 1;
          deta = -a_dt;
        }
      }
      // Alg. 4: flip when the countdown has run out; the state's force times dt
      T dGam = (T)0;
      if (HAS_D && onD) {
        if (sD <= 0) {
          d = 1 - d;
          jumps += 1;
          kD++;
          const uint4 w = philox_call(a.keys, g, STREAM_DICH, kD);
          sD = to_steps(M::exp_variate(w.x, d ? inv_mub : inv_mua));
        } else {
          sD -= 1;
        }
        dGam = (d ? (T)bp.Fb : -(T)bp.Fa) * dt;
      }
      // Alg. 1 as printed; the static load F (not in the paper) rides with -V'
      const T F1 = lit_force<T, POT>(x, A1, A2, F);
      T xb = x + F1 * dt + dxi;
      T F2 = lit_force<T, POT>(xb, A1, A2, F);
      xb = x + (T)0.5 * (F1 + F2) * dt + dxi;
      F2 = lit_force<T, POT>(xb, A1, A2, F);
      x = x + (T)0.5 * (F1 + F2) * dt + dxi + deta + dGam;
      fold();
      if (tracing && n + 1 <= n_trace) {
        trace[2 * n] = (double)wraps * Ld + (double)x;
        trace[2 * n + 1] = 0.0;
      }
      if (n + 1 == n_snap) { snap_x = x; snap_w = wraps; }
    }
    if (a.state != nullptr) {  // row f2: checkpoint (a float converts to double and back exactly)
      const StateIO io = state_io(a, g);
      io.putd(0, (double)x); io.put(1, (unsigned long long)(long long)wraps);
      io.put(2, (unsigned long long)(long long)sP); io.put(3, (unsigned long long)(long long)sD);
      io.putd(4, (double)z);
      io.put2(5, kP, kD);
      io.put2(6, (uint32_t)d, 0u);
      io.putd(7, (double)jumps);
      io.putd(8, (double)snap_x); io.put(9, (unsigned long long)(long long)snap_w);
    }
    // a10: eq. (30)
    const double span = (double)(a.n_steps - a.n_discard) * dtd;
    const double xT = (double)wraps * Ld + (double)x;
    const double vbar = ((double)(wraps - snap_w) * Ld + ((double)x - (double)snap_x)) / span;
    if (a.out_paths && a.step_end >= a.n_steps) {
      double *o = a.out_paths + g * BM_OUT_STRIDE;
      o[BM_OUT_XT] = xT; o[BM_OUT_VT] = 0.0; o[BM_OUT_VBAR] = vbar; o[BM_OUT_JUMPS] = (double)jumps;
      o[BM_OUT_SUBSTEPS] = (double)a.n_steps; o[BM_OUT_XTI] = (double)snap_w * Ld + (double)snap_x;
    }
    mine = leaf(vbar, xT, (double)jumps, (double)a.n_steps);
  }
  if (a.step_end < a.n_steps) return;  // not the last chunk (uniform over the grid)
  block_reduce_store(mine, a.partials + (long long)blockIdx.x * PARTIAL_STRIDE);
}

}  // namespace bm
