// sim_adaptive.cu -- row f4: the jump-adapted predictor-corrector scheme with dynamic step size control
// from chi = xbar_{n+1} - x_{n+1}, the difference between Alg. 1's predictor (line 4) and corrector (line 6), which
// PAPER.md:237 names as the quantity "to introduce a dynamic time step size control".  The paper gives no controller;
// DESIGN.md reading R14 does: a grid step dt is covered by intervals of length dt 2^-k (k = 0..K), each aligned to a
// multiple of its own length, so every grid point n dt is hit exactly; an interval is integrated as in the
// jump-adapted scheme (sub-steps end on the kicks and flips inside it, one Gaussian per sub-step, number m = running
// sub-step count); no step is rejected (its noise is drawn; a redo would need a Brownian bridge); the largest |chi| of
// an interval halves the NEXT interval if above tol and doubles it if below tol/8 and still aligned.
// fp64, over-damped, one thread = one realization with its own clock (the lanes of a warp are at different times: the
// loop runs until the slowest lane has reached the end).  Same Philox streams, fold and reduction as sim_f64.cuh.
#include "sim_f64.cuh"
#include "dispatch.cuh"

namespace bm {

template <int POT, int NOISE>
__global__ void __launch_bounds__(256) bm_paths_adaptive_f64(const __grid_constant__ SimArgs a) {
  constexpr bool HAS_G = NOISE & BM_NOISE_GAUSS, HAS_P = NOISE & BM_NOISE_POISSON, HAS_D = NOISE & BM_NOISE_DICH;
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
    P.Fa = bp.Fa; P.Fb = bp.Fb; P.mu_a = bp.mu_a;
    P.mu_b = bp.mu_b > 0.0 ? bp.mu_b : 0.0;  // mu_b <= 0: +Fb is absorbing (bm.h: bm_params)
    P.gamma = 0.0; P.amp = 0.0; P.omega = 0.0;
    P.c0 = bp.F - P.lambda * P.zeta;
    const double dt = step_length(a, point);
    const double L0 = (POT == BM_POT_QUAD) ? 1.0 : period_f64<POT>();
    const bool onP = HAS_P && P.lambda > 0.0, onD = HAS_D && P.mu_a > 0.0;
    const int K = a.adapt_levels;
    const long long TPC = 1LL << K;  // ticks per grid step
    const double tol = a.adapt_tol, tol8 = 0.125 * a.adapt_tol;
    // Per level k: the interval length dt 2^-k and the noise amplitude sqrt(2 D H) of a sub-step that covers a whole
    // interval -- the same expressions the time loop used to evaluate per interval and per sub-step (a library scalbn and
    // an fp64 square root each time), so the values are the same bits; a sub-step cut short by an event takes its own root.
    double H_of[21], amp_of[21];
    for (int k = 0; k <= K; ++k) {
      H_of[k] = scalbn(dt, -k);
      amp_of[k] = sqrt(2.0 * P.D * H_of[k]);
    }

    const uint4 wi = philox_call(a.keys, g, STREAM_INIT, 0);  // R4
    StateF64 s;
    s.xi = (bp.x0_fixed >= 0.0) ? bp.x0_fixed : L0 * ((double)wi.x * (1.0 / 4294967296.0));
    s.wraps = 0;
    s.v = 0.0;
    fold_f64<POT>(s);
    int d = onD ? ((u01_f64(wi.z) < P.mu_a / (P.mu_a + P.mu_b)) ? 1 : 0) : -1;
    uint32_t kP = 0, kD = 0;
    double rP = 0.0, rD = 0.0, z = 0.0;
    if (onP) {
      const uint4 w = philox_call(a.keys, g, STREAM_POISSON, 0);
      rP = -log(u01_f64(w.x)) / P.lambda;
      z = -P.zeta * log(u01_f64(w.y));
    }
    if (onD) {
      const uint4 w = philox_call(a.keys, g, STREAM_DICH, 0);
      rD = -log(u01_f64(w.x)) / (d ? P.mu_b : P.mu_a);
    }
    const bool tracing = a.out_trace != nullptr && (long long)g < a.trace_paths;
    double *trace = tracing ? a.out_trace + (long long)g * a.trace_steps * 2 : nullptr;

    unsigned long long m = 0;
    double jumps = 0.0, gq[4] = {0.0, 0.0, 0.0, 0.0};
    StateF64 snap = s;
    int k = 0;
    for (long long n = 0; n < a.n_steps; ++n) {
      long long tick = 0;
      while (tick < TPC) {
        const long long wd = TPC >> k;                  // interval width in ticks
        const double H = H_of[k];                       // its length, exactly dt 2^-k
        const double ampH = amp_of[k];
        double rem = H, chi_max = 0.0;
        while (rem > 0.0) {
          double h = rem;
          if (onP && rP < h) h = rP;
          if (onD && rD < h) h = rD;
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
          const double cst = P.c0 + (onD ? (d ? P.Fb : -P.Fa) : 0.0);
          const double dxi = HAS_G ? ((h == H) ? ampH : amp_of_substep_f64(P.D, h)) * gn : 0.0;
          // Alg. 1; chi = predictor (line 4) - corrector (line 6)
          const double x = s.xi;
          const double F1 = minus_dV_f64<POT>(P, x) + cst;
          double xb = x + F1 * h + dxi;
          double F2 = minus_dV_f64<POT>(P, xb) + cst;
          xb = x + 0.5 * (F1 + F2) * h + dxi;
          F2 = minus_dV_f64<POT>(P, xb) + cst;
          s.xi = x + 0.5 * (F1 + F2) * h + dxi;
          chi_max = fmax(chi_max, fabs(xb - s.xi));
          rem -= h;
          if (onP) {
            rP -= h;
            if (rP <= 0.0) {
              s.xi += z;
              jumps += 1.0;
              kP++;
              const uint4 w = philox_call(a.keys, g, STREAM_POISSON, kP);
              rP = -log(u01_f64(w.x)) / P.lambda;
              z = -P.zeta * log(u01_f64(w.y));
            }
          }
          if (onD) {
            rD -= h;
            if (rD <= 0.0) {
              d = 1 - d;
              jumps += 1.0;
              kD++;
              const uint4 w = philox_call(a.keys, g, STREAM_DICH, kD);
              rD = -log(u01_f64(w.x)) / (d ? P.mu_b : P.mu_a);
            }
          }
          fold_f64<POT>(s);
        }
        tick += wd;
        if (chi_max > tol && k < K) k += 1;
        else if (chi_max < tol8 && k > 0 && (tick & (2 * wd - 1)) == 0) k -= 1;  // wd is a power of two: aligned to 2 wd
      }
      if (tracing && n + 1 <= a.trace_steps) {
        trace[2 * n] = unfolded_f64<POT>(s);
        trace[2 * n + 1] = 0.0;
      }
      if (n + 1 == a.n_discard) snap = s;
    }
    const double span = (double)(a.n_steps - a.n_discard) * dt;
    const double xT = unfolded_f64<POT>(s);
    const double vbar = ((double)(s.wraps - snap.wraps) * period_f64<POT>() + (s.xi - snap.xi)) / span;
    if (a.out_paths) {
      double *o = a.out_paths + g * BM_OUT_STRIDE;
      o[BM_OUT_XT] = xT; o[BM_OUT_VT] = 0.0; o[BM_OUT_VBAR] = vbar; o[BM_OUT_JUMPS] = jumps;
      o[BM_OUT_SUBSTEPS] = (double)m; o[BM_OUT_XTI] = unfolded_f64<POT>(snap);
    }
    mine = leaf(vbar, xT, jumps, (double)m);
  }
  block_reduce_store(mine, a.partials + (long long)blockIdx.x * PARTIAL_STRIDE);
}

template <int POT>
static KernelFn pick_noise_ad(int noise) {
  switch (noise & 7) {
    case 0: return bm_paths_adaptive_f64<POT, 0>;
    case 1: return bm_paths_adaptive_f64<POT, 1>;
    case 2: return bm_paths_adaptive_f64<POT, 2>;
    case 3: return bm_paths_adaptive_f64<POT, 3>;
    case 4: return bm_paths_adaptive_f64<POT, 4>;
    case 5: return bm_paths_adaptive_f64<POT, 5>;
    case 6: return bm_paths_adaptive_f64<POT, 6>;
    default: return bm_paths_adaptive_f64<POT, 7>;
  }
}

KernelFn pick_adaptive_f64(int potential, int noise) {
  switch (potential) {
    case BM_POT_SINE2: return pick_noise_ad<BM_POT_SINE2>(noise);
    case BM_POT_PWL: return pick_noise_ad<BM_POT_PWL>(noise);
    case BM_POT_QUAD: return pick_noise_ad<BM_POT_QUAD>(noise);
    default: return nullptr;
  }
}

}  // namespace bm
