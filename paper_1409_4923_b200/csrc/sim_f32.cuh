// sim_f32.cuh -- fp32 path kernel (the throughput kernel).  One thread = one realization; position, clocks,
// Gaussian cache and observable snapshot stay in registers for the whole run.
//
// Same method as the fp64 kernel (R1-R9), but arranged for fp32 accuracy and for the SM's pipes:
//  * x is kept folded to [-1/2, 1/2) periods plus an int32 wrap counter, re-folded after
//    every sub-step with a round-to-nearest "magic add" (no F2I/FRND, which share the 16-lane XU pipe);
//  * time is (cell index n, offset tau in the cell); a jump clock is (cells to go, offset in its cell), so
//    nothing small is ever subtracted from something large (a float countdown would drift: DESIGN.md s.5);
//  * uniforms come from the top 23 bits of a Philox word through a mantissa splice (no I2F);
//  * transcendental functions: MUFU.{COS,SIN,LG2,SQRT} (SFU variant) or, for the force cosine,
//    an even polynomial on the FMA pipe (FMA variant) -- a measured choice (DESIGN.md s.6).
// fp32 results are judged statistically against the fp64 oracle (3 combined standard errors); because both
// use the same Philox words for the same purpose they are in fact strongly correlated path by path.
#pragma once
#include "common.cuh"

namespace bm {

__device__ __forceinline__ float cos_approx(float x) { float r; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sin_approx(float x) { float r; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float lg2_approx(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_approx(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

constexpr float TWO_PI_F = 6.283185307179586f;
constexpr float LN2_F = 0.6931471805599453f;

// u in (0,1] on a 2^-23 grid: ((w>>9)+1) 2^-23 ~ u(w) of R3 rounded up; exact float arithmetic.
__device__ __forceinline__ float u01_open0_f32(uint32_t w) { return 2.0f - __uint_as_float((w >> 9) ^ 0x3FFFFFFFu); }
// 1 + (w>>9) 2^-23 in [1,2): one period of phase, to be used modulo 1
__device__ __forceinline__ float turns12_f32(uint32_t w) { return __uint_as_float((w >> 9) | 0x3F800000u); }
// -ln u(w) >= 0
__device__ __forceinline__ float neg_log_u_f32(uint32_t w) { return -LN2_F * lg2_approx(u01_open0_f32(w)); }

// cos(2 pi x), x in periods.  SFU: FMUL, FMUL.RZ, MUFU.COS.  FMA: reduce to r in [-1/2,1/2] and evaluate an even
// polynomial in r (degree 12, |err| < 5e-7) -- 2 FADD + FMUL + 6 FFMA on the FMA pipe.
template <int SINCOS>
__device__ __forceinline__ float cos2pi(float x) {
  if (SINCOS == BM_SINCOS_SFU) {
    return cos_approx(x * TWO_PI_F);
  } else {
    const float magic = 12582912.0f;  // 1.5 * 2^23
    const float k = (x + magic) - magic;
    const float r = x - k;
    const float s = r * r;
    // cos(2 pi r) = sum c_j s^j, s = r^2 in [0,1/4]: Chebyshev-node interpolant of degree 6 in s
    // (approximation error 1.1e-8, fp32 Horner rounding ~4e-7: the same class as MUFU.COS)
    float p = 6.527705963e+00f;
    p = fmaf(p, s, -2.596688461e+01f);
    p = fmaf(p, s, 6.016742979e+01f);
    p = fmaf(p, s, -8.545011343e+01f);
    p = fmaf(p, s, 6.493911593e+01f);
    p = fmaf(p, s, -1.973920447e+01f);
    p = fmaf(p, s, 9.999999889e-01f);
    return p;
  }
}

// Box-Muller pair (R3), fp32: r = sqrt(-2 ln u(wa)), angle 2 pi u(wb)
__device__ __forceinline__ void box_muller_f32(uint32_t wa, uint32_t wb, float &g0, float &g1) {
  const float r = sqrt_approx(-2.0f * LN2_F * lg2_approx(u01_open0_f32(wa)));
  const float ang = turns12_f32(wb) * TWO_PI_F;
  g0 = r * cos_approx(ang);
  g1 = r * sin_approx(ang);
}

// Per-point constants, fp32
struct PointF32 {
  float K1, K2;      // SINE2: -V'(x) = K0 + c (K1 + K2 c), c = cos 2 pi x, in PERIODS per unit time (L = 1)
  float base;        // F - lambda zeta (+ 4 pi A2 for SINE2)
  float Ga, Gb;      // -Fa, +Fb
  float sdt;         // sqrt(2 D dt)  (position units)
  float D2;          // 2 D
  float inv_lam_dt;  // 1/(lambda dt): waiting time in cells = -ln u * inv_lam_dt
  float zeta;
  float inv_mua_dt, inv_mub_dt;
  float gamma;
  float amp, w_turns;  // drive amplitude, omega/(2 pi)
  float A1;            // PWL / QUAD slope
};

template <int POT, int SINCOS>
__device__ __forceinline__ float force_f32(const PointF32 &P, float x, float cst) {
  // x in position units; SINE2 has L = 1 so position == periods
  if (POT == BM_POT_SINE2) {
    const float c = cos2pi<SINCOS>(x);
    return fmaf(c, fmaf(P.K2, c, P.K1), cst);
  } else if (POT == BM_POT_PWL) {
    // folded x in [-1,1): -V' = +A1 on [0,1), -A1 on [-1,0); stage values may step outside by a little
    float y = x;
    y = (y >= 1.0f) ? y - 2.0f : y;
    y = (y < -1.0f) ? y + 2.0f : y;
    return cst + ((y >= 0.0f) ? P.A1 : -P.A1);
  } else {
    return fmaf(-P.A1, x, cst);
  }
}

// fold x to [-L/2, L/2) by round-to-nearest; accumulates the raw "magic" integers (a9)
template <int POT>
__device__ __forceinline__ void fold_f32(float &x, int &wraps) {
  if (POT == BM_POT_QUAD) return;
  const float magic = 12582912.0f;  // 1.5*2^23: (y + magic) has ulp 1 -> rounds y to nearest integer
  if (POT == BM_POT_SINE2) {
    const float t = x + magic;
    x -= (t - magic);
    wraps += __float_as_int(t) - 0x4B400000;
  } else {  // L = 2
    const float t = fmaf(x, 0.5f, magic);
    x = fmaf(t - magic, -2.0f, x);
    wraps += __float_as_int(t) - 0x4B400000;
  }
}

template <int POT>
__device__ __forceinline__ float period_f32() { return POT == BM_POT_SINE2 ? 1.0f : (POT == BM_POT_PWL ? 2.0f : 0.0f); }

// (cells to go, offset in that cell) of an event W cells ahead of offset tau (in units of dt)
__device__ __forceinline__ void schedule_f32(float tau, float dt, float inv_dt, float Wcells, int &cells, float &off) {
  const float q = fmaf(tau, inv_dt, Wcells);
  float c = floorf(q);
  float f = (q - c) * dt;
  if (f >= dt) { f = 0.0f; c += 1.0f; }
  if (c == 0.0f) f = fmaxf(f, tau);  // never schedule into the past of this cell
  c = fminf(c, 2.0e9f);
  cells = (int)c;
  off = f;
}

template <int MODEL, int POT, int NOISE, int SINCOS>
__global__ void __launch_bounds__(256) bm_paths_f32(const __grid_constant__ SimArgs a) {
  constexpr bool HAS_G = NOISE & BM_NOISE_GAUSS, HAS_P = NOISE & BM_NOISE_POISSON, HAS_D = NOISE & BM_NOISE_DICH;
  constexpr bool INERTIAL = MODEL == BM_INERTIAL;
  const int point = blockIdx.x / a.blocks_per_point;
  const int chunk = blockIdx.x - point * a.blocks_per_point;
  const long long p = (long long)chunk * blockDim.x + threadIdx.x;
  Partial mine = partial_zero();

  if (p < a.n_paths) {
    const unsigned long long g = (unsigned long long)point * (unsigned long long)a.n_paths + (unsigned long long)p;
    const bm_params bp = a.params[point];
    const float dt = (float)a.dt;
    const float inv_dt = (float)(1.0 / a.dt);
    const double lam = HAS_P ? bp.lambda : 0.0, zet = HAS_P ? bp.zeta : 0.0, Dd = HAS_G ? bp.D : 0.0;
    PointF32 P;
    if (POT == BM_POT_SINE2) {
      // -V' = -2 pi A1 c - 4 pi A2 (2 c^2 - 1)
      P.K1 = (float)(-2.0 * M_PI * bp.A1);
      P.K2 = (float)(-8.0 * M_PI * bp.A2);
      P.base = (float)(bp.F - lam * zet + 4.0 * M_PI * bp.A2);
    } else {
      P.K1 = 0.f; P.K2 = 0.f;
      P.base = (float)(bp.F - lam * zet);
    }
    P.A1 = (float)bp.A1;
    P.Ga = (float)(-bp.Fa); P.Gb = (float)bp.Fb;
    P.sdt = (float)sqrt(2.0 * Dd * a.dt);
    P.D2 = (float)(2.0 * Dd);
    P.inv_lam_dt = (lam > 0.0) ? (float)(1.0 / (lam * a.dt)) : 0.f;
    P.zeta = (float)zet;
    P.inv_mua_dt = (HAS_D && bp.mu_a > 0.0) ? (float)(1.0 / (bp.mu_a * a.dt)) : 0.f;
    P.inv_mub_dt = (HAS_D && bp.mu_b > 0.0) ? (float)(1.0 / (bp.mu_b * a.dt)) : 0.f;
    P.gamma = (float)bp.gamma;
    P.amp = (float)bp.amp;
    P.w_turns = (float)(bp.omega / (2.0 * M_PI));
    const float L = period_f32<POT>();

    // R4: initial condition
    const uint4 wi = philox_call(a.keys, g, STREAM_INIT, 0);
    float x;
    int wraps = 0;
    {
      const double L0 = (POT == BM_POT_QUAD) ? 1.0 : (double)L;
      const double x0 = (bp.x0_fixed >= 0.0) ? bp.x0_fixed : L0 * ((double)wi.x * (1.0 / 4294967296.0));
      if (POT == BM_POT_QUAD) {
        x = (float)x0;
      } else {  // fold in fp64 once
        const double k = rint(x0 / L0);
        x = (float)(x0 - k * L0);
        wraps = (int)k;
        fold_f32<POT>(x, wraps);
      }
    }
    float v = 0.f;
    if (INERTIAL) v = (float)(bp.v0_lo + (bp.v0_hi - bp.v0_lo) * (((double)wi.y + 0.5) * (1.0 / 4294967296.0)));
    int d = 0;
    if (HAS_D) d = ((((double)wi.z + 0.5) * (1.0 / 4294967296.0)) < bp.mu_a / (bp.mu_a + bp.mu_b)) ? 1 : 0;

    // jump clocks: (cells to go, offset inside that cell)
    int cP = 0x7FFFFFFF, cD = 0x7FFFFFFF;
    float fP = 0.f, fD = 0.f, z = 0.f;
    uint32_t kP = 0, kD = 0;
    if (HAS_P && lam > 0.0) {
      const uint4 w = philox_call(a.keys, g, STREAM_POISSON, 0);
      schedule_f32(0.f, dt, inv_dt, neg_log_u_f32(w.x) * P.inv_lam_dt, cP, fP);
      z = P.zeta * neg_log_u_f32(w.y);
    }
    if (HAS_D) {
      const uint4 w = philox_call(a.keys, g, STREAM_DICH, 0);
      schedule_f32(0.f, dt, inv_dt, neg_log_u_f32(w.x) * (d ? P.inv_mub_dt : P.inv_mua_dt), cD, fD);
    }

    // drive phase in 2^-64 turns per cell (inertial): exact integer accumulation, no float time
    unsigned long long ph = 0, dph = 0;
    float drive0 = 0.f;
    if (INERTIAL) {
      double turns_per_cell = bp.omega * a.dt / (2.0 * M_PI);
      turns_per_cell -= floor(turns_per_cell);
      dph = (unsigned long long)(turns_per_cell * 18446744073709551616.0);
      drive0 = P.amp;  // cos(0)
    }

    const int n_steps = (int)a.n_steps, n_discard = (int)a.n_discard;
    int n = 0;
    uint32_t blk = 0;  // Gaussian block counter = m/4
    float tau = 0.f;
    int jumps = 0;
    uint32_t m = 0;
    float snap_x = x;
    int snap_w = wraps;
    float cst = P.base + (HAS_D ? (d ? P.Gb : P.Ga) : 0.f);

    while (n < n_steps) {
      float gq[4] = {0.f, 0.f, 0.f, 0.f};
      if (HAS_G) {
        const uint4 w = philox_call(a.keys, g, STREAM_GAUSS, blk);
        box_muller_f32(w.x, w.y, gq[0], gq[1]);
        box_muller_f32(w.z, w.w, gq[2], gq[3]);
      }
      blk++;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        // a5: sub-step ends at the earliest of {grid point, kick, flip} inside this cell
        float end = dt;
        float eP = dt, eD = dt;
        if (HAS_P) { eP = (cP == 0) ? fP : dt; end = fminf(end, eP); }
        if (HAS_D) { eD = (cD == 0) ? fD : dt; end = fminf(end, eD); }
        const float h = end - tau;
        const float hh = 0.5f * h;
        float dxi = 0.f;
        if (HAS_G) {
          float ampl = P.sdt;
          if (h != dt) ampl = sqrt_approx(P.D2 * h);
          dxi = ampl * gq[j];
        }
        m++;
        if (!INERTIAL) {
          // a6: Alg. 1
          const float xs = x + dxi;
          const float F1 = force_f32<POT, SINCOS>(P, x, cst);
          float xb = fmaf(F1, h, xs);
          float F2 = force_f32<POT, SINCOS>(P, xb, cst);
          xb = fmaf(F1 + F2, hh, xs);
          F2 = force_f32<POT, SINCOS>(P, xb, cst);
          x = fmaf(F1 + F2, hh, xs);
        } else {
          // a7: R7; drive at t (carried over) and at t+h (one new cosine)
          const float ph_f = __uint_as_float((uint32_t)(ph >> 41) | 0x3F800000u);  // [1,2) turns at the cell start
          const float drive1 = P.amp * cos2pi<SINCOS>(fmaf(end, P.w_turns, ph_f));
          const float vs = v + dxi;
          const float b0 = cst + drive0, b1 = cst + drive1;
          const float A1v = fmaf(-P.gamma, v, force_f32<POT, SINCOS>(P, x, b0));
          float xb = fmaf(v, h, x);
          float vb = fmaf(A1v, h, vs);
          float A2v = fmaf(-P.gamma, vb, force_f32<POT, SINCOS>(P, xb, b1));
          xb = fmaf(v + vb, hh, x);
          vb = fmaf(A1v + A2v, hh, vs);
          A2v = fmaf(-P.gamma, vb, force_f32<POT, SINCOS>(P, xb, b1));
          x = fmaf(v + vb, hh, x);
          v = fmaf(A1v + A2v, hh, vs);
          drive0 = drive1;
        }
        tau = end;
        if (HAS_P) {
          if (cP == 0 && end == eP) {  // a8: kick
            if (!INERTIAL) x += z; else v += z;
            jumps++;
            kP++;
            const uint4 w = philox_call(a.keys, g, STREAM_POISSON, kP);
            schedule_f32(tau, dt, inv_dt, neg_log_u_f32(w.x) * P.inv_lam_dt, cP, fP);
            z = P.zeta * neg_log_u_f32(w.y);
            if (POT != BM_POT_QUAD && !INERTIAL) {  // a kick may span several periods: fold with full range
              const float k = rintf(x / L);
              x = fmaf(-k, L, x);
              wraps += (int)k;
            }
          }
        }
        if (HAS_D) {
          if (cD == 0 && end == eD) {  // a8: flip
            d ^= 1;
            jumps++;
            kD++;
            cst = P.base + (d ? P.Gb : P.Ga);
            const uint4 w = philox_call(a.keys, g, STREAM_DICH, kD);
            schedule_f32(tau, dt, inv_dt, neg_log_u_f32(w.x) * (d ? P.inv_mub_dt : P.inv_mua_dt), cD, fD);
          }
        }
        fold_f32<POT>(x, wraps);
        if (end == dt) {  // grid point reached
          n++;
          tau = 0.f;
          if (HAS_P) cP--;
          if (HAS_D) cD--;
          if (INERTIAL) ph += dph;
          if (n == n_discard) { snap_x = x; snap_w = wraps; }
          if (n >= n_steps) break;
        }
      }
    }
    // a10: eq. (30), assembled once per path in fp64
    const double Ld = (double)L;
    const double span = (double)(a.n_steps - a.n_discard) * a.dt;
    const double xT = (double)wraps * Ld + (double)x;
    const double xTi = (double)snap_w * Ld + (double)snap_x;
    const double vbar = ((double)(wraps - snap_w) * Ld + ((double)x - (double)snap_x)) / span;
    if (a.out_paths) {
      double *o = a.out_paths + g * BM_OUT_STRIDE;
      o[BM_OUT_XT] = xT; o[BM_OUT_VT] = (double)v; o[BM_OUT_VBAR] = vbar; o[BM_OUT_JUMPS] = (double)jumps;
      o[BM_OUT_SUBSTEPS] = (double)m; o[BM_OUT_XTI] = xTi;
    }
    mine = leaf(vbar, xT, (double)jumps, (double)m);
  }
  block_reduce_store(mine, a.partials + (long long)blockIdx.x * PARTIAL_STRIDE);
}

}  // namespace bm
