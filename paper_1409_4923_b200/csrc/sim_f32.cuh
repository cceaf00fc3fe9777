// sim_f32.cuh -- fp32 path kernel (the throughput kernel), v2.  One thread = one realization; position, clocks,
// Gaussian cache and observable snapshot stay in registers for the whole run.
//
// Same method as the fp64 kernel (R1-R9), arranged for fp32 accuracy and for the SM's pipes
// (profiles/r1_c1_f32_v1.md is the measurement this layout answers):
//  * the position is carried as theta = 2 pi x / L (radians of the potential's phase), folded to [-pi, pi) with an
//    int32 wrap counter by a round-to-nearest "magic add" (no F2I/FRND, which share the 16-lane XU
//    pipe with MUFU).  In these units a force cosine is FMUL.RZ + MUFU.COS with no scaling multiply in front;
//  * Alg. 1 is evaluated with the step length folded into the constants:
//    x1 = (xs + h K0) + c (h K1 + h K2 c), so every stage is 2 FFMA behind its cosine;
//  * time is (cell index n, offset tau in the cell); a jump clock is (cell index, offset in that cell), so nothing
//    small is ever subtracted from something large;
//  * a warp takes the FAST path (full grid step, all constants hoisted) when no lane has a jump or an observable
//    boundary in its current cell (one vote), else every lane takes the GENERAL sub-step (a5-a8);
//  * the Box-Muller radius carries the noise amplitude (sqrt(-2 ln u) * sqrt(2 D dt) in one MUFU.SQRT);
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
constexpr float INV_TWO_PI_F = 0.15915494309189535f;
constexpr float LN2_F = 0.6931471805599453f;
constexpr float MAGIC_F = 12582912.0f;  // 1.5 * 2^23: (y + MAGIC) has ulp 1, i.e. rounds y to the nearest integer
constexpr int MAGIC_BITS = 0x4B400000;

// u in (0,1] on a 2^-23 grid: ((w>>9)+1) 2^-23 ~ u(w) of R3 rounded up; exact float arithmetic.
__device__ __forceinline__ float u01_open0_f32(uint32_t w) { return __uint_as_float((w >> 9) | 0x3F800000u) - 0.99999988079071044921875f; }
// 1 + (w>>9) 2^-23 in [1,2): one period of phase, to be used modulo 1
__device__ __forceinline__ float turns12_f32(uint32_t w) { return __uint_as_float((w >> 9) | 0x3F800000u); }
// -ln u(w) >= 0
__device__ __forceinline__ float neg_log_u_f32(uint32_t w) { return -LN2_F * lg2_approx(u01_open0_f32(w)); }

// cos(2 pi t), t in turns, on the FMA pipe: reduce to r in [-1/2,1/2], even polynomial of degree 6 in r^2
// (Chebyshev-node interpolant; approximation error 1.1e-8, fp32 Horner rounding ~4e-7: the class of MUFU.COS).
__device__ __forceinline__ float cos_turns_poly(float t) {
  const float k = (t + MAGIC_F) - MAGIC_F;
  const float r = t - k;
  const float s = r * r;
  float p = 6.527705963e+00f;
  p = fmaf(p, s, -2.596688461e+01f);
  p = fmaf(p, s, 6.016742979e+01f);
  p = fmaf(p, s, -8.545011343e+01f);
  p = fmaf(p, s, 6.493911593e+01f);
  p = fmaf(p, s, -1.973920447e+01f);
  p = fmaf(p, s, 9.999999889e-01f);
  return p;
}

// cos(theta), theta in radians.  SFU: FMUL.RZ (the 1/2pi of cos.approx) + MUFU.COS.
template <int SINCOS>
__device__ __forceinline__ float cos_theta(float th) {
  return SINCOS == BM_SINCOS_SFU ? cos_approx(th) : cos_turns_poly(th * INV_TWO_PI_F);
}
// cos(2 pi t), t in turns
template <int SINCOS>
__device__ __forceinline__ float cos_turns(float t) {
  return SINCOS == BM_SINCOS_SFU ? cos_approx(t * TWO_PI_F) : cos_turns_poly(t);
}

// Box-Muller pair (R3), fp32 standard normals: r = sqrt(-2 ln u(wa)), angle 2 pi u(wb).  (bm_gauss_fill.)
__device__ __forceinline__ void box_muller_f32(uint32_t wa, uint32_t wb, float &g0, float &g1) {
  const float r = sqrt_approx(-2.0f * LN2_F * lg2_approx(u01_open0_f32(wa)));
  const float ang = turns12_f32(wb) * TWO_PI_F;
  g0 = r * cos_approx(ang);
  g1 = r * sin_approx(ang);
}
// The same pair left in factors, with the amplitude inside the root: r = sqrt(cn * lg2 u), cn = -2 ln2 * s^2,
// so that s*g0 = r*c and s*g1 = r*s cost one FFMA each at the point of use.
__device__ __forceinline__ void box_muller_factors_f32(uint32_t wa, uint32_t wb, float cn, float &r, float &c, float &s) {
  r = sqrt_approx(cn * lg2_approx(u01_open0_f32(wa)));
  const float ang = turns12_f32(wb) * TWO_PI_F;
  c = cos_approx(ang);
  s = sin_approx(ang);
}

// theta units: theta = SCALE * x; the potential has period PERIOD_TH in theta and PERIOD_X in x
template <int POT> struct Units {
  static constexpr float SCALE = POT == BM_POT_SINE2 ? TWO_PI_F : 1.0f;
  static constexpr float PERIOD_TH = POT == BM_POT_SINE2 ? TWO_PI_F : 2.0f;
  static constexpr float INV_PERIOD_TH = POT == BM_POT_SINE2 ? INV_TWO_PI_F : 0.5f;
  static constexpr double PERIOD_X = POT == BM_POT_SINE2 ? 1.0 : (POT == BM_POT_PWL ? 2.0 : 0.0);
};

// a9: fold theta to [-P/2, P/2) by round-to-nearest (any magnitude below 2^22 periods) and count the wraps
template <int POT>
__device__ __forceinline__ void fold_f32(float &x, int &wraps) {
  if (POT == BM_POT_QUAD) return;
  const float t = fmaf(x, Units<POT>::INV_PERIOD_TH, MAGIC_F);
  x = fmaf(t - MAGIC_F, -Units<POT>::PERIOD_TH, x);
  wraps += __float_as_int(t) - MAGIC_BITS;
}

// base + s * (-V'(x)) for a step-scaled potential: SINE2: c (k1 + k2 c), c = cos theta (the constant part of
// -V' travels in `base`); PWL (eq. 2; x in [-1,1) up to a stage excursion): +-k1; QUAD: -k1 x.
template <int POT, int SINCOS>
__device__ __forceinline__ float stage_f32(float base, float x, float k1, float k2) {
  if (POT == BM_POT_SINE2) {
    const float c = cos_theta<SINCOS>(x);
    return fmaf(c, fmaf(k2, c, k1), base);
  } else if (POT == BM_POT_PWL) {
    float y = x;
    y = (y >= 1.0f) ? y - 2.0f : y;
    y = (y < -1.0f) ? y + 2.0f : y;
    return base + ((y >= 0.0f) ? k1 : -k1);
  } else {
    return fmaf(-k1, x, base);
  }
}

// a6: Alg. 1 over a sub-step h with drift a(x) = K0 + f(x), f = -V' without its constant:
//   x1 = xs + h a(x);  x2 = xs + h/2 (a(x) + a(x1));  x' = xs + h/2 (a(x) + a(x2)),   xs = x + noise.
// k0 = h K0, k1 = h K1, k2 = h K2 (and their halves).  With xh = (xs + x1)/2 + k0/2 = xs + h/2 a(x) + k0/2 the
// last two stages are xh + (h/2) f(.).  `xarg` is where a(x) is evaluated (x before folding: same angle).
template <int POT, int SINCOS>
__device__ __forceinline__ float pc_overdamped_f32(float xarg, float xs, float k0, float k1, float k2, float k0h,
                                                   float k1h, float k2h) {
  const float x1 = stage_f32<POT, SINCOS>(xs + k0, xarg, k1, k2);
  const float xh = fmaf(0.5f, x1, fmaf(0.5f, xs, k0h));
  const float x2 = stage_f32<POT, SINCOS>(xh, x1, k1h, k2h);
  return stage_f32<POT, SINCOS>(xh, x2, k1h, k2h);
}

// a7: R7.  y = (x, v), A = (v, -gamma v + f(x) + b(t)); noise in v only (vs = v + noise).  b0 = constant force +
// drive at t, b1 = the same at t + h; kk1, kk2 are the (unscaled) potential constants in theta units.
template <int SINCOS>
__device__ __forceinline__ void pc_inertial_f32(float &x, float &v, float xf, float vs, float h, float hh, float gamma,
                                                float kk1, float kk2, float b0, float b1) {
  const float c1 = cos_theta<SINCOS>(x);
  const float xb1 = fmaf(h, v, xf);
  const float c2 = cos_theta<SINCOS>(xb1);  // does not wait for c1
  const float a1 = fmaf(c1, fmaf(kk2, c1, kk1), fmaf(-gamma, v, b0));
  const float vb1 = fmaf(h, a1, vs);
  const float xh = fmaf(hh, v, xf), vh = fmaf(hh, a1, vs);
  const float a2 = fmaf(c2, fmaf(kk2, c2, kk1), fmaf(-gamma, vb1, b1));
  const float xb2 = fmaf(hh, vb1, xh);
  const float c3 = cos_theta<SINCOS>(xb2);
  const float vb2 = fmaf(hh, a2, vh);
  const float a3 = fmaf(c3, fmaf(kk2, c3, kk1), fmaf(-gamma, vb2, b1));
  x = fmaf(hh, vb2, xh);
  v = fmaf(hh, a3, vh);
}

// Cell index and offset of an event W cells after (n, tau); offsets are in time units, 0 <= off < dt.
__device__ __forceinline__ void schedule_f32(int n, float tau, float dt, float inv_dt, float Wcells, int &cell, float &off) {
  const float q = fmaf(tau, inv_dt, Wcells);
  float c = floorf(q);
  float f = (q - c) * dt;
  if (f >= dt) { f = 0.0f; c += 1.0f; }
  if (c == 0.0f) f = fmaxf(f, tau);  // never schedule into the past of this cell
  c = fminf(c, 2.0e9f);
  const long long t = (long long)n + (long long)c;
  cell = t > 0x7FFFFFFFLL ? 0x7FFFFFFF : (int)t;
  off = f;
}


// ---- warp specialisation: Gaussian producer warps feed the stepping (consumer) warps through shared memory -----
// The three cosines of Alg. 1 are one serial chain (~90 cycles per step for a lone warp, measured) and C1 gives a
// scheduler only 3-4 path warps, so a kernel that also draws its normals in the path warp is latency bound
// (profiles/r1_c1_f32_v2.md).  Philox + Box-Muller have no serial dependence at all (counter-based, R1-R2), so they
// move to a partner warp of the same block: consumer warp w steps 32 paths, producer warp w + W draws the normals
// of exactly those paths (lane l <-> lane l) STAGE by STAGE into a ring; the hardware scheduler then fills the
// consumer's latency bubbles with producer instructions.
constexpr int RING_STAGES = 3;  // stages in flight per warp pair
constexpr int RING_BLOCKS = 4;  // Gaussian blocks (4 normals each) per stage = 16 sub-steps
struct GaussSlot {              // one Gaussian block of one warp: (ra, ca, sa, rb), (cb, sb) per lane; 768 B
  float4 a[32];
  float2 b[32];
};
struct PairRing {
  GaussSlot slot[RING_STAGES][RING_BLOCKS];
  unsigned long long full[RING_STAGES], empty[RING_STAGES];  // mbarriers, one arrival each (lane 0 of the warp)
  int done;  // consumer -> producer: no more stages needed
  int pad[3];
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(void *bar) {  // release at CTA scope
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(void *bar, uint32_t parity) {  // acquire at CTA scope
  uint32_t ok;
  asm volatile(
      "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
// the same with a suspend-time hint (ns): the waiting warp leaves the issue slots to the others
__device__ __forceinline__ bool mbar_try_wait_hint(void *bar, uint32_t parity, uint32_t ns) {
  uint32_t ok;
  asm volatile(
      "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\nselp.u32 %0, 1, 0, p;\n}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity), "r"(ns)
      : "memory");
  return ok != 0;
}

// Gaussian cache: one Philox call = two Box-Muller pairs = the normals of four consecutive sub-steps (R2, R3),
// kept as (radius, cos, sin) factors with the full-step amplitude inside the radius.
struct Gauss4 { float ra, ca, sa, rb, cb, sb; };

__device__ __forceinline__ Gauss4 draw_gauss_f32(const PhiloxKeys &K, unsigned long long g, uint32_t b, float cn) {
  Gauss4 q;
  const uint4 w = philox_call(K, g, STREAM_GAUSS, b);
  box_muller_factors_f32(w.x, w.y, cn, q.ra, q.ca, q.sa);
  box_muller_factors_f32(w.z, w.w, cn, q.rb, q.cb, q.sb);
  return q;
}

// Per-point constants, fp32, theta units (theta = SCALE x)
struct PointF32 {
  float kk1, kk2;    // SINE2: SCALE * (-V') = base-part + c (kk1 + kk2 c), c = cos theta.  PWL/QUAD: kk1 = A1
  float base;        // SCALE * (F - lambda zeta (+ 4 pi A2 for SINE2))
  float Ga, Gb;      // SCALE * (-Fa), SCALE * (+Fb)
  float cn;          // -2 ln2 * SCALE^2 * 2 D dt: Box-Muller radius^2 per unit of lg2 u, full grid step
  float inv_lam_dt;  // 1/(lambda dt): waiting time in cells = -ln u * inv_lam_dt
  float zeta;        // SCALE * zeta
  float inv_mua_dt, inv_mub_dt;
  float gamma;
  float amp;         // SCALE * drive amplitude
  float w_turns;     // omega/(2 pi): drive turns per unit time
};

// WS = warp specialised (blockDim.x = 2 x path threads; needs dynamic shared memory of one PairRing per path warp)
template <int MODEL, int POT, int NOISE, int SINCOS, bool WS>
__global__ void __launch_bounds__(512) bm_paths_f32(const __grid_constant__ SimArgs a) {
  constexpr bool HAS_G = NOISE & BM_NOISE_GAUSS, HAS_P = NOISE & BM_NOISE_POISSON, HAS_D = NOISE & BM_NOISE_DICH;
  constexpr bool INERTIAL = MODEL == BM_INERTIAL;
  constexpr bool RING = WS && HAS_G;  // without Gaussian noise there is nothing to produce
  constexpr float S = Units<POT>::SCALE;
  constexpr unsigned FULL = 0xffffffffu;
  extern __shared__ __align__(16) unsigned char ring_mem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int path_threads = RING ? (int)(blockDim.x >> 1) : (int)blockDim.x;
  const int path_warps = path_threads >> 5;
  const bool producer = RING && warp >= path_warps;
  const int pair = producer ? warp - path_warps : warp;
  PairRing *ring = RING ? reinterpret_cast<PairRing *>(ring_mem) + pair : nullptr;

  const int point = blockIdx.x / a.blocks_per_point;
  const int chunk = blockIdx.x - point * a.blocks_per_point;
  const long long p = (long long)chunk * path_threads + pair * 32 + lane;
  const bool valid = p < a.n_paths;  // lanes past a ragged end run along (the warp votes) and contribute nothing
  const unsigned long long g =
      (unsigned long long)point * (unsigned long long)a.n_paths + (unsigned long long)(valid ? p : 0);

  if (RING) {
    if (!producer && lane == 0) {
      for (int s = 0; s < RING_STAGES; ++s) { mbar_init(&ring->full[s], 1); mbar_init(&ring->empty[s], 1); }
      ring->done = 0;
    }
    __syncthreads();
  }

  const PhiloxKeys &K = a.keys;
  const bm_params bp = a.params[point];
  const double Dd = HAS_G ? bp.D : 0.0;
  const float cn = (float)(-2.0 * M_LN2 * (double)S * (double)S * 2.0 * Dd * a.dt);
  Partial mine = partial_zero();

  if (producer) {
    // ---- a3 + a4 for the partner warp: stage after stage until the consumer says stop -----------------------
    uint32_t b = 0, stage = 0, phase = 0;
    for (;;) {
      bool stop = false;
      while (!mbar_try_wait_hint(&ring->empty[stage], phase ^ 1u, 2000u)) {
        if (*reinterpret_cast<volatile int *>(&ring->done)) { stop = true; break; }
        __nanosleep(256);
      }
      if (stop || *reinterpret_cast<volatile int *>(&ring->done)) break;
#pragma unroll
      for (int i = 0; i < RING_BLOCKS; i += 2) {  // two independent Philox calls in flight
        const Gauss4 q0 = draw_gauss_f32(K, g, b + i, cn);
        const Gauss4 q1 = draw_gauss_f32(K, g, b + i + 1, cn);
        GaussSlot &s0 = ring->slot[stage][i], &s1 = ring->slot[stage][i + 1];
        s0.a[lane] = make_float4(q0.ra, q0.ca, q0.sa, q0.rb);
        s0.b[lane] = make_float2(q0.cb, q0.sb);
        s1.a[lane] = make_float4(q1.ra, q1.ca, q1.sa, q1.rb);
        s1.b[lane] = make_float2(q1.cb, q1.sb);
      }
      b += RING_BLOCKS;
      __syncwarp();
      if (lane == 0) mbar_arrive(&ring->full[stage]);
      if (++stage == RING_STAGES) { stage = 0; phase ^= 1u; }
    }
  } else {
    const float dt = (float)a.dt;
    const float inv_dt = (float)(1.0 / a.dt);
    const double lam = HAS_P ? bp.lambda : 0.0, zet = HAS_P ? bp.zeta : 0.0;
    PointF32 P;
    if (POT == BM_POT_SINE2) {
      // -V' = -2 pi A1 c - 4 pi A2 (2 c^2 - 1)
      P.kk1 = (float)((double)S * (-2.0 * M_PI * bp.A1));
      P.kk2 = (float)((double)S * (-8.0 * M_PI * bp.A2));
      P.base = (float)((double)S * (bp.F - lam * zet + 4.0 * M_PI * bp.A2));
    } else {
      P.kk1 = (float)bp.A1;
      P.kk2 = 0.f;
      P.base = (float)(bp.F - lam * zet);
    }
    P.Ga = (float)((double)S * (-bp.Fa));
    P.Gb = (float)((double)S * bp.Fb);
    P.cn = cn;
    P.inv_lam_dt = (lam > 0.0) ? (float)(1.0 / (lam * a.dt)) : 0.f;
    P.zeta = (float)((double)S * zet);
    P.inv_mua_dt = (HAS_D && bp.mu_a > 0.0) ? (float)(1.0 / (bp.mu_a * a.dt)) : 0.f;
    P.inv_mub_dt = (HAS_D && bp.mu_b > 0.0) ? (float)(1.0 / (bp.mu_b * a.dt)) : 0.f;
    P.gamma = (float)bp.gamma;
    P.amp = (float)((double)S * bp.amp);
    P.w_turns = (float)(bp.omega / (2.0 * M_PI));

    // R4: initial condition
    const uint4 wi = philox_call(K, g, STREAM_INIT, 0);
    float x;  // theta; between sub-steps within about one period of [-P/2, P/2) (folded where it is used as a base)
    int wraps = 0;
    {
      const double L0 = (POT == BM_POT_QUAD) ? 1.0 : Units<POT>::PERIOD_X;
      const double x0 = (bp.x0_fixed >= 0.0) ? bp.x0_fixed : L0 * ((double)wi.x * (1.0 / 4294967296.0));
      if (POT == BM_POT_QUAD) {
        x = (float)x0;
      } else {  // fold in fp64 once
        const double k = rint(x0 / L0);
        x = (float)((double)S * (x0 - k * L0));
        wraps = (int)k;
        fold_f32<POT>(x, wraps);
      }
    }
    float v = 0.f;  // theta units per unit time
    if (INERTIAL)
      v = (float)((double)S * (bp.v0_lo + (bp.v0_hi - bp.v0_lo) * (((double)wi.y + 0.5) * (1.0 / 4294967296.0))));
    int d = 0;
    if (HAS_D) d = ((((double)wi.z + 0.5) * (1.0 / 4294967296.0)) < bp.mu_a / (bp.mu_a + bp.mu_b)) ? 1 : 0;

    const int n_steps = (int)a.n_steps, n_discard = (int)a.n_discard;
    // jump clocks: (cell index, offset inside that cell); INT_MAX = never
    int nP = 0x7FFFFFFF, nD = 0x7FFFFFFF;
    float fP = 0.f, fD = 0.f, z = 0.f;
    uint32_t kP = 0, kD = 0;
    if (HAS_P && lam > 0.0) {
      const uint4 w = philox_call(K, g, STREAM_POISSON, 0);
      schedule_f32(0, 0.f, dt, inv_dt, neg_log_u_f32(w.x) * P.inv_lam_dt, nP, fP);
      z = P.zeta * neg_log_u_f32(w.y);
    }
    if (HAS_D) {
      const uint4 w = philox_call(K, g, STREAM_DICH, 0);
      schedule_f32(0, 0.f, dt, inv_dt, neg_log_u_f32(w.x) * (d ? P.inv_mub_dt : P.inv_mua_dt), nD, fD);
    }

    // drive phase in 2^-64 turns per cell (inertial): exact integer accumulation, no float time
    unsigned long long ph = 0, dph = 0;
    float drive0 = 0.f;  // SCALE * amp * cos(omega t) at the current time
    if (INERTIAL) {
      double turns_per_cell = bp.omega * a.dt / (2.0 * M_PI);
      turns_per_cell -= floor(turns_per_cell);
      dph = (unsigned long long)(turns_per_cell * 18446744073709551616.0);
      drive0 = P.amp;  // cos(0)
    }

    int n = valid ? 0 : n_steps;  // current cell; n == n_steps: finished
    // the cell whose completion needs attention: last discarded cell (snapshot after it), then the last cell
    int nB = (n_discard > 0) ? n_discard - 1 : n_steps - 1;
    int nNext = valid ? min(nB, min(nP, nD)) : n_steps;
    float tau = 0.f;
    int jumps = 0, extra = 0;  // extra = sub-steps that ended inside a cell
    float snap_x = x;
    int snap_w = wraps;
    float cst = P.base + (HAS_D ? (d ? P.Gb : P.Ga) : 0.f);
    const float hh_full = 0.5f * dt;

    // ---- FAST: a full grid step without events (h = dt: every step-scaled constant is loop invariant) ------
    auto fast_step = [&](float gr, float gc, bool do_fold) {
      float xf = x;
      if (do_fold) fold_f32<POT>(xf, wraps);
      if (!INERTIAL) {
        const float xs = HAS_G ? fmaf(gr, gc, xf) : xf;
        x = pc_overdamped_f32<POT, SINCOS>(x, xs, dt * cst, dt * P.kk1, dt * P.kk2, hh_full * cst, hh_full * P.kk1,
                                           hh_full * P.kk2);
      } else {
        ph += dph;
        const float drive1 = P.amp * cos_turns<SINCOS>(__uint_as_float((uint32_t)(ph >> 41) | 0x3F800000u));
        const float vs = HAS_G ? fmaf(gr, gc, v) : v;
        pc_inertial_f32<SINCOS>(x, v, xf, vs, dt, hh_full, P.gamma, P.kk1, P.kk2, cst + drive0, cst + drive1);
        drive0 = drive1;
      }
      n++;
    };

    // ---- GENERAL: a5 sub-step to the earliest of {grid point, kick, flip} in this cell, then a8, a10.  Written
    // with selects; the only branches are the (rare, divergent) kick and flip bodies.  A finished lane takes a
    // zero-length sub-step, which changes nothing.
    auto general_step = [&](float gr, float gc) {
      const bool live = n < n_steps;
      const bool inP = HAS_P && nP == n, inD = HAS_D && nD == n;
      float end = dt;
      if (inP) end = fminf(end, fP);
      if (inD) end = fminf(end, fD);
      if (!live) end = tau;
      const bool at_grid = live && (end == dt);
      const float h = end - tau, hh = 0.5f * h;
      float noise = 0.f;
      if (HAS_G) {
        const float rs = (h == dt) ? 1.0f : sqrt_approx(h * inv_dt);  // Var ~ h (A9)
        noise = gr * gc * rs;
      }
      fold_f32<POT>(x, wraps);
      if (!INERTIAL) {
        x = pc_overdamped_f32<POT, SINCOS>(x, x + noise, h * cst, h * P.kk1, h * P.kk2, hh * cst, hh * P.kk1, hh * P.kk2);
      } else {
        const unsigned long long ph1 = ph + dph;
        const float t1 = at_grid ? __uint_as_float((uint32_t)(ph1 >> 41) | 0x3F800000u)
                                 : fmaf(end, P.w_turns, __uint_as_float((uint32_t)(ph >> 41) | 0x3F800000u));
        const float drive1 = P.amp * cos_turns<SINCOS>(t1);
        const float xf = x;
        pc_inertial_f32<SINCOS>(x, v, xf, v + noise, h, hh, P.gamma, P.kk1, P.kk2, cst + drive0, cst + drive1);
        drive0 = drive1;
      }
      tau = end;
      if (HAS_P) {
        if (inP && live && end == fP) {  // a8: kick
          if (!INERTIAL) x += z; else v += z;
          jumps++;
          kP++;
          const uint4 w = philox_call(K, g, STREAM_POISSON, kP);
          schedule_f32(n, tau, dt, inv_dt, neg_log_u_f32(w.x) * P.inv_lam_dt, nP, fP);
          z = P.zeta * neg_log_u_f32(w.y);
        }
      }
      if (HAS_D) {
        if (inD && live && end == fD) {  // a8: flip
          d ^= 1;
          jumps++;
          kD++;
          cst = P.base + (d ? P.Gb : P.Ga);
          const uint4 w = philox_call(K, g, STREAM_DICH, kD);
          schedule_f32(n, tau, dt, inv_dt, neg_log_u_f32(w.x) * (d ? P.inv_mub_dt : P.inv_mua_dt), nD, fD);
        }
      }
      fold_f32<POT>(x, wraps);  // a kick may span several periods
      n += at_grid ? 1 : 0;
      tau = at_grid ? 0.f : tau;
      extra += (live && !at_grid) ? 1 : 0;
      if (INERTIAL) ph += at_grid ? dph : 0ull;
      if (at_grid && n == n_discard) {  // a10: t_i
        snap_x = x;
        snap_w = wraps;
      }
      nB = (n < n_discard) ? n_discard - 1 : n_steps - 1;
      // a lane inside a cell (tau > 0) stays on the GENERAL path until that cell is complete
      nNext = (n >= n_steps) ? n_steps : ((at_grid || !live) ? min(nB, min(nP, nD)) : n);
    };

    // Every lane of a warp takes one sub-step per slot, so the Gaussian index m = 4 blk + j is warp-uniform.
    // One vote per block of four slots, taken a block ahead: if no lane meets a jump, a boundary or its end within
    // four cells the warp runs four FAST steps as one basic block; otherwise each slot votes FAST or GENERAL.
    uint32_t blk = 0, stage = 0, phase = 0;
    Gauss4 qn{0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    if (HAS_G && !RING) qn = draw_gauss_f32(K, g, 0, P.cn);
    bool fastable = !__any_sync(FULL, nNext - n < 4);
    for (;;) {
      if (RING) {
        while (!mbar_try_wait(&ring->full[stage], phase)) {}
      }
#pragma unroll 1
      for (int bb = 0; bb < RING_BLOCKS; ++bb) {
        Gauss4 q = qn;
        if (RING) {
          const float4 qa = ring->slot[stage][bb].a[lane];
          const float2 qb = ring->slot[stage][bb].b[lane];
          q = Gauss4{qa.x, qa.y, qa.z, qa.w, qb.x, qb.y};
        }
        blk++;
        if (fastable) {
          fast_step(q.ra, q.ca, true);
          fastable = !__any_sync(FULL, nNext - n < 7);  // n is 3 short of the block's end here
          if (HAS_G && !RING) qn = draw_gauss_f32(K, g, blk, P.cn);
          fast_step(q.ra, q.sa, false);
          fast_step(q.rb, q.cb, false);
          fast_step(q.rb, q.sb, false);
        } else {
          if (HAS_G && !RING) qn = draw_gauss_f32(K, g, blk, P.cn);
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const float gr = (j < 2) ? q.ra : q.rb;
            const float gc = (j == 0) ? q.ca : (j == 1) ? q.sa : (j == 2) ? q.cb : q.sb;
            if (!__any_sync(FULL, n == nNext)) fast_step(gr, gc, true);
            else general_step(gr, gc);
          }
          fastable = !__any_sync(FULL, nNext - n < 4);
        }
      }
      if (RING) {
        __syncwarp();
        if (lane == 0) mbar_arrive(&ring->empty[stage]);
        if (++stage == RING_STAGES) { stage = 0; phase ^= 1u; }
      }
      if (!__any_sync(FULL, n < n_steps)) break;
    }
    if (RING) {
      __syncwarp();
      if (lane == 0) {
        *reinterpret_cast<volatile int *>(&ring->done) = 1;
        __threadfence_block();
      }
    }

    if (valid) {
      // a10: eq. (30), assembled once per path in fp64
      fold_f32<POT>(x, wraps);
      const double Ld = Units<POT>::PERIOD_X, iS = 1.0 / (double)S;
      const double span = (double)(a.n_steps - a.n_discard) * a.dt;
      const double xT = (double)wraps * Ld + (double)x * iS;
      const double xTi = (double)snap_w * Ld + (double)snap_x * iS;
      const double vbar = ((double)(wraps - snap_w) * Ld + ((double)x - (double)snap_x) * iS) / span;
      const double msub = (double)a.n_steps + (double)extra;
      if (a.out_paths) {
        double *o = a.out_paths + g * BM_OUT_STRIDE;
        o[BM_OUT_XT] = xT; o[BM_OUT_VT] = (double)v * iS; o[BM_OUT_VBAR] = vbar; o[BM_OUT_JUMPS] = (double)jumps;
        o[BM_OUT_SUBSTEPS] = msub; o[BM_OUT_XTI] = xTi;
      }
      mine = leaf(vbar, xT, (double)jumps, msub);
    }
  }
  block_reduce_store(mine, a.partials + (long long)blockIdx.x * PARTIAL_STRIDE);
}

}  // namespace bm
