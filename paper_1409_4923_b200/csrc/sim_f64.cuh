// sim_f64.cuh -- fp64 path kernel: one thread = one realization, state in registers for the whole run
// (Alg. 5 :367-374 without the per-launch load/store of steps 2 and 6).
// It follows DESIGN.md readings R3-R9 operation by operation, so that per-path results track the fp64
// oracle to ~1e-13 (only libm-vs-CUDA transcendental rounding and FMA contraction differ).
#pragma once
#include <type_traits>

#include "common.cuh"

namespace bm {

template <int POT>
__device__ __forceinline__ double period_f64() { return POT == BM_POT_SINE2 ? 1.0 : (POT == BM_POT_PWL ? 2.0 : 0.0); }

// u(w) = (w + 1/2) 2^-32  (R3)
__device__ __forceinline__ double u01_f64(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

// ---- elementary functions of the Gaussian stream, written for the arguments they get here ------------------------
// Branch-free (so that the time loop can interleave them with the predictor-corrector chain, see the kernel) and with
// their coefficients in constant memory (a DFMA takes c[bank][offset] as an operand; the library routines load each
// 64-bit coefficient with two UMOV).  Coefficients: csrc/make_poly_f64.py.  Each is within ~1 ulp of the correctly rounded
// value on its range; tests/test_gpu_parity.py compares the resulting normals with the oracle's (libm) to 5e-15.
__constant__ double SINPI_C[8] = {3.141592653589793, -5.16771278004997, 2.5501640398773415, -0.5992645293202978,
                                  0.08214588658005621, -0.007370429884712669, 0.00046628272951211076, -2.1717401400090533e-05};
__constant__ double COSPI_C[8] = {1.0, -4.934802200544679, 4.058712126416747, -1.3352627688519174, 0.23533063019088787,
                                  -0.025806885652951306, 0.0019294657440800042, -0.00010356747255199479};
__constant__ double LOGP_C[7] = {0.666666666666667, 0.39999999999899444, 0.2857142862600327, 0.22222211130259878,
                                 0.18182889455674947, 0.15331710618210773, 0.14616585424888623};

// u(w) of R3 without an integer conversion: 2^52 + w has w in its low mantissa bits
__device__ __forceinline__ double u01_bits_f64(uint32_t w) {
  const double t = __hiloint2double(0x43300000, (int)w) - 4503599627370496.0;  // = w, exactly
  return fma(t, 1.0 / 4294967296.0, 1.0 / 8589934592.0);                        // (w + 1/2) 2^-32, exactly
}

// ln u for a normal u in (0, 1): u = 2^k m, m in [sqrt(1/2), sqrt(2)); with f = m - 1, s = f / (2 + f), z = s^2:
// ln m = 2 atanh s = f - s (f - z P(z)).  The quotient by a reciprocal seed, one Newton step, then one correction.
__device__ __forceinline__ double log_u_f64(double u) {
  int hi = __double2hiint(u);
  hi += 0x3ff00000 - 0x3fe6a09e;  // mantissas above sqrt(2) carry into the exponent
  const int k = (hi >> 20) - 0x3ff;
  const double m = __hiloint2double((hi & 0x000fffff) + 0x3fe6a09e, __double2loint(u));
  const double f = m - 1.0, y = 2.0 + f;
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(y));
  const double e = fma(-y, r, 1.0);
  r = fma(r, e, r);  // one Newton step on the seed: a relative error of ~2^-40; the correction below squares it again
  double sq = f * r;
  sq = fma(fma(-y, sq, f), r, sq);  // s = f / y
  const double z = sq * sq;
  double p = LOGP_C[6];
  p = fma(p, z, LOGP_C[5]);
  p = fma(p, z, LOGP_C[4]);
  p = fma(p, z, LOGP_C[3]);
  p = fma(p, z, LOGP_C[2]);
  p = fma(p, z, LOGP_C[1]);
  p = fma(p, z, LOGP_C[0]);
  const double lm = fma(-sq, fma(-z, p, f), f);  // f - s (f - z P)
  const double dk = (double)k;
  return fma(dk, 0.6931471803691238, fma(dk, 1.9082149292705877e-10, lm));  // k ln2 in two parts: the first product is exact
}

// sqrt x for a normal x > 0: reciprocal-root seed, one coupled Newton step on (g, h) -> (sqrt x, 1 / (2 sqrt x)), one correction
__device__ __forceinline__ double sqrt_pos_f64(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  const double r = fma(-g, h, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);  // one coupled step on the seed: ~2^-40; the correction below squares it again
  return fma(fma(-g, g, x), h, g);
}

// (sin pi a, cos pi a) for 0 <= a <= 2: q = nearest integer to 2a, r = a - q/2 in [-1/4, 1/4] (exact), polynomials in
// r^2 (two independent Horner chains), then the quadrant: swap for odd q, signs from q and q + 1.
__device__ __forceinline__ void sincospi_f64(double a, double &sn, double &cs) {
  const double MAGIC = 6755399441055744.0;  // 1.5 * 2^52
  const double t = fma(a, 2.0, MAGIC);
  const int q = __double2loint(t);
  const double r = fma(t - MAGIC, -0.5, a);
  const double z = r * r;
  double ps = SINPI_C[7], pc = COSPI_C[7];
  ps = fma(ps, z, SINPI_C[6]); pc = fma(pc, z, COSPI_C[6]);
  ps = fma(ps, z, SINPI_C[5]); pc = fma(pc, z, COSPI_C[5]);
  ps = fma(ps, z, SINPI_C[4]); pc = fma(pc, z, COSPI_C[4]);
  ps = fma(ps, z, SINPI_C[3]); pc = fma(pc, z, COSPI_C[3]);
  ps = fma(ps, z, SINPI_C[2]); pc = fma(pc, z, COSPI_C[2]);
  ps = fma(ps, z, SINPI_C[1]); pc = fma(pc, z, COSPI_C[1]);
  ps = fma(ps, z, SINPI_C[0]); pc = fma(pc, z, COSPI_C[0]);
  ps *= r;
  const bool odd = q & 1;
  const double s0 = odd ? pc : ps, c0 = odd ? ps : pc;
  // sin: q = 0, 1 -> +, 2, 3 -> -;   cos: q = 0 -> +, 1, 2 -> -, 3 -> + (q = 4 as q = 0)
  sn = __hiloint2double(__double2hiint(s0) ^ ((q & 2) << 30), __double2loint(s0));
  cs = __hiloint2double(__double2hiint(c0) ^ (((q + 1) & 2) << 30), __double2loint(c0));
}

// cos x for the drive of the inertial model, |x| < 2^20 (omega t: 1.3e4 at the end of C3): k = nearest integer to
// x 2/pi, r = x - k pi/2 with pi/2 in three pieces (the first two products are exact), sin r and cos r as polynomials in
// r^2 on |r| <= pi/4 (both evaluated: two independent chains), then the quadrant.  Branch-free, constants from constant
// memory; the library's cos spends ~30 UMOV per call on its coefficients and keeps a branch for huge arguments.
__constant__ double SIN_C[8] = {1.0, -0.16666666666666666, 0.008333333333333321, -0.0001984126984125347, 2.755731921355806e-06,
                                -2.5052104778015328e-08, 1.6058352290975984e-10, -7.57808328312409e-13};
__constant__ double COS_C[8] = {1.0, -0.5, 0.04166666666666645, -0.0013888888888861082, 2.4801587283874084e-05,
                                -2.755731309595641e-07, 2.0875582146477433e-09, -1.1353367957830792e-11};
__device__ __forceinline__ double cos_drive_f64(double x) {
  const double MAGIC = 6755399441055744.0;  // 1.5 * 2^52
  const double t = fma(x, 0.6366197723675814, MAGIC);
  const int q = __double2loint(t);
  const double k = t - MAGIC;
  double r = fma(-k, 1.5707963267341256, x);
  r = fma(-k, 6.077100506303966e-11, r);
  r = fma(-k, 2.0222662487959506e-21, r);
  const double z = r * r;
  double ps = SIN_C[7], pc = COS_C[7];
  ps = fma(ps, z, SIN_C[6]); pc = fma(pc, z, COS_C[6]);
  ps = fma(ps, z, SIN_C[5]); pc = fma(pc, z, COS_C[5]);
  ps = fma(ps, z, SIN_C[4]); pc = fma(pc, z, COS_C[4]);
  ps = fma(ps, z, SIN_C[3]); pc = fma(pc, z, COS_C[3]);
  ps = fma(ps, z, SIN_C[2]); pc = fma(pc, z, COS_C[2]);
  ps = fma(ps, z, SIN_C[1]); pc = fma(pc, z, COS_C[1]);
  ps = fma(ps, z, SIN_C[0]); pc = fma(pc, z, COS_C[0]);
  ps *= r;
  // cos(r + q pi/2): q = 0 -> cos r, 1 -> -sin r, 2 -> -cos r, 3 -> sin r
  const double v = (q & 1) ? ps : pc;
  return __hiloint2double(__double2hiint(v) ^ (((q + 1) & 2) << 30), __double2loint(v));
}

// Box-Muller pair from two words (R3): r = sqrt(-2 ln u(wa)); (r cos 2 pi u(wb), r sin 2 pi u(wb))
__device__ __forceinline__ double bm_radius_f64(uint32_t wa) { return sqrt_pos_f64(-2.0 * log_u_f64(u01_bits_f64(wa))); }
__device__ __forceinline__ void bm_angle_f64(uint32_t wb, double r, double &g0, double &g1) {
  double sn, cs;
  sincospi_f64(2.0 * u01_bits_f64(wb), sn, cs);
  g0 = r * cs;
  g1 = r * sn;
}
__device__ __forceinline__ void box_muller_f64(uint32_t wa, uint32_t wb, double &g0, double &g1) {
  bm_angle_f64(wb, bm_radius_f64(wa), g0, g1);
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

// cos(2 pi x) for the force evaluations, branch-free (so that the chains of a thread's paths interleave) and without the
// generality of cospi: 2x is rounded to the nearest integer k with a magic addition (|x| < 2^50), r = x - k/2 lies in
// [-1/4, 1/4], cos 2 pi x = (-1)^k cos 2 pi r, and cos 2 pi r is a degree-12 polynomial in r^2 (interpolant at the
// Chebyshev nodes of [0, 1/16]; approximation error 9.5e-17, evaluated in two interleaved Horner chains; absolute
// error of the result below 3e-16, where the oracle's cos(2 pi xi) itself carries 7e-16 from rounding 2 pi xi).
__constant__ double COS2PI_E[7] = {2.253668089082175e-05, 0.0037798236737849045, 0.28200596842351006, 7.903536371318447,
                                    60.24464137187666, 64.9393940226683, 1.0};
__constant__ double COS2PI_O[6] = {-0.00032289025049633054, -0.03638284043309509, -1.7143907110876637, -26.4262567833744,
                                    -85.45681720669373, -19.739208802178716};
__device__ __forceinline__ double cos2pi_f64(double x) {
  const double MAGIC = 6755399441055744.0;  // 1.5 * 2^52: (y + MAGIC) has ulp 1
  const double t = fma(x, 2.0, MAGIC);
  const double k = t - MAGIC;
  const double r = fma(k, -0.5, x);
  const double u = r * r, w = u * u;
  // the coefficients come from constant memory: a DFMA takes c[bank][offset] as an operand, where an immediate costs
  // two UMOV issue slots per coefficient and evaluation
  double e = COS2PI_E[0], o = COS2PI_O[0];
  e = fma(e, w, COS2PI_E[1]);   o = fma(o, w, COS2PI_O[1]);
  e = fma(e, w, COS2PI_E[2]);   o = fma(o, w, COS2PI_O[2]);
  e = fma(e, w, COS2PI_E[3]);   o = fma(o, w, COS2PI_O[3]);
  e = fma(e, w, COS2PI_E[4]);   o = fma(o, w, COS2PI_O[4]);
  e = fma(e, w, COS2PI_E[5]);   o = fma(o, w, COS2PI_O[5]);
  e = fma(e, w, COS2PI_E[6]);
  const double c = fma(o, u, e);
  // (-1)^k: the parity of k is the lowest mantissa bit of t
  const int hi = __double2hiint(c) ^ (__double2loint(t) << 31);
  return __hiloint2double(hi, __double2loint(c));
}

// -V'(x) on the (nearly) folded coordinate
template <int POT>
__device__ __forceinline__ double minus_dV_f64(const PointF64 &P, double x) {
  if (POT == BM_POT_SINE2) {
    const double c = cos2pi_f64(x);
    const double c2 = fma(2.0 * c, c, -1.0);  // cos 4 pi x = 2 cos^2 2 pi x - 1: one cosine per force evaluation
    return -(2.0 * M_PI * P.A1 * c + 4.0 * M_PI * P.A2 * c2);
  } else if (POT == BM_POT_PWL) {
    const double y = x - 2.0 * floor(x * 0.5);
    return (y < 1.0) ? P.A1 : -P.A1;
  } else {
    return -P.A1 * x;
  }
}

// a(x) = -V'(x) + cst for the path kernels.  SINE2: -V' = -2 pi A1 c - 4 pi A2 (2 c^2 - 1), c = cos 2 pi x, summed in
// Horner form, c (k1 + k2 c) + (cst + 4 pi A2): two DFMA behind the cosine instead of five FP64 operations (the sum is
// the oracle's up to the order of its roundings; per-path parity is 1e-8).  k = (k1, k2, 4 pi A2).
template <int POT>
__device__ __forceinline__ double drift_f64(const PointF64 &P, const double (&k)[3], double x, double cst) {
  if (POT == BM_POT_SINE2) {
    const double c = cos2pi_f64(x);
    return fma(c, fma(k[1], c, k[0]), cst + k[2]);
  }
  return minus_dV_f64<POT>(P, x) + cst;
}

// noise amplitude of a sub-step cut short by an event (kept out of line: inlined, the compiler evaluates the square
// root in every iteration and selects afterwards -- ten FP64 operations per sub-step for the one in 500 that needs them)
static __device__ __noinline__ double amp_of_substep_f64(double D, double h) { return sqrt(2.0 * D * h); }

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
// the same kernel changes the register allocation of the time loop (6 % slower on C1).
// NPATH realizations per thread (path q of thread t in block-chunk c of a point is p = (c * NPATH + q) * blockDim + t):
// one fp64 sub-step is a dependent chain of ~700 cycles (three software cosines behind each other), so a small
// ensemble (C1, C2: 3.5 warps per scheduler) leaves the FP64 pipe idle most of the time; two independent chains per
// thread fill it.  A path's arithmetic does not depend on NPATH (same operations in the same order per path).
template <int MODEL, int POT, int NOISE, bool CHUNKED, int NPATH>
__global__ void __launch_bounds__(256, 2) bm_paths_f64(const __grid_constant__ SimArgs a) {  // two blocks of 256 per SM: <= 128 registers (C2: 256 blocks on 148 SMs)
  constexpr bool HAS_G = NOISE & BM_NOISE_GAUSS, HAS_P = NOISE & BM_NOISE_POISSON, HAS_D = NOISE & BM_NOISE_DICH;
  constexpr bool INERTIAL = MODEL == BM_INERTIAL;
  constexpr int N = NPATH;
  const int point = blockIdx.x / a.blocks_per_point;
  const int chunk = blockIdx.x - point * a.blocks_per_point;

  const bm_params bp = a.params[point];
  PointF64 P;
  P.A1 = bp.A1; P.A2 = bp.A2; P.D = HAS_G ? bp.D : 0.0;
  P.lambda = HAS_P ? bp.lambda : 0.0; P.zeta = HAS_P ? bp.zeta : 0.0;
  P.Fa = bp.Fa; P.Fb = bp.Fb; P.mu_a = bp.mu_a;
  P.mu_b = bp.mu_b > 0.0 ? bp.mu_b : 0.0;  // mu_b <= 0: +Fb is absorbing (bm.h: bm_params) -- an infinite sojourn, never a negative one
  P.gamma = bp.gamma; P.amp = bp.amp; P.omega = bp.omega;
  P.c0 = bp.F - P.lambda * P.zeta;  // constant part of the drift a(x), all three stages (R6)
  const double dt = step_length(a, point);
  const double L0 = (POT == BM_POT_QUAD) ? 1.0 : period_f64<POT>();
  // a non-positive rate switches its source off at this point (lambda; mu_a: Gamma = 0, as the oracle)
  const bool onP = HAS_P && P.lambda > 0.0;
  const bool onD = HAS_D && P.mu_a > 0.0;
  const long long n_end = CHUNKED ? a.step_end : a.n_steps;
  const double amp_dt = sqrt(2.0 * P.D * dt);  // noise amplitude of an unsplit grid step (the same expression as below)
  const double kf[3] = {-2.0 * M_PI * P.A1, -8.0 * M_PI * P.A2, 4.0 * M_PI * P.A2};  // drift_f64

  bool valid[N], tracing[N];
  unsigned long long g[N], m[N];
  StateF64 s[N], snap[N];
  int d[N];
  uint32_t kP[N], kD[N];
  // normals in flight: one Philox block of four (a single launch), two blocks (CHUNKED, see the time loop)
  constexpr int GQ = CHUNKED ? 8 : 4;
  double rP[N], rD[N], z[N], rem[N], gq[N][GQ];
  unsigned long long blk0[N];  // CHUNKED: Gaussian block the path was in when the launch started
  double *trace[N];
  long long n[N];
#pragma unroll
  for (int q = 0; q < N; ++q) {
    const long long p = ((long long)chunk * N + q) * blockDim.x + threadIdx.x;
    valid[q] = p < a.n_paths;
    g[q] = (unsigned long long)point * (unsigned long long)a.n_paths + (unsigned long long)(valid[q] ? p : 0);
    // R4: initial condition from init-stream call 0
    const uint4 wi = philox_call(a.keys, g[q], STREAM_INIT, 0);
    s[q].xi = (bp.x0_fixed >= 0.0) ? bp.x0_fixed : L0 * ((double)wi.x * (1.0 / 4294967296.0));
    s[q].wraps = 0;
    s[q].v = INERTIAL ? bp.v0_lo + (bp.v0_hi - bp.v0_lo) * u01_f64(wi.y) : 0.0;
    fold_f64<POT>(s[q]);
    d[q] = onD ? ((u01_f64(wi.z) < P.mu_a / (P.mu_a + P.mu_b)) ? 1 : 0) : -1;
    kP[q] = 0; kD[q] = 0; rP[q] = 0.0; rD[q] = 0.0; z[q] = 0.0;
    if (onP) {
      const uint4 w = philox_call(a.keys, g[q], STREAM_POISSON, 0);
      rP[q] = -log(u01_f64(w.x)) / P.lambda;
      z[q] = -P.zeta * log(u01_f64(w.y));
    }
    if (onD) {
      const uint4 w = philox_call(a.keys, g[q], STREAM_DICH, 0);
      rD[q] = -log(u01_f64(w.x)) / (d[q] ? P.mu_b : P.mu_a);
    }
    tracing[q] = valid[q] && a.out_trace != nullptr && (long long)g[q] < a.trace_paths;
    trace[q] = tracing[q] ? a.out_trace + (long long)g[q] * a.trace_steps * 2 : nullptr;
    n[q] = CHUNKED ? a.step_begin : 0;
    m[q] = 0;
    rem[q] = dt;
#pragma unroll
    for (int j = 0; j < GQ; ++j) gq[q][j] = 0.0;
    snap[q] = s[q];
    if (CHUNKED && a.state != nullptr && a.step_begin > 0 && valid[q]) {  // row f2: continue a run from its checkpoint
      CkptF64 c;
      ckpt_load_f64(a, g[q], c);
      s[q].xi = c.xi; s[q].wraps = c.wraps; s[q].v = c.v; rP[q] = c.rP; rD[q] = c.rD; z[q] = c.z; kP[q] = c.kP; kD[q] = c.kD;
      d[q] = c.d; m[q] = c.m; snap[q].xi = c.sxi; snap[q].wraps = c.swraps; snap[q].v = c.sv;
    }
    blk0[q] = m[q] >> 2;
    if (CHUNKED && HAS_G) {  // the block the path is in (the next one is drawn in iteration 0 of the loop)
      double t[4];
      regen_gauss_block_f64(a.keys, g[q], (uint32_t)blk0[q], t);
      const int o = (int)(blk0[q] & 1ull) * 4;
#pragma unroll
      for (int j = 0; j < 8; ++j)
        if ((j & 4) == o) gq[q][j % GQ] = t[j & 3];
    }
    if (!valid[q]) n[q] = n_end;  // a path past the ragged end does nothing
  }

  // CHUNKED: a launch that resumes a run finds its paths at the same grid step but, after kicks or flips, at different
  // sub-step counts m, i.e. at different places inside their Philox blocks of four normals; drawing a block whenever
  // a lane runs out would then happen in every iteration for a quarter of the lanes.  Every iteration is one sub-step
  // of every active lane, so instead each lane keeps TWO blocks and the whole warp draws the next one every fourth
  // iteration: by then the older block is used up whatever the lane's phase.  (A single launch starts all lanes at
  // m = 0; they stay in phase and one block is enough.)
  // One iteration = one sub-step of every active path.  J >= 0 (a single launch): the sub-step takes normal J of the
  // Philox block in flight -- the lanes of a warp stay in phase, so the time loop is unrolled by four and the index
  // of the normal is static; J = 0 draws the block.  J < 0: the index follows the path's own m.
  uint4 gw = make_uint4(0u, 0u, 0u, 0u);  // unrolled form: words, an intermediate and the normals of the block in production
  double glog = 0.0, gnx[4] = {0.0, 0.0, 0.0, 0.0};
  auto iteration = [&](auto JT, unsigned long long it) -> bool {
    constexpr int J = decltype(JT)::value;
    bool act[N], any = false;
#pragma unroll
    for (int q = 0; q < N; ++q) { act[q] = n[q] < n_end; any |= act[q]; }
    if (!any) return false;
    // a5: sub-step length; a3/a4: the sub-step's Gaussian
    double h[N], gn[N], cst[N], dxi[N];
#pragma unroll
    for (int q = 0; q < N; ++q) {
      h[q] = rem[q];
      if (onP && rP[q] < h[q]) h[q] = rP[q];
      if (onD && rD[q] < h[q]) h[q] = rD[q];
      gn[q] = 0.0;
      if (HAS_G && act[q]) {
        if (!CHUNKED) {
          if (J < 0 && (m[q] & 3ull) == 0) {
            const uint4 w = philox_call(a.keys, g[q], STREAM_GAUSS, (uint32_t)(m[q] >> 2));
            box_muller_f64(w.x, w.y, gq[q][0], gq[q][1]);
            box_muller_f64(w.z, w.w, gq[q][2], gq[q][3]);
          }
          const int j = J >= 0 ? J : (int)(m[q] & 3ull);
          gn[q] = (j == 0) ? gq[q][0] : (j == 1) ? gq[q][1] : (j == 2) ? gq[q][2] : gq[q][3];
        } else {
          if ((it & 3ull) == 0) {  // warp-uniform: the block after the one this iteration's normal comes from
            const unsigned long long b = blk0[q] + (it >> 2) + 1ull;
            const uint4 w = philox_call(a.keys, g[q], STREAM_GAUSS, (uint32_t)b);
            double t0, t1, t2, t3;
            box_muller_f64(w.x, w.y, t0, t1);
            box_muller_f64(w.z, w.w, t2, t3);
            const bool hi = (b & 1ull) != 0;
            gq[q][0 % GQ] = hi ? gq[q][0 % GQ] : t0; gq[q][1 % GQ] = hi ? gq[q][1 % GQ] : t1;
            gq[q][2 % GQ] = hi ? gq[q][2 % GQ] : t2; gq[q][3 % GQ] = hi ? gq[q][3 % GQ] : t3;
            gq[q][4 % GQ] = hi ? t0 : gq[q][4 % GQ]; gq[q][5 % GQ] = hi ? t1 : gq[q][5 % GQ];
            gq[q][6 % GQ] = hi ? t2 : gq[q][6 % GQ]; gq[q][7 % GQ] = hi ? t3 : gq[q][7 % GQ];
          }
          const int j = (int)(m[q] & 7ull);
          const double lo = (j & 2) ? ((j & 1) ? gq[q][3 % GQ] : gq[q][2 % GQ]) : ((j & 1) ? gq[q][1 % GQ] : gq[q][0 % GQ]);
          const double hi = (j & 2) ? ((j & 1) ? gq[q][7 % GQ] : gq[q][6 % GQ]) : ((j & 1) ? gq[q][5 % GQ] : gq[q][4 % GQ]);
          gn[q] = (j & 4) ? hi : lo;
        }
      }
      const double Gd = onD ? (d[q] ? P.Fb : -P.Fa) : 0.0;
      cst[q] = P.c0 + Gd;
      double amp = amp_dt;
      if (HAS_G && h[q] != dt) amp = amp_of_substep_f64(P.D, h[q]);
      dxi[q] = HAS_G ? __dmul_rn(amp, gn[q]) : 0.0;  // (never contracted into the sums that use it: a path must not depend on which copy of the code runs it)
    }
    // Unrolled form: a quarter of the NEXT block of normals is produced beside each sub-step -- branch-free code in the
    // same basic block as the predictor-corrector chain, whose stalls (three cosines behind each other) it fills.
    // J = 0: the Philox call and ln u_a; 1: radius and angle of pair a; 2: ln u_b and radius b; 3: angle of pair b.
    if (J >= 0 && HAS_G) {
      if (J == 0) {
        gw = philox_call(a.keys, g[0], STREAM_GAUSS, (uint32_t)(m[0] >> 2) + 1u);
        glog = log_u_f64(u01_bits_f64(gw.x));
      } else if (J == 1) {
        bm_angle_f64(gw.y, sqrt_pos_f64(-2.0 * glog), gnx[0], gnx[1]);
      } else if (J == 2) {
        glog = sqrt_pos_f64(-2.0 * log_u_f64(u01_bits_f64(gw.z)));
      } else {
        bm_angle_f64(gw.w, glog, gnx[2], gnx[3]);
      }
    }
    // a6 / a7: the predictor-corrector sub-step, stage by stage over the thread's paths (independent chains)
    double xn[N], vn[N];
    if (!INERTIAL) {
      // Alg. 1
      double F1[N], xb[N], F2[N];
#pragma unroll
      for (int q = 0; q < N; ++q) F1[q] = drift_f64<POT>(P, kf, s[q].xi, cst[q]);
#pragma unroll
      for (int q = 0; q < N; ++q) xb[q] = s[q].xi + F1[q] * h[q] + dxi[q];
#pragma unroll
      for (int q = 0; q < N; ++q) F2[q] = drift_f64<POT>(P, kf, xb[q], cst[q]);
#pragma unroll
      for (int q = 0; q < N; ++q) xb[q] = s[q].xi + 0.5 * (F1[q] + F2[q]) * h[q] + dxi[q];
#pragma unroll
      for (int q = 0; q < N; ++q) F2[q] = drift_f64<POT>(P, kf, xb[q], cst[q]);
#pragma unroll
      for (int q = 0; q < N; ++q) { xn[q] = s[q].xi + 0.5 * (F1[q] + F2[q]) * h[q] + dxi[q]; vn[q] = s[q].v; }
      // (an empty asm that takes the stage's results together with xn: the compiler would otherwise sink the stage
      // below the branches of the event handling, out of the block it is meant to share with the chain)
      if (J >= 0 && HAS_G) {
        if (J == 0 || J == 2) asm volatile("" : "+d"(xn[0]), "+d"(glog));
        if (J == 1) asm volatile("" : "+d"(xn[0]), "+d"(gnx[0]), "+d"(gnx[1]));
        if (J == 3) asm volatile("" : "+d"(xn[0]), "+d"(gnx[2]), "+d"(gnx[3]));
      }
    } else {
      // R7: two-component version, additive noise in v only, drive evaluated at t and t+h
      double A1v[N], xb[N], vb[N], drive[N], A2x[N], A2v[N];
#pragma unroll
      for (int q = 0; q < N; ++q) {
        const double t = __dadd_rn(__dmul_rn((double)n[q], dt), __dsub_rn(dt, rem[q]));
        A1v[q] = -P.gamma * s[q].v + drift_f64<POT>(P, kf, s[q].xi, cst[q]) + P.amp * cos_drive_f64(P.omega * t);
        drive[q] = P.amp * cos_drive_f64(P.omega * __dadd_rn(t, h[q]));
      }
#pragma unroll
      for (int q = 0; q < N; ++q) { xb[q] = s[q].xi + s[q].v * h[q]; vb[q] = s[q].v + A1v[q] * h[q] + dxi[q]; }
#pragma unroll
      for (int q = 0; q < N; ++q) { A2x[q] = vb[q]; A2v[q] = -P.gamma * vb[q] + drift_f64<POT>(P, kf, xb[q], cst[q]) + drive[q]; }
#pragma unroll
      for (int q = 0; q < N; ++q) {
        xb[q] = s[q].xi + 0.5 * (s[q].v + A2x[q]) * h[q];
        vb[q] = s[q].v + 0.5 * (A1v[q] + A2v[q]) * h[q] + dxi[q];
      }
#pragma unroll
      for (int q = 0; q < N; ++q) { A2x[q] = vb[q]; A2v[q] = -P.gamma * vb[q] + drift_f64<POT>(P, kf, xb[q], cst[q]) + drive[q]; }
#pragma unroll
      for (int q = 0; q < N; ++q) {
        xn[q] = s[q].xi + 0.5 * (s[q].v + A2x[q]) * h[q];
        vn[q] = s[q].v + 0.5 * (A1v[q] + A2v[q]) * h[q] + dxi[q];
      }
    }
    // a8, a9 and the bookkeeping of the grid step, path by path
#pragma unroll
    for (int q = 0; q < N; ++q) {
      if (!act[q]) continue;
      s[q].xi = xn[q];
      s[q].v = vn[q];
      m[q]++;
      rem[q] -= h[q];
      if (onP) {
        rP[q] -= h[q];
        if (rP[q] <= 0.0) {  // kick kP (a8)
          if (!INERTIAL) s[q].xi += z[q]; else s[q].v += z[q];
          kP[q]++;
          const uint4 w = philox_call(a.keys, g[q], STREAM_POISSON, kP[q]);
          rP[q] = -log(u01_f64(w.x)) / P.lambda;
          z[q] = -P.zeta * log(u01_f64(w.y));
        }
      }
      if (onD) {
        rD[q] -= h[q];
        if (rD[q] <= 0.0) {  // flip
          d[q] = 1 - d[q];
          kD[q]++;
          const uint4 w = philox_call(a.keys, g[q], STREAM_DICH, kD[q]);
          rD[q] = -log(u01_f64(w.x)) / (d[q] ? P.mu_b : P.mu_a);
        }
      }
      fold_f64<POT>(s[q]);
      if (rem[q] <= 0.0) {
        n[q]++;
        rem[q] = dt;
        if (tracing[q] && n[q] <= a.trace_steps) {
          trace[q][2 * (n[q] - 1)] = unfolded_f64<POT>(s[q]);
          trace[q][2 * (n[q] - 1) + 1] = s[q].v;
        }
        if (n[q] == a.n_discard) snap[q] = s[q];
      }
    }
    if (J == 3 && HAS_G) {
#pragma unroll
      for (int j = 0; j < 4; ++j) gq[0][j] = gnx[j];
    }
    return true;
  };
  // unrolled: the over-damped kernel with one path per thread (measured: C1 89.5 -> 84.7 ms unrolled, -> 76.4 with the
  // next block of normals produced beside the sub-steps; the inertial kernel, with 117 registers and a longer body, loses
  // to the larger code: C2 266 -> 280 ms unrolled, 249.5 -> 253.8 ms unrolled and staged, 128 registers and spills)
  if (CHUNKED || N > 1 || INERTIAL) {
    for (unsigned long long it = 0; iteration(std::integral_constant<int, -1>(), it); ++it) {}
  } else {
    if (HAS_G) {  // block 0 in place; from then on block b + 1 is produced while block b is used
      const uint4 w = philox_call(a.keys, g[0], STREAM_GAUSS, 0u);
      box_muller_f64(w.x, w.y, gq[0][0], gq[0][1]);
      box_muller_f64(w.z, w.w, gq[0][2], gq[0][3]);
    }
    while (iteration(std::integral_constant<int, 0>(), 0ull)) {
      iteration(std::integral_constant<int, 1>(), 0ull);
      iteration(std::integral_constant<int, 2>(), 0ull);
      iteration(std::integral_constant<int, 3>(), 0ull);
    }
  }

  Partial mine = partial_zero();
#pragma unroll
  for (int q = 0; q < N; ++q) {
    if (!valid[q]) continue;
    if (CHUNKED && a.state != nullptr) {  // row f2: checkpoint (chunks end on completed grid steps, so rem = dt)
      CkptF64 c;
      c.xi = s[q].xi; c.wraps = s[q].wraps; c.v = s[q].v; c.rP = rP[q]; c.rD = rD[q]; c.z = z[q]; c.kP = kP[q]; c.kD = kD[q];
      c.d = d[q]; c.m = m[q]; c.jumps = (double)(kP[q] + kD[q]); c.sxi = snap[q].xi; c.swraps = snap[q].wraps; c.sv = snap[q].v;
      ckpt_store_f64(a, g[q], c);
    }
    // a10: eq. (30)
    const double span = (double)(a.n_steps - a.n_discard) * dt;
    const double xT = unfolded_f64<POT>(s[q]);
    const double vbar = ((double)(s[q].wraps - snap[q].wraps) * period_f64<POT>() + (s[q].xi - snap[q].xi)) / span;
    if (a.out_paths && (!CHUNKED || a.step_end >= a.n_steps)) {
      double *o = a.out_paths + g[q] * BM_OUT_STRIDE;
      o[BM_OUT_XT] = xT; o[BM_OUT_VT] = s[q].v; o[BM_OUT_VBAR] = vbar; o[BM_OUT_JUMPS] = (double)(kP[q] + kD[q]);
      o[BM_OUT_SUBSTEPS] = (double)m[q]; o[BM_OUT_XTI] = unfolded_f64<POT>(snap[q]);
    }
    mine = merge(mine, leaf(vbar, xT, (double)(kP[q] + kD[q]), (double)m[q]));  // events applied = the two stream indices
  }
  if (CHUNKED && a.step_end < a.n_steps) return;  // not the last chunk: the partials are not used (uniform over the grid)
  block_reduce_store(mine, a.partials + (long long)blockIdx.x * PARTIAL_STRIDE);
}

}  // namespace bm
