// sim_f32.cuh -- fp32 path kernel (the throughput kernel), v7.  One thread = one realization; position, next events,
// Gaussian cache and observable snapshot stay in registers for the whole run.
//
// Same method as the fp64 kernel (R1-R9), arranged for fp32 accuracy and for the SM's pipes
// (profiles/r2_f32_v7.md holds the measurements this layout answers):
//  * the position is carried as theta = 2 pi x / L (radians of the potential's phase), folded to [-pi, pi) with an
//    int32 wrap counter by a round-to-nearest "magic add" (no F2I/FRND, which share the 16-lane XU
//    pipe with MUFU).  In these units a force cosine is FMUL.RZ + MUFU.COS with no scaling multiply in front;
//  * Alg. 1 is evaluated with the step length folded into the constants:
//    x1 = (xs + h K0) + c (h K1 + h K2 c), so every stage is 2 FFMA behind its cosine;
//  * ALL lanes of a warp are always in the SAME grid cell n (the cell counter is warp-uniform).  A cell without a
//    kick or flip in any lane is one FAST step with loop-invariant constants; NB such cells (one Philox call of
//    normals) form one basic block when no lane has an event within them (one vote per block).  Otherwise the warp
//    forms a uniform control word (REDUX.OR of the lanes' event bits) and runs the block pair slot by pair slot: a
//    slot without an event is the clean path's two-cell code, a cell with an event in some lane is a SLOW cell;
//  * the Box-Muller pair of cells (2i+2, 2i+3) is formed while cells (2i, 2i+1) run, and the ten Philox rounds of
//    the next Gaussian call are spread over the pair slots, so the integer and MUFU work of the Gaussians sits in
//    the stalls of the serial cosine chain of Alg. 1 instead of in a phase of its own;
//  * kick and flip times do not depend on the motion, so they are drawn AHEAD of time into per-path rings in shared
//    memory, refilled by the whole warp at once (v6: a slow cell no longer holds a Philox call that one or two lanes
//    execute while thirty wait; see "event queues" below);
//  * a lane with events inside the current cell integrates up to each event on its own (a divergent loop:
//    sub-step of length h, a8, next event from the ring), then every lane finishes the cell together with its own
//    remaining length (a5).  The Gaussian of a grid cell comes from the Gaussian stream indexed by the CELL, the
//    Gaussian of a sub-step that ends at event k from the spare word of call k of that event's stream (R13), so the
//    normal cache never gets out of phase between lanes;
//  * a jump clock is (cell index, offset in that cell), so nothing small is ever subtracted from something large;
//  * the Box-Muller radius carries the noise amplitude (sqrt(-2 ln u) * sqrt(2 D dt) in one MUFU.SQRT);
//  * uniforms come from Philox words through a mantissa splice (no I2F).  BM_GAUSS_W32: one word per uniform,
//    four normals per call (the oracle's assignment R3, so a jump-free fp32 path follows the oracle's path);
//    BM_GAUSS_W16: radius from the top 23 bits and angle from the low 16 bits of ONE word, eight normals per
//    call -- half the integer work (IMAD.WIDE is a quarter-rate instruction on sm_100, DESIGN.md s.6);
//    BM_GAUSS_W16P: W16 with the angle's sine and cosine as polynomials on the FMA pipe (two MUFU per pair);
//  * transcendental functions: MUFU.{COS,SIN,LG2,SQRT} (SFU variant) or, for the force cosine,
//    an even polynomial on the FMA pipe (FMA variant) -- a measured choice (DESIGN.md s.6).
//  * where events are dense (more than 0.02 per path and cell) the over-damped kernel runs in its LANES form instead:
//    per-lane clocks in a sliding window of two blocks (bm_config.event_mode; "LANES form" below).  Both forms perform
//    the same operations per path -- products and sums that the compiler could contract differently in the two are
//    written out (fmaf, __fmul_rn, FMUL2) -- so their results agree bit for bit;
// fp32 results are judged statistically against the fp64 oracle (3 combined standard errors).
#pragma once
#include <type_traits>

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
    return __fadd_rn(base, (y >= 0.0f) ? k1 : -k1);
  } else {
    return fmaf(-k1, x, base);
  }
}

// a6: Alg. 1 over a sub-step h with drift a(x) = K0 + f(x), f = -V' without its constant:
//   x1 = xs + h a(x);  x2 = xs + h/2 (a(x) + a(x1));  x' = xs + h/2 (a(x) + a(x2)),   xs = x + noise.
// k1 = h K1, k2 = h K2, k0h = h/2 K0, k1h, k2h likewise.  With xh = (xs + x1)/2 + k0/2 = xs + h/2 a(x) + k0/2 the
// last two stages are xh + (h/2) f(.).  `xarg` is where a(x) is evaluated (x before folding: same angle).
// The constant part of the first stage enters as ONE multiply-add, fma(h, K0, xs): written out, so that every path
// through the kernels rounds it alike (left to the compiler, xs + h K0 is contracted in one place and not in another),
// and no register has to hold h K0.
template <int POT, int SINCOS>
__device__ __forceinline__ float pc_overdamped_f32(float xarg, float xs, float h, float K0, float k1, float k2, float k0h,
                                                   float k1h, float k2h) {
  const float x1 = stage_f32<POT, SINCOS>(fmaf(h, K0, xs), xarg, k1, k2);
  const float xh = fmaf(0.5f, x1, fmaf(0.5f, xs, k0h));
  const float x2 = stage_f32<POT, SINCOS>(xh, x1, k1h, k2h);
  return stage_f32<POT, SINCOS>(xh, x2, k1h, k2h);
}

// Two independent fp32 multiply-adds in one instruction (FFMA2 on sm_100; PTX fma.rn.f32x2): each half is rounded
// exactly as a scalar FFMA, so packing changes the issue-slot count, not the result.  (ptxas takes a half that is
// the same register in both lanes of an operand as a broadcast operand.)
__device__ __forceinline__ void ffma2(float a0, float a1, float b0, float b1, float c0, float c1, float &r0, float &r1) {
  unsigned long long pa, pb, pc, pr;
  asm("mov.b64 %0, {%1, %2};" : "=l"(pa) : "f"(a0), "f"(a1));
  asm("mov.b64 %0, {%1, %2};" : "=l"(pb) : "f"(b0), "f"(b1));
  asm("mov.b64 %0, {%1, %2};" : "=l"(pc) : "f"(c0), "f"(c1));
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(pr) : "l"(pa), "l"(pb), "l"(pc));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(r0), "=f"(r1) : "l"(pr));
}

// Two independent fp32 products in one instruction (FMUL2): a * (b0, b1), each half rounded as a scalar FMUL.
__device__ __forceinline__ void fmul2(float a, float b0, float b1, float &r0, float &r1) {
  unsigned long long pa, pb, pr;
  asm("mov.b64 %0, {%1, %2};" : "=l"(pa) : "f"(a), "f"(a));
  asm("mov.b64 %0, {%1, %2};" : "=l"(pb) : "f"(b0), "f"(b1));
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(pr) : "l"(pa), "l"(pb));
  asm("mov.b64 {%0, %1}, %2;" : "=f"(r0), "=f"(r1) : "l"(pr));
}

// a7: R7.  y = (x, v), A = (v, -gamma v + f(x) + b(t)); noise in v only (vs = v + noise).  b0 = constant force +
// drive at t, b1 = the same at t + h; kk1, kk2 are the (unscaled) potential constants in theta units.
// The two components of the model give pairs of independent multiply-adds at every stage -- (x + h v, x + h/2 v),
// (kk1 + kk2 c, b - gamma v), (v + h a, v + h/2 a) -- which are issued as FFMA2: 12 instead of 17 FP instructions
// behind the three cosines, same operations, same roundings.
template <int SINCOS>
__device__ __forceinline__ void pc_inertial_f32(float &x, float &v, float xf, float vs, float h, float hh, float gamma,
                                                float kk1, float kk2, float b0, float b1) {
  const float ng = -gamma;
  const float c1 = cos_theta<SINCOS>(x);
  float xb1, xh;
  ffma2(h, hh, v, v, xf, xf, xb1, xh);
  const float c2 = cos_theta<SINCOS>(xb1);  // does not wait for c1
  float p, q;
  ffma2(kk2, ng, c1, v, kk1, b0, p, q);
  const float a1 = fmaf(c1, p, q);
  float vb1, vh;
  ffma2(h, hh, a1, a1, vs, vs, vb1, vh);
  ffma2(kk2, ng, c2, vb1, kk1, b1, p, q);
  const float a2 = fmaf(c2, p, q);
  const float xb2 = fmaf(hh, vb1, xh);
  const float c3 = cos_theta<SINCOS>(xb2);
  const float vb2 = fmaf(hh, a2, vh);
  ffma2(kk2, ng, c3, vb2, kk1, b1, p, q);
  const float a3 = fmaf(c3, p, q);
  x = fmaf(hh, vb2, xh);
  v = fmaf(hh, a3, vh);
}

// Cell index and offset of an event W cells after (n, tau); offsets are in time units, 0 <= off < dt.
__device__ __forceinline__ void schedule_f32(int n, float tau, float dt, float inv_dt, float Wcells, int &cell, float &off) {
  const float q = fmaf(tau, inv_dt, Wcells);
  float c = floorf(q);
  float f = (q - c) * dt;
  if (!(Wcells < 2.0e9f)) { cell = 0x7FFFFFFF; off = 0.0f; return; }  // beyond any run (also a rate of zero: never)
  if (f >= dt) { f = 0.0f; c += 1.0f; }
  if (c == 0.0f) f = fmaxf(f, tau);  // never schedule into the past of this cell
  // c <= 2e9 < 2^31: the 32-bit conversion is exact, and n + c < 2^32 cannot wrap as unsigned
  const unsigned t = (unsigned)n + (unsigned)__float2int_rz(c);
  cell = (int)min(t, 0x7FFFFFFFu);
  off = f;
}

// ---- Gaussian cache (a3 + a4) ---------------------------------------------------------------------------------
// A Box-Muller pair left in factors, with the amplitude inside the root: r = sqrt(cn * lg2 u), cn = -2 ln2 * s^2,
// so that s*g0 = r*c and s*g1 = r*s cost one FFMA each at the point of use.
struct Pair { float r, c, s; };

// R3 assignment: radius from word wa, angle from word wb (top 23 bits of each)
__device__ __forceinline__ Pair pair_w32(uint32_t wa, uint32_t wb, float cn) {
  Pair p;
  p.r = sqrt_approx(cn * lg2_approx(u01_open0_f32(wa)));
  const float ang = turns12_f32(wb) * TWO_PI_F;
  p.c = cos_approx(ang);
  p.s = sin_approx(ang);
  return p;
}
// compact assignment: radius from the top 23 bits of w (u on a 2^-23 grid), angle 2 pi k / 65536 from its low 16 bits
// (k spliced into the low mantissa bits: t = 1 + k 2^-23, angle = (t - 1) * 2^7 * 2 pi in one FFMA, one rounding)
__device__ __forceinline__ Pair pair_w16(uint32_t w, float cn) {
  Pair p;
  p.r = sqrt_approx(cn * lg2_approx(u01_open0_f32(w)));
  const float t = __uint_as_float((w & 0xFFFFu) | 0x3F800000u);
  const float ang = fmaf(t, 128.0f * TWO_PI_F, -128.0f * TWO_PI_F);
  p.c = cos_approx(ang);
  p.s = sin_approx(ang);
  return p;
}

// W16P: the W16 assignment with the angle's sine and cosine on the FMA pipe: r = k/65536 - 1/2 turns (exact),
// cos 2 pi r and sin 2 pi r / r as degree-5 polynomials in r^2 (Chebyshev-node fits on |r| <= 1/2; absolute error
// with fp32 Horner evaluation 1.3e-6 and 6e-7: the class of MUFU.COS / MUFU.SIN).  Two MUFU per pair instead of four.
__device__ __forceinline__ Pair pair_w16p(uint32_t w, float cn) {
  Pair p;
  p.r = sqrt_approx(cn * lg2_approx(u01_open0_f32(w)));
  const float t = __uint_as_float((w & 0xFFFFu) | 0x3F800000u);
  const float r = fmaf(t, 128.0f, -128.5f);
  const float s = r * r;
  // coefficients negated: the angle is 2 pi k / 65536 = 2 pi r + pi (the same angle as W16)
  float c = 2.107110563e+01f, q = 1.247124353e+01f;
  c = fmaf(c, s, -5.879049212e+01f); q = fmaf(q, s, -4.134288235e+01f);
  c = fmaf(c, s, 8.527162153e+01f);  q = fmaf(q, s, 7.661447253e+01f);
  c = fmaf(c, s, -6.492865742e+01f); q = fmaf(q, s, -8.159994333e+01f);
  c = fmaf(c, s, 1.973898036e+01f);  q = fmaf(q, s, 4.134158923e+01f);
  c = fmaf(c, s, -9.999992108e-01f); q = fmaf(q, s, -6.283184916e+00f);
  p.c = c;
  p.s = q * r;
  return p;
}

// Gaussian-stream call b serves NB = 4 (W32) or 8 (W16, W16P) consecutive grid cells = NB/2 Box-Muller pairs
// Standard normal of a sub-step that ends on an event, from the third word of the event's own Philox call (R13): radius
// from the word's top 23 bits, angle from its low 16 (the W16 assignment), cosine member of the pair.  Used by the path
// kernels and, on given words, by bm_event_normal_words.
__device__ __forceinline__ float event_normal_f32(uint32_t w) {
  const float r = sqrt_approx(-2.0f * LN2_F * lg2_approx(u01_open0_f32(w)));
  const float t = __uint_as_float((w & 0xFFFFu) | 0x3F800000u);
  return r * cos_approx(fmaf(t, 128.0f * TWO_PI_F, -128.0f * TWO_PI_F));
}

template <int GW> struct GaussLayout {
  static constexpr int NB = GW == BM_GAUSS_W32 ? 4 : 8;
  static constexpr int NP = NB / 2;
};

// pair I of the call whose words are w (I is a compile-time constant at every use)
template <int GW>
__device__ __forceinline__ Pair pair_of(const uint4 &w, int I, float cn) {
  if (GW == BM_GAUSS_W32) return I == 0 ? pair_w32(w.x, w.y, cn) : pair_w32(w.z, w.w, cn);
  const uint32_t ww = I == 0 ? w.x : I == 1 ? w.y : I == 2 ? w.z : w.w;
  return GW == BM_GAUSS_W16P ? pair_w16p(ww, cn) : pair_w16(ww, cn);
}

// Standard normals of call b in cell order (bm_gauss_fill)
template <int GW>
__device__ __forceinline__ void gauss_block_standard_f32(const PhiloxKeys &K, unsigned long long g, uint32_t b, float *out) {
  const uint4 w = philox_call(K, g, STREAM_GAUSS, b);
#pragma unroll
  for (int i = 0; i < GaussLayout<GW>::NP; ++i) {
    const Pair q = pair_of<GW>(w, i, -2.0f * LN2_F);
    out[2 * i] = q.r * q.c;
    out[2 * i + 1] = q.r * q.s;
  }
}

// ---- event queues (a5, a8) -----------------------------------------------------------------------------------
// The kick and flip times of a path do not depend on its motion, so they are drawn AHEAD of time: per path and jump
// stream the next event sits in registers (cell, offset, amplitude, normal of the sub-step that ends on it) and up to
// EVQ later ones in a ring in shared memory (one record per thread, odd word stride: see the layout in the kernel).
// The rings are refilled by the whole warp at once, in uniform control flow at the top of a block of cells, EVK
// events per lane and episode, so one pass of Philox rounds serves up to 32 events instead of the one or two lanes
// that happen to have an event in a cell.  An episode starts when the last queued event of some lane falls into the
// block about to run; afterwards every event of the block is known (the block is COVERED) unless a lane has more than
// EVQ of them, in which case the block runs cell by cell with refills in between (CAREFUL).
// EVQ (ring capacity), EVK (refill passes per episode) and the shared-memory layout: common.cuh

// covered non-clean blocks: unrolled pair slots (1) or one rolled copy of the slot code (0) -- a measured choice
#ifndef BM_F32_UNROLLED
#define BM_F32_UNROLLED(inertial) (!(inertial))
#endif

// register budget of the path kernel (experiment builds override it with -DBM_F32_MAXNREG=n)
// OCC = 1: the over-damped kernel within 64 registers, for grids of many blocks per SM (C4: 8 instead of 5 resident
// 128-thread blocks); OCC = 0: what the code asks for (~95 registers; no re-materialised constants), for ensembles
// that fit the device in one wave anyway (C1).  A measured choice.
#ifdef BM_F32_MAXNREG
#define BM_F32_BOUNDS(model, occ) __maxnreg__(BM_F32_MAXNREG)
#else
#define BM_F32_BOUNDS(model, occ) __launch_bounds__((model) == BM_INERTIAL ? 256 : 512, ((model) != BM_INERTIAL && (occ)) ? 2 : 1)
#endif

// A thread's record in dynamic shared memory, addressed in the shared state space: one 32-bit base kept in a register and
// immediate word offsets.  (Through generic pointers the 64-register class rebuilt the shared window's base -- S2R, MOV,
// IADD3, LEA, S2R, IMAD -- in every slow cell.)  volatile + "memory": a load is never moved across a store of the record.
struct SmemRec {
  uint32_t base;
  template <int W>
  __device__ __forceinline__ uint32_t ld(uint32_t dyn_bytes = 0u) const {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(base + dyn_bytes), "n"(4 * W) : "memory");
    return v;
  }
  template <int W>
  __device__ __forceinline__ void st(uint32_t v, uint32_t dyn_bytes = 0u) const {
    asm volatile("st.shared.u32 [%0+%1], %2;" : : "r"(base + dyn_bytes), "n"(4 * W), "r"(v) : "memory");
  }
};

// Per-point constants, fp32, theta units (theta = SCALE x)
struct PointF32 {
  float kk1, kk2;    // SINE2: SCALE * (-V') = base-part + c (kk1 + kk2 c), c = cos theta.  PWL/QUAD: kk1 = A1
  float base;        // SCALE * (F - lambda zeta (+ 4 pi A2 for SINE2))
  float Ga, Gb;      // SCALE * (-Fa), SCALE * (+Fb)
  float cn;          // -2 ln2 * SCALE^2 * 2 D dt: Box-Muller radius^2 per unit of lg2 u, full grid step
  float s2;          // SCALE^2 * 2 D: variance of the Gaussian increment per unit time
  float inv_lam_dt;  // 1/(lambda dt): waiting time in cells = -ln u * inv_lam_dt
  float zeta;        // SCALE * zeta
  float inv_mua_dt, inv_mub_dt;
  float gamma;
  float amp;         // SCALE * drive amplitude
  float w_turns;     // omega/(2 pi): drive turns per unit time
};

template <int MODEL, int POT, int NOISE, int SINCOS, int GW, int OCC, int LCLK = 0>
__global__ void BM_F32_BOUNDS(MODEL, OCC) bm_paths_f32(const __grid_constant__ SimArgs a) {
  constexpr bool HAS_G = NOISE & BM_NOISE_GAUSS, HAS_P = NOISE & BM_NOISE_POISSON, HAS_D = NOISE & BM_NOISE_DICH;
  constexpr bool HAS_EV = HAS_P || HAS_D;
  constexpr bool INERTIAL = MODEL == BM_INERTIAL;
  static_assert(!LCLK || (HAS_EV && !INERTIAL), "per-lane clocks: over-damped model with a jump source");
  static_assert(EVQ == 8, "the ring pop clears bit 3 of the read slot");
  constexpr int NB = GaussLayout<GW>::NB, NP = GaussLayout<GW>::NP;  // grid cells, pairs per Gaussian call
  constexpr float S = Units<POT>::SCALE;
  constexpr unsigned FULL = 0xffffffffu;
  constexpr int NEVER = 0x7FFFFFFF;
  constexpr int NFP = HAS_P ? EV_FIELDS_P : 0, NFD = HAS_D ? EV_FIELDS_D : 0;

  extern __shared__ uint32_t smem_words[];
  const int tid = threadIdx.x;
  // One record of REC words per thread, [ring P][ring D][cold]( + [normals] in the LANES form), REC odd: every offset
  // inside the record is an immediate of the load or store, and the few lanes that pop an event at the same time rarely
  // share a bank (lanes 32 / gcd apart in the odd stride).  (A field-major layout [slot][field][thread] is conflict-free
  // whatever slot each lane is at, but its strides are run-time values: the 64-register class rebuilt the addresses at
  // every pop, ~10 instructions; measured: C1 12.79 -> 12.70 ms, C2 39.0 -> 38.5 ms with the records.)
  constexpr int RECW = EVQ * NFP + EVQ * NFD + 4 + (HAS_G ? (LCLK ? 4 * NB : (GW == BM_GAUSS_W32 ? 0 : 4)) : 0), REC = RECW | 1;
  constexpr int OFF_D = EVQ * NFP, OFF_COLD = EVQ * (NFP + NFD), OFF_NRM = OFF_COLD + 4;  // word offsets in the record
  // [ring P: EVQ x NFP][ring D: EVQ x NFD][cold: snap_x, snap_w, drawnP, drawnD][LANES: normals of two blocks; CELLS, W16:
  // the four words the rolled paths form their pairs from]
  // State that is touched a few times per run lives here, not in registers: the snapshot at t_i and, per stream, the
  // number of events drawn so far.  The index of a stream's next event = events drawn - events queued - 1 = events
  // applied, so no counter has to follow the events themselves.
  SmemRec R;
  R.base = (uint32_t)__cvta_generic_to_shared(smem_words + tid * REC);
  asm volatile("" : "+r"(R.base));  // a value to keep, not an address to rebuild

  const int point = blockIdx.x / a.blocks_per_point;
  const int chunk = blockIdx.x - point * a.blocks_per_point;
  const long long p = (long long)chunk * blockDim.x + threadIdx.x;
  const bool valid = p < a.n_paths;  // lanes past a ragged end run along (the warp votes) and contribute nothing
  const unsigned long long g =
      (unsigned long long)point * (unsigned long long)a.n_paths + (unsigned long long)(valid ? p : 0);

  const PhiloxKeys &K = a.keys;
  const bm_params bp = a.params[point];
  // the two forms of the kernel share a launch grid: each takes the parameter points of its own event mode
  if (HAS_EV && MODEL == BM_OVERDAMPED && lane_clock_point(a, bp, step_length(a, point), NOISE) != (LCLK != 0)) return;
  const double Dd = HAS_G ? bp.D : 0.0;
  const double dtd = step_length(a, point);
  float dt = (float)dtd;
  // (an empty asm makes dt a value the compiler has to keep: in the 64-register class it would rather convert the double
  // kernel parameter again at every use -- an F2F on the XU pipe in each of the slow-cell copies)
  asm volatile("" : "+f"(dt));
  const float inv_dt = (float)(1.0 / dtd);
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
  // a non-positive rate of leaving -Fa switches the dichotomous source off at this point (Gamma = 0, as the oracle);
  // a non-positive rate of leaving +Fb makes that state absorbing
  const bool onD = HAS_D && bp.mu_a > 0.0;
  P.Ga = onD ? (float)((double)S * (-bp.Fa)) : 0.f;
  P.Gb = onD ? (float)((double)S * bp.Fb) : 0.f;
  P.cn = (float)(-2.0 * M_LN2 * (double)S * (double)S * 2.0 * Dd * dtd);
  P.s2 = (float)((double)S * (double)S * 2.0 * Dd);
  P.inv_lam_dt = (lam > 0.0) ? (float)(1.0 / (lam * dtd)) : 0.f;
  P.zeta = (float)((double)S * zet);
  P.inv_mua_dt = onD ? (float)(1.0 / (bp.mu_a * dtd)) : 0.f;
  P.inv_mub_dt = (onD && bp.mu_b > 0.0) ? (float)(1.0 / (bp.mu_b * dtd)) : __int_as_float(0x7f800000);
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
  if (onD) d = ((((double)wi.z + 0.5) * (1.0 / 4294967296.0)) < bp.mu_a / (bp.mu_a + (bp.mu_b > 0.0 ? bp.mu_b : 0.0))) ? 1 : 0;  // mu_b <= 0: +Fb absorbing, every path starts there

  // Standard normal of the sub-step that ends on an event, from the third word of the event's Philox call (R13):
  // radius from its top 23 bits, angle from its low 16 (the W16 assignment).
  auto event_normal = [](uint32_t w) -> float { return event_normal_f32(w); };

  const int n_discard = (int)a.n_discard;
  // next event of each stream: (cell index, offset inside that cell); NEVER = switched off at this point.  qP, qD:
  // ring read slot (bits 0-3) and fill (bits 4-); the index of the event in its stream follows from the draw count.
  int nP = NEVER, nD = NEVER;
  float fP = 0.f, fD = 0.f, z = 0.f, gP = 0.f, gD = 0.f;
  uint32_t drawnP = 0, drawnD = 0;  // stored to `cold` below; registers only during the set-up
  int qP = 0, qD = 0;
  // lanes past a ragged end stay inert: no events, no checkpoint traffic (they must not steer the warp's votes)
  if (HAS_P && lam > 0.0 && valid) {
    const uint4 w = philox_call(K, g, STREAM_POISSON, 0);
    schedule_f32(0, 0.f, dt, inv_dt, neg_log_u_f32(w.x) * P.inv_lam_dt, nP, fP);
    z = P.zeta * neg_log_u_f32(w.y);
    if (HAS_G) gP = event_normal(w.z);
    drawnP = 1;
  }
  if (onD && valid) {
    const uint4 w = philox_call(K, g, STREAM_DICH, 0);
    schedule_f32(0, 0.f, dt, inv_dt, neg_log_u_f32(w.x) * (d ? P.inv_mub_dt : P.inv_mua_dt), nD, fD);
    if (HAS_G) gD = event_normal(w.z);
    drawnD = 1;
  }

  // drive phase in 2^-64 turns per cell (inertial): exact integer accumulation, no float time.  n is the same in
  // every lane, so ph and the drive at the cell boundaries are warp-uniform values.
  unsigned long long ph = 0, dph = 0;
  float drive0 = 0.f;  // SCALE * amp * cos(omega n dt)
  if (INERTIAL) {
    double turns_per_cell = bp.omega * dtd / (2.0 * M_PI);
    turns_per_cell -= floor(turns_per_cell);
    dph = (unsigned long long)(turns_per_cell * 18446744073709551616.0);
    drive0 = P.amp;  // cos(0)
  }

  float snap_x = x;  // stored to `cold` below
  int snap_w = wraps;
  // row f2: a launch that continues a run reloads everything the lines above initialised (the Philox calls of the
  // initialisation are wasted then, once per launch).  The rings are not part of the state: they restart empty and
  // refill with the same events (an event is a function of its predecessor and its Philox call only).
  const int n_begin = (int)a.step_begin, n_end = (int)a.step_end;
  if (a.state != nullptr && n_begin > 0 && valid) {
    const StateIO io = state_io(a, g);
    uint32_t lo, hi;
    io.get2(0, lo, hi); x = __uint_as_float(lo); wraps = (int)hi;
    io.get2(1, lo, hi); v = __uint_as_float(lo);  // (hi: events applied = the two stream indices below)
    io.get2(2, lo, hi); nP = (int)lo; fP = __uint_as_float(hi);
    io.get2(3, lo, hi); z = __uint_as_float(lo); drawnP = (nP != NEVER || hi != 0u) ? hi + 1u : 0u;
    io.get2(4, lo, hi); gP = __uint_as_float(lo); gD = __uint_as_float(hi);
    io.get2(5, lo, hi); nD = (int)lo; fD = __uint_as_float(hi);
    io.get2(6, lo, hi); drawnD = (nD != NEVER || lo != 0u) ? lo + 1u : 0u; d = (int)hi;
    ph = io.get(7);
    io.get2(8, lo, hi); drive0 = __uint_as_float(lo); snap_x = __uint_as_float(hi);
    io.get2(9, lo, hi); snap_w = (int)lo;
  }
  R.template st<OFF_COLD + 0>(__float_as_uint(snap_x));
  R.template st<OFF_COLD + 1>((uint32_t)snap_w);
  R.template st<OFF_COLD + 2>(drawnP);
  R.template st<OFF_COLD + 3>(drawnD);
  int cov = min(nP, nD);  // cell of the last event known to this lane, minimum over the streams
  float cst = P.base + (HAS_D ? (d ? P.Gb : P.Ga) : 0.f);
  const float hh_full = 0.5f * dt;
  // full-step constants of Alg. 1 (loop invariant; k0h follows cst across a flip)
  // (products by __fmul_rn: the compiler must not contract them into the additions that follow, or the CELLS and the
  // LANES form of the kernel, and fast_cell and sub_step, would round differently)
  float k1f = __fmul_rn(dt, P.kk1), k2f = __fmul_rn(dt, P.kk2), k1h = __fmul_rn(hh_full, P.kk1), k2h = __fmul_rn(hh_full, P.kk2);
  float k0h = __fmul_rn(hh_full, cst);
  // (64-register class: kept as values, or the compiler multiplies them out again in every pair of cells)
  if (OCC && !LCLK) asm volatile("" : "+f"(k1f), "+f"(k2f), "+f"(k1h), "+f"(k2h));

  // ---- one refill pass: every lane with room appends one event per stream; returns whether this lane still has a
  //      stream whose last event lies before `limit` and whose ring has room ------------------------------------
  auto refill_pass = [&](int limit, bool &did) -> bool {
    bool more = false;
    int tailP = NEVER, tailD = NEVER;
    if (HAS_P) {
      const int rd = qP & 15, cnt = qP >> 4;
      int tc = nP;
      float tf = fP;
      if (cnt > 0) {
        const int s = (rd + cnt - 1) & (EVQ - 1);
        tc = (int)R.template ld<0>(s * (NFP * 4));
        tf = __uint_as_float(R.template ld<1>(s * (NFP * 4)));
      }
      tailP = tc;
      if (cnt < EVQ && tc != NEVER) {
        const uint32_t drawn = R.template ld<OFF_COLD + 2>();
        R.template st<OFF_COLD + 2>(drawn + 1u);
        const uint4 w = philox_call(K, g, STREAM_POISSON, drawn);
        int c;
        float f;
        schedule_f32(tc, tf, dt, inv_dt, neg_log_u_f32(w.x) * P.inv_lam_dt, c, f);
        const int s = (rd + cnt) & (EVQ - 1);
        R.template st<0>((uint32_t)c, s * (NFP * 4));
        R.template st<1>(__float_as_uint(f), s * (NFP * 4));
        R.template st<2>(__float_as_uint(P.zeta * neg_log_u_f32(w.y)), s * (NFP * 4));
        if (HAS_G) R.template st<3>(__float_as_uint(event_normal(w.z)), s * (NFP * 4));
        qP += 16;
        tailP = c;
        did = true;
        more |= (c < limit) && (cnt + 1 < EVQ);
      }
    }
    if (HAS_D) {
      const int rd = qD & 15, cnt = qD >> 4;
      int tc = nD;
      float tf = fD;
      if (cnt > 0) {
        const int s = (rd + cnt - 1) & (EVQ - 1);
        tc = (int)R.template ld<OFF_D + 0>(s * (NFD * 4));
        tf = __uint_as_float(R.template ld<OFF_D + 1>(s * (NFD * 4)));
      }
      tailD = tc;
      if (cnt < EVQ && tc != NEVER) {
        const uint32_t drawn = R.template ld<OFF_COLD + 3>();
        R.template st<OFF_COLD + 3>(drawn + 1u);
        const uint4 w = philox_call(K, g, STREAM_DICH, drawn);
        const int dn = d ^ ((cnt + 1) & 1);  // the state entered by the last queued flip
        int c;
        float f;
        schedule_f32(tc, tf, dt, inv_dt, neg_log_u_f32(w.x) * (dn ? P.inv_mub_dt : P.inv_mua_dt), c, f);
        const int s = (rd + cnt) & (EVQ - 1);
        R.template st<OFF_D + 0>((uint32_t)c, s * (NFD * 4));
        R.template st<OFF_D + 1>(__float_as_uint(f), s * (NFD * 4));
        if (HAS_G) R.template st<OFF_D + 2>(__float_as_uint(event_normal(w.z)), s * (NFD * 4));
        qD += 16;
        tailD = c;
        did = true;
        more |= (c < limit) && (cnt + 1 < EVQ);
      }
    }
    cov = min(tailP, tailD);
    return more;
  };
  // an episode: at least EVK passes (every lane with room takes part, so a pass is shared by the whole warp), then on
  // until no lane that is still short of `limit` has room
  auto refill_episode = [&](int limit) {
    for (int pass = 0;; ++pass) {
      bool did = false;
      const bool more = refill_pass(limit, did);
      if (!__any_sync(FULL, did)) break;
      if (pass + 1 >= EVK && !__any_sync(FULL, more)) break;
    }
  };
  // (a popped event always has a queued successor: the block is covered, or -- careful path -- the rings were refilled
  // before the turn; so the ring is never empty here)
  auto pop_P = [&]() {
    const int s = qP & 15;
    nP = (int)R.template ld<0>(s * (NFP * 4));
    fP = __uint_as_float(R.template ld<1>(s * (NFP * 4)));
    z = __uint_as_float(R.template ld<2>(s * (NFP * 4)));
    if (HAS_G) gP = __uint_as_float(R.template ld<3>(s * (NFP * 4)));
    qP = (qP - 15) & ~EVQ;  // one event less queued, read slot + 1 modulo EVQ (EVQ = 8: bit 3 of the slot is the wrap)
  };
  auto pop_D = [&]() {
    const int s = qD & 15;
    nD = (int)R.template ld<OFF_D + 0>(s * (NFD * 4));
    fD = __uint_as_float(R.template ld<OFF_D + 1>(s * (NFD * 4)));
    if (HAS_G) gD = __uint_as_float(R.template ld<OFF_D + 2>(s * (NFD * 4)));
    qD = (qD - 15) & ~EVQ;
  };

  // ---- FAST: a full grid step without events in this lane (h = dt); noise = gr * gc ----------------------------
  auto fast_cell = [&](float gr, float gc, bool do_fold) {
    float xf = x;
    if (do_fold || POT != BM_POT_SINE2) fold_f32<POT>(xf, wraps);
    if (!INERTIAL) {
      const float xs = HAS_G ? fmaf(gr, gc, xf) : xf;
      x = pc_overdamped_f32<POT, SINCOS>(POT == BM_POT_SINE2 ? x : xf, xs, dt, cst, k1f, k2f, k0h, k1h, k2h);
    } else {
      ph += dph;
      const float drive1 = P.amp * cos_turns<SINCOS>(__uint_as_float((uint32_t)(ph >> 41) | 0x3F800000u));
      const float vs = HAS_G ? fmaf(gr, gc, v) : v;
      pc_inertial_f32<SINCOS>(x, v, xf, vs, dt, hh_full, P.gamma, P.kk1, P.kk2, cst + drive0, cst + drive1);
      drive0 = drive1;
    }
  };

  // ---- a5-a8: a sub-step of length h from the lane's current state; noise = na * nb; dr0/dr1 = drive at its ends.
  //      With h = dt, refold = false and (na, nb) = (gr, gc) this is fast_cell(gr, gc, first) operation by operation, so a lane
  //      without an event gets the same result whichever way its warp takes through a cell. -----------------------
  //      `first`: the lane's first sub-step in a block of NB cells.  The position is re-folded there (a9); when that
  //      sub-step is a whole cell the force is still evaluated at the position as it stands (the same angle), so the
  //      cosine does not wait for the fold -- in every path through the kernel, clean block or not.
  auto sub_step = [&](float h, float na, float nb, float dr0, float dr1, bool refold, bool first) {
    const float hh = 0.5f * h;
    float xf = x;
    int wf = wraps;
    fold_f32<POT>(xf, wf);
    if (refold || POT != BM_POT_SINE2) { wraps = wf; x = xf; }  // base and argument folded
    else if (first) wraps = wf;                                  // base folded, argument as it stands
    else xf = x;
    if (!INERTIAL) {
      const float xs = HAS_G ? fmaf(na, nb, xf) : xf;
      float k1, k2, k1h, k2h;
      fmul2(h, P.kk1, P.kk2, k1, k2);
      fmul2(hh, P.kk1, P.kk2, k1h, k2h);
      x = pc_overdamped_f32<POT, SINCOS>(x, xs, h, cst, k1, k2, __fmul_rn(hh, cst), k1h, k2h);
    } else {
      const float vs = HAS_G ? fmaf(na, nb, v) : v;
      pc_inertial_f32<SINCOS>(x, v, xf, vs, h, hh, P.gamma, P.kk1, P.kk2, cst + dr0, cst + dr1);
    }
  };

  // One event of this lane in cell c (the lane's earliest; a tie applies the kick first, R5): integrate to it, apply
  // it (a8) and take the next event of that stream from the ring.
  auto do_event = [&](float &tau, float &dr_tau, float phf) {
    const bool isP = HAS_P && (!HAS_D || nP < nD || (nP == nD && fP <= fD));
    const float te = isP ? fP : fD;
    const float h = fmaxf(te - tau, 0.f);
    float dr1 = 0.f;
    if (INERTIAL) dr1 = P.amp * cos_turns<SINCOS>(fmaf(te, P.w_turns, phf));
    sub_step(h, HAS_G ? (isP ? gP : gD) : 0.f, HAS_G ? sqrt_approx(h * P.s2) : 0.f, dr_tau, dr1, true, false);  // Var ~ h (A9)
    dr_tau = dr1;
    tau = te;
    if (HAS_P && isP) {  // a8: kick
      if (!INERTIAL) x = __fadd_rn(x, z); else v += z;
      pop_P();
    }
    if (HAS_D && !isP) {  // a8: flip
      d ^= 1;
      cst = P.base + (d ? P.Gb : P.Ga);
      k0h = __fmul_rn(hh_full, cst);
      pop_D();
    }
  };

  // ---- SLOW: a cell in which at least one lane of the warp has a kick or a flip.  Event lanes integrate up to each
  //      of their events on their own, then every lane finishes the cell with its own remaining length (a5): the
  //      whole cell, with the fast cell's arithmetic, for a lane without events. ----------------------------------
  auto finish_cell = [&](float gr, float gc, float tau, float dr_tau, bool first) {
    const bool whole = tau == 0.f;
    const float h = dt - tau;
    float na = gr, nb = gc;
    if (HAS_G && !whole) { na = gr * gc; nb = sqrt_approx(h * inv_dt); }
    float drive1 = 0.f;
    if (INERTIAL) {
      ph += dph;
      drive1 = P.amp * cos_turns<SINCOS>(__uint_as_float((uint32_t)(ph >> 41) | 0x3F800000u));
    }
    sub_step(h, na, nb, dr_tau, drive1, !whole, first);
    drive0 = drive1;
  };
  auto slow_cell = [&](int c, float gr, float gc, bool first) {
    float tau = 0.f;         // the lane's offset inside cell c
    float dr_tau = drive0;   // drive at that time
    const float phf = INERTIAL ? __uint_as_float((uint32_t)(ph >> 41) | 0x3F800000u) : 0.f;  // 1 + frac(omega c dt / 2 pi)
    while ((HAS_P && nP == c) || (HAS_D && nD == c)) do_event(tau, dr_tau, phf);
    finish_cell(gr, gc, tau, dr_tau, first);
  };

  // Events of this lane in cells [n, n+32) as a bit mask (bit = cell - n; shl.b32 clamps a shift >= 32 to zero, so
  // NEVER and any far cell give 0).
  auto ev_bits = [&](int n) -> unsigned {
    unsigned bits = 0, t;
    if (HAS_P) { asm("shl.b32 %0, 1, %1;" : "=r"(t) : "r"((unsigned)(nP - n))); bits |= t; }
    if (HAS_D) { asm("shl.b32 %0, 1, %1;" : "=r"(t) : "r"((unsigned)(nD - n))); bits |= t; }
    return bits;
  };

  // ---- time loop: blocks of NB cells = one Gaussian call -------------------------------------------------------
  // A block is CLEAN when no lane of the warp has an event in it and it holds neither t_i nor the end of the run:
  // NB fast cells, one vote.  Otherwise the warp makes sure the block's events are queued, builds a uniform control
  // word (bit j: some lane has an event in cell n+j; bit 8+j: cell n+j is the snapshot cell or lies beyond the end)
  // and tests one bit pair per cell.  The Box-Muller pair of cells (2i+2, 2i+3) is formed while cells (2i, 2i+1) run
  // (its consumer is near, so the instruction scheduler fills the stalls of the serial predictor-corrector chain with
  // it), and the Philox call of the next block is issued at the top of the block.
  constexpr bool UNROLLED = BM_F32_UNROLLED(INERTIAL);  // covered non-clean blocks: unrolled pair slots or a rolled slot loop
  constexpr bool FIRST = !INERTIAL;  // re-fold in the lane's first sub-step of a non-clean block
  uint4 w = make_uint4(0u, 0u, 0u, 0u);
  Pair cur = Pair{0.f, 0.f, 0.f};
  if (HAS_G && !LCLK) {
    w = philox_call(K, g, STREAM_GAUSS, (uint32_t)(n_begin / NB));
    cur = pair_of<GW>(w, 0, P.cn);
  }
  // rounds of the next Gaussian call done in pair slot i: NP = 4: 4 + 3 + 3 + 0, NP = 2: 10 + 0
  auto next_rounds = [&](uint4 &c, int i) {
    if (NP == 4) {
      if (i == 0) philox_rounds<0, 4>(c, K);
      if (i == 1) philox_rounds<4, 7>(c, K);
      if (i == 2) philox_rounds<7, 10>(c, K);
    } else if (i == 0) {
      philox_rounds<0, 10>(c, K);
    }
  };
  // a10: the snapshot at t_i, or nothing at all beyond the end of the run (returns false)
  auto special_cell = [&](int n, int j, unsigned ctl) -> bool {
    if ((ctl >> j) & 0x100u) {
      if (n + j >= n_end) return false;
      fold_f32<POT>(x, wraps);
      R.template st<OFF_COLD + 0>(__float_as_uint(x));
      R.template st<OFF_COLD + 1>((uint32_t)wraps);
    }
    return true;
  };
  // pair I of the block's Gaussian call, or the first pair of the next one, with a run-time index (rolled slot loop)
  auto pair_dyn = [&](const uint4 &w0, const uint4 &w1, int i) -> Pair {
    if (GW == BM_GAUSS_W32) {
      const bool last = i + 1 >= NP;
      return pair_w32(last ? w1.x : w0.z, last ? w1.y : w0.w, P.cn);
    }
    // (the word of pair i + 1 with a run-time i: from the record, where stash_words put w0.y, w0.z, w0.w, w1.x -- one
    // load instead of a four-way select)
    const uint32_t ww = R.template ld<OFF_NRM>((uint32_t)i * 4u);
    return GW == BM_GAUSS_W16P ? pair_w16p(ww, P.cn) : pair_w16(ww, P.cn);
  };
  auto stash_words = [&](const uint4 &w0, const uint4 &w1) {
    if (HAS_G && GW != BM_GAUSS_W32) {
      R.template st<OFF_NRM + 0>(w0.y);
      R.template st<OFF_NRM + 1>(w0.z);
      R.template st<OFF_NRM + 2>(w0.w);
      R.template st<OFF_NRM + 3>(w1.x);
    }
  };

  // ---- LANES form: per-lane clocks in a sliding window ------------------------------------------------------------
  // Every lane walks through the run on its own: one sub-step per pass, from its (cell c, offset tau) to its next event
  // in that cell or to the cell's end.  The warp only agrees on a WINDOW: lo = the block of NB cells its slowest lane
  // is in, G = the cell up to which the normals (two blocks in shared memory, at a per-lane index) and the events are
  // known; a lane that has reached G waits.  A lane that falls behind by an event is caught up with while the others
  // wait at most for one block, so the number of passes per cell tends to 1 + (events per cell), where blocks taken in
  // lock-step cost 1 + (the largest number of events of any lane in the block) / NB.  Per lane the operations are those
  // of the CELLS form: a cell crossed without an event is fast_cell, a sub-step that ends on an event do_event's, the
  // rest of a cell after its last event finish_cell's: the results agree bit for bit.  Blocks that hold t_i or the end
  // of the run, and blocks in which a lane has more events than its ring holds, are taken by all lanes together, cell
  // by cell (the CAREFUL path of the CELLS form).
  if (LCLK) {
    constexpr int WC = 2 * NB;  // cells in the window; nrm: angle parts [WC] at c mod WC, then the radius of each cell [WC]
    int c = n_begin;            // the lane's cell
    float tau = 0.f;            // and its offset inside it
    int lo = n_begin, G = n_begin, tried = -1;
    for (;;) {  // uniform over the warp
      if (G - lo < WC && G < n_end && tried != lo) {
        bool ok = !(((unsigned)(n_discard - G) < (unsigned)NB) || (G + NB > n_end));
        if (ok && __any_sync(FULL, cov < G + NB)) {
          refill_episode(G + NB);
          ok = !__any_sync(FULL, cov < G + NB);  // else: a ring is full; try again when the slowest lane has moved on
        }
        if (ok) {
          if (HAS_G) {
            const uint4 wg = philox_call(K, g, STREAM_GAUSS, (uint32_t)(G / NB));
            const uint32_t dst = (uint32_t)(G & (WC - 1)) * 4u;
            auto put_pair = [&](auto IT, const Pair &q) {
              constexpr int I = decltype(IT)::value;
              R.template st<OFF_NRM + 2 * I>(__float_as_uint(q.c), dst);
              R.template st<OFF_NRM + 2 * I + 1>(__float_as_uint(q.s), dst);
              R.template st<OFF_NRM + WC + 2 * I>(__float_as_uint(q.r), dst);
              R.template st<OFF_NRM + WC + 2 * I + 1>(__float_as_uint(q.r), dst);
            };
            put_pair(std::integral_constant<int, 0>(), pair_of<GW>(wg, 0, P.cn));
            put_pair(std::integral_constant<int, 1>(), pair_of<GW>(wg, 1, P.cn));
            if (NP == 4) {
              put_pair(std::integral_constant<int, 2>(), pair_of<GW>(wg, 2, P.cn));
              put_pair(std::integral_constant<int, 3>(), pair_of<GW>(wg, 3, P.cn));
            }
          }
          G += NB;
          continue;
        }
        tried = lo;
        if (lo == G) {
          // every lane stands at the start of block G: cell by cell, all lanes together
          uint4 wg = make_uint4(0u, 0u, 0u, 0u);
          if (HAS_G) wg = philox_call(K, g, STREAM_GAUSS, (uint32_t)(G / NB));
#pragma unroll 1
          for (int j = 0; j < NB; ++j) {
            const int cc = G + j;
            if (cc >= n_end) break;
            if (cc == n_discard) {  // a10: snapshot at t_i
              fold_f32<POT>(x, wraps);
              R.template st<OFF_COLD + 0>(__float_as_uint(x));
              R.template st<OFF_COLD + 1>((uint32_t)wraps);
            }
            Pair q = Pair{0.f, 0.f, 0.f};
            if (HAS_G) {
              const int i = j >> 1;
              if (GW == BM_GAUSS_W32) {
                q = pair_w32(i ? wg.z : wg.x, i ? wg.w : wg.y, P.cn);
              } else {
                const uint32_t ww = i == 0 ? wg.x : i == 1 ? wg.y : i == 2 ? wg.z : wg.w;
                q = GW == BM_GAUSS_W16P ? pair_w16p(ww, P.cn) : pair_w16(ww, P.cn);
              }
            }
            float tj = 0.f, dr_tau = 0.f;
            for (;;) {
              if (__any_sync(FULL, cov <= cc)) refill_episode(cc + 1);
              const bool mine = (HAS_P && nP == cc) || (HAS_D && nD == cc);
              if (!__any_sync(FULL, mine)) break;
              if (mine) do_event(tj, dr_tau, 0.f);
            }
            finish_cell(q.r, (j & 1) ? q.s : q.c, tj, dr_tau, j == 0);
          }
          G += NB;
          lo = G;
          c = G;
          tau = 0.f;
          tried = -1;
          continue;
        }
      }
      if (lo >= n_end) break;
      // passes, until the slowest lane has left block lo (then the window may move on).  lo < G here, so some lane is
      // below G in every pass.
      const int lo_end = lo + NB;
      do {
      if (c < G) {
        const bool evP = HAS_P && nP == c, evD = HAS_D && nD == c;
        const bool ev = evP || evD;
        const bool isP = evP && (!evD || fP <= fD);  // a tie applies the kick first (R5), as do_event
        const float te = ev ? (isP ? fP : fD) : dt;
        const bool whole = !ev && tau == 0.f;
        const bool first = (c & (NB - 1)) == 0;  // (only looked at when `whole`)
        const float h = fmaxf(te - tau, 0.f);
        float na = 0.f, nb = 0.f;
        if (HAS_G) {
          const uint32_t q = (uint32_t)(c & (WC - 1)) * 4u;
          const float gc = __uint_as_float(R.template ld<OFF_NRM>(q)), gr = __uint_as_float(R.template ld<OFF_NRM + WC>(q));
          const float sq = sqrt_approx(h * (ev ? P.s2 : inv_dt));
          na = ev ? (isP ? gP : gD) : (whole ? gr : gr * gc);
          nb = whole ? gc : sq;
        }
        {  // sub_step(h, na, nb, ., ., !whole, first), the choice of the fold as a select on the rounding constant
          float xf = x, xa = x;
          if (POT != BM_POT_QUAD) {
            float t = fmaf(x, Units<POT>::INV_PERIOD_TH, MAGIC_F);
            if (POT == BM_POT_SINE2 && whole && !first) t = MAGIC_F;  // no re-fold: zero periods taken off, exactly
            xf = fmaf(t - MAGIC_F, -Units<POT>::PERIOD_TH, x);
            wraps += __float_as_int(t) - MAGIC_BITS;
            xa = (POT == BM_POT_SINE2 && whole) ? x : xf;
          }
          const float hh = 0.5f * h;
          const float xs = HAS_G ? fmaf(na, nb, xf) : xf;
          float k1, k2, k1h, k2h;
          fmul2(h, P.kk1, P.kk2, k1, k2);
          fmul2(hh, P.kk1, P.kk2, k1h, k2h);
          x = pc_overdamped_f32<POT, SINCOS>(xa, xs, h, cst, k1, k2, __fmul_rn(hh, cst), k1h, k2h);
        }
        tau = 0.f;
        c += 1;
        if (ev) {  // the lane stays in its cell, at the time of the event
          tau = te;
          c -= 1;
          if (HAS_P && isP) {  // a8: kick
            x = __fadd_rn(x, z);
            const int s = qP & 15;
            nP = (int)R.template ld<0>(s * (NFP * 4));
            fP = __uint_as_float(R.template ld<1>(s * (NFP * 4)));
            z = __uint_as_float(R.template ld<2>(s * (NFP * 4)));
            if (HAS_G) gP = __uint_as_float(R.template ld<3>(s * (NFP * 4)));
            qP = (qP - 15) & ~EVQ;  // one event less queued, read slot + 1 modulo EVQ
          }
          if (HAS_D && !isP) {  // a8: flip
            d ^= 1;
            cst = P.base + (d ? P.Gb : P.Ga);
            const int s = qD & 15;
            nD = (int)R.template ld<OFF_D + 0>(s * (NFD * 4));
            fD = __uint_as_float(R.template ld<OFF_D + 1>(s * (NFD * 4)));
            if (HAS_G) gD = __uint_as_float(R.template ld<OFF_D + 2>(s * (NFD * 4)));
            qD = (qD - 15) & ~EVQ;
          }
        }
      }
      } while (!__all_sync(FULL, c >= lo_end));
      lo = lo_end;
    }
  }

  uint32_t blk = (uint32_t)(n_begin / NB);
  if (!LCLK)
  for (int n = n_begin; n < n_end; n += NB) {
    blk++;
    const bool special = ((unsigned)(n_discard - n) < (unsigned)NB) || (n + NB > n_end);
    const bool clean = !special && !(HAS_EV && __any_sync(FULL, min(nP, nD) < n + NB));
    // counter of the next Gaussian call; its ten rounds are spread over the pair slots of this block
    uint4 wn = make_uint4(blk, (uint32_t)STREAM_GAUSS, (uint32_t)g, (uint32_t)(g >> 32));
    if (clean) {
#pragma unroll
      for (int i = 0; i < NP; ++i) {
        Pair nxt = cur;
        if (HAS_G) {
          next_rounds(wn, i);
          nxt = (i + 1 < NP) ? pair_of<GW>(w, i + 1, P.cn) : pair_of<GW>(wn, 0, P.cn);
        }
        fast_cell(cur.r, cur.c, i == 0);
        fast_cell(cur.r, cur.s, false);
        cur = nxt;
      }
    } else {
      bool careful = false;
      if (HAS_EV && __any_sync(FULL, cov < n + NB)) {
        refill_episode(n + NB);
        careful = __any_sync(FULL, cov < n + NB);  // a lane with more than EVQ events in this block
      }
      unsigned ctl = 0;
      if (HAS_EV) ctl = __reduce_or_sync(FULL, ev_bits(n)) & 0xFFu;
      if (special) {
        if ((unsigned)(n_discard - n) < (unsigned)NB) ctl |= 0x100u << (n_discard - n);
        if (n + NB > n_end) ctl |= (0xFF00u << (n_end - n)) & 0xFF00u;
      }
      // the inertial kernel (one form only) folds once at the top of a non-clean block; the over-damped one folds in
      // the lane's first sub-step of the block (FIRST), which is what its two forms can both do
      if (INERTIAL) fold_f32<POT>(x, wraps);
      if (careful || special) {
        // CAREFUL (some lane has more events in this block than its ring holds; also the two blocks of a run that hold
        // t_i and its end, so that the covered paths below carry no test for them): every cell is taken as a slow cell,
        // in turns of one event per lane with a refill before each turn, so that a lane's next event is always
        // known before it is needed.  Same arithmetic per lane as the covered path.
        if (HAS_G) philox_rounds<0, 10>(wn, K);
        stash_words(w, wn);
#pragma unroll 1
        for (int i = 0; i < NP; ++i) {
          Pair nxt = cur;
          if (HAS_G) nxt = pair_dyn(w, wn, i);
#pragma unroll 1
          for (int jj = 0; jj < 2; ++jj) {
            const int j = 2 * i + jj, c = n + j;
            if (!special_cell(n, j, ctl)) break;
            float tau = 0.f, dr_tau = drive0;
            const float phf = INERTIAL ? __uint_as_float((uint32_t)(ph >> 41) | 0x3F800000u) : 0.f;
            for (;;) {  // uniform over the warp
              if (__any_sync(FULL, cov <= c)) refill_episode(c + 1);
              const bool mine = (HAS_P && nP == c) || (HAS_D && nD == c);
              if (!__any_sync(FULL, mine)) break;
              if (mine) do_event(tau, dr_tau, phf);
            }
            finish_cell(cur.r, jj ? cur.s : cur.c, tau, dr_tau, FIRST && j == 0);
          }
          cur = nxt;
        }
      } else if (UNROLLED) {
        // COVERED, pair slot by pair slot, unrolled: a slot without event or special cell is the clean path's code
        // for two cells (with the next block's Philox rounds and Box-Muller pair formed alongside, as there)
#pragma unroll
        for (int i = 0; i < NP; ++i) {
          Pair nxt = cur;
          if (HAS_G) {
            next_rounds(wn, i);
            nxt = (i + 1 < NP) ? pair_of<GW>(w, i + 1, P.cn) : pair_of<GW>(wn, 0, P.cn);
          }
          if (((ctl >> (2 * i)) & 3u) == 0u) {
            fast_cell(cur.r, cur.c, FIRST && i == 0);
            fast_cell(cur.r, cur.s, false);
          } else {
#pragma unroll
            for (int jj = 0; jj < 2; ++jj) {
              const int j = 2 * i + jj;
              const float gc = jj ? cur.s : cur.c;
              if (HAS_EV && ((ctl >> j) & 1u)) {
                slow_cell(n + j, cur.r, gc, FIRST && j == 0);
                ctl |= __reduce_or_sync(FULL, ev_bits(n)) & 0xFFu;  // later events of the same lanes in this block
              } else {
                fast_cell(cur.r, gc, FIRST && j == 0);
              }
            }
          }
          cur = nxt;
        }
      } else {
        // COVERED, rolled over the pair slots (one copy of the slow-cell code)
        if (HAS_G) philox_rounds<0, 10>(wn, K);
        stash_words(w, wn);
#pragma unroll 1
        for (int i = 0; i < NP; ++i) {
          Pair nxt = cur;
          if (HAS_G) nxt = pair_dyn(w, wn, i);
          if (((ctl >> (2 * i)) & 3u) == 0u) {
            fast_cell(cur.r, cur.c, FIRST && i == 0);
            fast_cell(cur.r, cur.s, false);
          } else {
#pragma unroll 1
            for (int jj = 0; jj < 2; ++jj) {
              const int j = 2 * i + jj;
              const float gc = jj ? cur.s : cur.c;
              if (HAS_EV && ((ctl >> j) & 1u)) {
                slow_cell(n + j, cur.r, gc, FIRST && j == 0);
                ctl |= __reduce_or_sync(FULL, ev_bits(n)) & 0xFFu;  // later events of the same lanes in this block
              } else {
                fast_cell(cur.r, gc, FIRST && j == 0);
              }
            }
          }
          cur = nxt;
        }
      }
    }
    w = wn;
  }

  // events applied per stream = events drawn - events still queued (the ring and the head); it is also the index of
  // the stream's next event, i.e. of the Philox call it came from
  const uint32_t kP = (HAS_P && R.template ld<OFF_COLD + 2>() > 0u) ? R.template ld<OFF_COLD + 2>() - (uint32_t)(qP >> 4) - 1u : 0u;
  const uint32_t kD = (HAS_D && R.template ld<OFF_COLD + 3>() > 0u) ? R.template ld<OFF_COLD + 3>() - (uint32_t)(qD >> 4) - 1u : 0u;
  const int jumps = (int)(kP + kD);
  snap_x = __uint_as_float(R.template ld<OFF_COLD + 0>());
  snap_w = (int)R.template ld<OFF_COLD + 1>();
  if (a.state != nullptr && valid) {  // row f2: checkpoint
    const StateIO io = state_io(a, g);
    io.put2(0, __float_as_uint(x), (uint32_t)wraps);
    io.put2(1, __float_as_uint(v), (uint32_t)jumps);
    io.put2(2, (uint32_t)nP, __float_as_uint(fP));
    io.put2(3, __float_as_uint(z), kP);
    io.put2(4, __float_as_uint(gP), __float_as_uint(gD));
    io.put2(5, (uint32_t)nD, __float_as_uint(fD));
    io.put2(6, kD, (uint32_t)d);
    io.put(7, ph);
    io.put2(8, __float_as_uint(drive0), __float_as_uint(snap_x));
    io.put2(9, (uint32_t)snap_w, 0u);
  }
  if (a.step_end < a.n_steps) return;  // not the last chunk: no outputs yet (uniform over the grid)

  Partial mine = partial_zero();
  if (valid) {
    // a10: eq. (30), assembled once per path in fp64
    fold_f32<POT>(x, wraps);
    const double Ld = Units<POT>::PERIOD_X, iS = 1.0 / (double)S;
    const double span = (double)(a.n_steps - a.n_discard) * dtd;
    const double xT = (double)wraps * Ld + (double)x * iS;
    const double xTi = (double)snap_w * Ld + (double)snap_x * iS;
    const double vbar = ((double)(wraps - snap_w) * Ld + ((double)x - (double)snap_x) * iS) / span;
    const double msub = (double)a.n_steps + (double)jumps;
    if (a.out_paths) {
      double *o = a.out_paths + g * BM_OUT_STRIDE;
      o[BM_OUT_XT] = xT; o[BM_OUT_VT] = (double)v * iS; o[BM_OUT_VBAR] = vbar; o[BM_OUT_JUMPS] = (double)jumps;
      o[BM_OUT_SUBSTEPS] = msub; o[BM_OUT_XTI] = xTi;
    }
    mine = leaf(vbar, xT, (double)jumps, msub);
  }
  block_reduce_store(mine, a.partials + (long long)blockIdx.x * PARTIAL_STRIDE);
}

}  // namespace bm
