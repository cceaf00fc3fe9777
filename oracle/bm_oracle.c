/*
 * oracle/bm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See bm_oracle.h.
 *
 * Everything is fp64, libm transcendental functions, one path at a time, in the paper's order and
 * notation.  No blocking, no fusion, no reordering beyond what DESIGN.md's readings state.
 *
 * Build: gcc -O2 -std=c11 -fopenmp -fPIC -shared -o libbm_oracle.so bm_oracle.c -lm
 *        (no -ffast-math: the oracle is the near-correctly-rounded side of every comparison)
 */
#include "bm_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* ------------------------------------------------------------------------------------------------
 * R1  Philox4x32-10.  Counter c=(c0..c3), key k=(k0,k1).  One round:
 *       (hi0,lo0) = M0*c0 ; (hi1,lo1) = M1*c2 ; c <- (hi1^c1^k0, lo1, hi0^c3^k1, lo0)
 *     ten rounds, the key bumped by (W0,W1) before rounds 2..10.
 * ---------------------------------------------------------------------------------------------- */
#define PHILOX_M0 0xD2511F53u
#define PHILOX_M1 0xCD9E8D57u
#define PHILOX_W0 0x9E3779B9u
#define PHILOX_W1 0xBB67AE85u

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += PHILOX_W0; k1 += PHILOX_W1; }
    uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
    uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R2  key = (seed mod 2^32, seed >> 32); counter = (idx, stream, g mod 2^32, g >> 32). */
enum { STREAM_INIT = 0, STREAM_GAUSS = 1, STREAM_POISSON = 2, STREAM_DICH = 3 };

void orc_philox_call(uint64_t seed, uint64_t g, uint32_t stream, uint32_t idx, uint32_t out[4]) {
  uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
  uint32_t ctr[4] = { idx, stream, (uint32_t)g, (uint32_t)(g >> 32) };
  orc_philox4x32_10(ctr, key, out);
}

/* R3  u(w) = (w + 1/2) 2^-32, exact in fp64, never 0 or 1. */
double orc_u01(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

/* R3  Box-Muller on the four words of Gaussian-stream call b:
 *       r = sqrt(-2 ln u(w0)), g[4b] = r cos(2 pi u(w1)), g[4b+1] = r sin(2 pi u(w1)),
 *       r'= sqrt(-2 ln u(w2)), g[4b+2] = r' cos(2 pi u(w3)), g[4b+3] = r' sin(2 pi u(w3)). */
void orc_gauss_block(uint64_t seed, uint64_t g, uint32_t b, double out[4]) {
  uint32_t w[4];
  orc_philox_call(seed, g, STREAM_GAUSS, b, w);
  double r = sqrt(-2.0 * log(orc_u01(w[0])));
  double a = 2.0 * M_PI * orc_u01(w[1]);
  out[0] = r * cos(a);
  out[1] = r * sin(a);
  r = sqrt(-2.0 * log(orc_u01(w[2])));
  a = 2.0 * M_PI * orc_u01(w[3]);
  out[2] = r * cos(a);
  out[3] = r * sin(a);
}

double orc_gauss(uint64_t seed, uint64_t g, uint64_t m) {
  double blk[4];
  orc_gauss_block(seed, g, (uint32_t)(m >> 2), blk);
  return blk[m & 3u];
}

/* ------------------------------------------------------------------------------------------------
 * Potentials.  SINE2: V = A1 sin(2 pi x) + A2 sin(4 pi x), period 1 (BASELINE.json configs; reading D3).
 *              PWL:   eq. (2) PAPER.md:92-95 scaled by A1, period 2: V = A1(1+x) on [-1,0), A1(1-x) on [0,1].
 *                     On the folded coordinate xi in [0,2): -V' = +A1 on [0,1), -A1 on [1,2).
 *              QUAD:  V = A1 x^2 / 2 (Ornstein-Uhlenbeck pin only; not periodic, never folded).
 * ---------------------------------------------------------------------------------------------- */
double orc_period(int potential) {
  if (potential == ORC_POT_SINE2) return 1.0;
  if (potential == ORC_POT_PWL) return 2.0;
  return 0.0;
}

double orc_minus_dV(const orc_params *p, int potential, double xi) {
  if (potential == ORC_POT_SINE2)
    return -(2.0 * M_PI * p->A1 * cos(2.0 * M_PI * xi) + 4.0 * M_PI * p->A2 * cos(4.0 * M_PI * xi));
  if (potential == ORC_POT_PWL) {
    double y = xi - 2.0 * floor(xi / 2.0); /* stage values may leave [0,2) by a little */
    return (y < 1.0) ? p->A1 : -p->A1;
  }
  return -p->A1 * xi;
}

/* R6  a(x) = -V'(x) + F - lambda*zeta + Gamma_d : the constant forces enter at all three stages
 *     (reading R6/A1; the paper-literal scheme below adds them in the corrector line only). */
static double gamma_d(const orc_params *p, int d) {
  if (d < 0) return 0.0;
  return d ? p->Fb : -p->Fa;
}

double orc_drift(const orc_params *p, int potential, double xi, int d) {
  return orc_minus_dV(p, potential, xi) + p->F - p->lambda * p->zeta + gamma_d(p, d);
}

/* Alg. 1, with a(x) of R6 and  d xi = sqrt(2 D h) g. */
double orc_substep_overdamped(const orc_params *p, int potential, int d, double x, double h, double g,
                              double stages[5]) {
  double dxi = sqrt(2.0 * p->D * h) * g;
  double F1 = orc_drift(p, potential, x, d);          /* line 1 */
  double xb = x + F1 * h + dxi;                       /* line 2 */
  double F2 = orc_drift(p, potential, xb, d);         /* line 3 */
  double xb2 = x + 0.5 * (F1 + F2) * h + dxi;         /* line 4: predictor */
  double F2c = orc_drift(p, potential, xb2, d);       /* line 5 */
  double xn = x + 0.5 * (F1 + F2c) * h + dxi;         /* line 6: corrector */
  if (stages) { stages[0] = F1; stages[1] = xb; stages[2] = F2; stages[3] = xb2; stages[4] = F2c; }
  return xn;
}

/* R7  inertial generalisation of Alg. 1 to y=(x,v):
 *       A(y,t) = ( v , -gamma v - V'(x) + amp cos(omega t) + F - lambda zeta + Gamma_d ),
 *       N = (0, sqrt(2 D h) g),  D := gamma*Q.
 *     S1: A1=A(y_n,t);      yb = y_n + A1 h + N
 *     S2: A2=A(yb ,t+h);    yb = y_n + (A1+A2) h/2 + N
 *     S3: A2=A(yb ,t+h);    y_{n+1} = y_n + (A1+A2) h/2 + N                                     */
static void inertial_A(const orc_params *p, int potential, int d, double x, double v, double t, double A[2]) {
  A[0] = v;
  A[1] = -p->gamma * v + orc_minus_dV(p, potential, x) + p->amp * cos(p->omega * t) + p->F - p->lambda * p->zeta +
         gamma_d(p, d);
}

void orc_substep_inertial(const orc_params *p, int potential, int d, double t, double h, double g, double xv[2]) {
  double x = xv[0], v = xv[1];
  double nv = sqrt(2.0 * p->D * h) * g;
  double A1[2], A2[2];
  inertial_A(p, potential, d, x, v, t, A1);
  double xb = x + A1[0] * h, vb = v + A1[1] * h + nv;
  inertial_A(p, potential, d, xb, vb, t + h, A2);
  xb = x + 0.5 * (A1[0] + A2[0]) * h;
  vb = v + 0.5 * (A1[1] + A2[1]) * h + nv;
  inertial_A(p, potential, d, xb, vb, t + h, A2);
  xv[0] = x + 0.5 * (A1[0] + A2[0]) * h;
  xv[1] = v + 0.5 * (A1[1] + A2[1]) * h + nv;
}

/* ------------------------------------------------------------------------------------------------
 * Path state shared by both schemes.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
  double xi;      /* folded coordinate in [0,L) (unfolded when L == 0) */
  int64_t wraps;  /* x = wraps*L + xi  (folding: PAPER.md:407; reading R8: also in fp64) */
  double v;
} pos_t;

/* R8  fold: xi <- x - L floor(x/L), wraps += floor(x/L). */
static void fold(pos_t *s, double L) {
  if (L <= 0.0) return;
  double k = floor(s->xi / L);
  if (k != 0.0) {
    s->xi -= k * L;
    s->wraps += (int64_t)k;
    /* guard the two rounding corners so that xi stays in [0,L) */
    if (s->xi < 0.0) { s->xi += L; s->wraps -= 1; }
    if (s->xi >= L) { s->xi -= L; s->wraps += 1; }
  }
}

static double unfolded(const pos_t *s, double L) { return (double)s->wraps * L + s->xi; }

/* R4  initial condition from init-stream call 0: x0 = L w0 2^-32 (or x0_fixed), v0 = v0_lo + (v0_hi-v0_lo) u(w1),
 *     d = 1 (state +Fb) iff u(w2) < mu_a/(mu_a+mu_b)  (stationary law of eq. 14). */
/* Rate of leaving the dichotomous state d (eq. 14).  A non-positive mu_b means that +Fb is never left (the reading
 * include/bm.h states for bm_params.mu_b and DESIGN.md section 1 repeats: "mu_b = 0 with mu_a > 0 makes +F_b absorbing"):
 * the rate is taken as 0, so the sojourn -ln(u)/0 is +infinity and the stationary weight of +Fb is 1 -- never a negative
 * waiting time. */
static double mu_leave(const orc_params *p, int d) { return d ? (p->mu_b > 0.0 ? p->mu_b : 0.0) : p->mu_a; }

static void init_path(const orc_config *cfg, const orc_params *p, uint64_t seed, uint64_t g, double L, pos_t *s,
                      int *d) {
  uint32_t w[4];
  orc_philox_call(seed, g, STREAM_INIT, 0, w);
  double L0 = (L > 0.0) ? L : 1.0;
  s->xi = (p->x0_fixed >= 0.0) ? p->x0_fixed : L0 * ((double)w[0] * (1.0 / 4294967296.0));
  s->wraps = 0;
  s->v = (cfg->model == ORC_INERTIAL) ? p->v0_lo + (p->v0_hi - p->v0_lo) * orc_u01(w[1]) : 0.0;
  fold(s, L);
  *d = (p->mu_a > 0.0) ? (orc_u01(w[2]) < p->mu_a / (p->mu_a + mu_leave(p, 1)) ? 1 : 0) : -1;
}

/* ------------------------------------------------------------------------------------------------
 * R5  Jump-adapted time loop ("variable time steps which must be adapted to each sequence
 *     of Poisson times"; reading D2).  Three countdown clocks: rem (to the next grid point), rP (to the
 *     next Poisson kick), rD (to the next dichotomous flip).  Every sub-step has length
 *     h = min(rem, rP, rD), consumes exactly one Gaussian (number m = running sub-step count) and ends
 *     on the event(s) whose clock reached zero.
 * ---------------------------------------------------------------------------------------------- */
static void path_jump_adapted(const orc_config *cfg, const orc_params *p, uint64_t g, int64_t n_steps, double dt,
                              uint64_t seed, double *out, double *trace, int64_t trace_steps) {
  const double L = orc_period(cfg->potential);
  const int has_P = p->lambda > 0.0, has_D = p->mu_a > 0.0;
  pos_t s; int d;
  init_path(cfg, p, seed, g, L, &s, &d);

  uint32_t w[4];
  uint32_t kP = 0, kD = 0;
  double rP = INFINITY, rD = INFINITY, z = 0.0;
  if (has_P) { /* call 0: w0 -> waiting time before kick 0 (eq. 27, :299-301), w1 -> its amplitude (eq. 5) */
    orc_philox_call(seed, g, STREAM_POISSON, kP, w);
    rP = -log(orc_u01(w[0])) / p->lambda;
    z = -p->zeta * log(orc_u01(w[1]));
  }
  if (has_D) { /* call 0: w0 -> residual duration of the initial sojourn (eq. 28, :347; memoryless) */
    orc_philox_call(seed, g, STREAM_DICH, kD, w);
    rD = -log(orc_u01(w[0])) / mu_leave(p, d);
  }

  int64_t n = 0; uint64_t m = 0; double rem = dt; double jumps = 0.0;
  double gblk[4] = {0, 0, 0, 0};
  pos_t snap = s;
  while (n < n_steps) {
    double h = rem;
    if (has_P && rP < h) h = rP;
    if (has_D && rD < h) h = rD;
    double t = (double)n * dt + (dt - rem);
    if ((m & 3u) == 0) orc_gauss_block(seed, g, (uint32_t)(m >> 2), gblk);
    double gn = gblk[m & 3u];
    m++;
    if (cfg->model == ORC_OVERDAMPED) {
      s.xi = orc_substep_overdamped(p, cfg->potential, d, s.xi, h, gn, NULL);
    } else {
      double xv[2] = { s.xi, s.v };
      orc_substep_inertial(p, cfg->potential, d, t, h, gn, xv);
      s.xi = xv[0]; s.v = xv[1];
    }
    rem -= h;
    if (has_P) rP -= h;
    if (has_D) rD -= h;
    if (has_P && rP <= 0.0) { /* kick kP: jump z in x (eq. 3, :103; :301), in v for the inertial model (R7) */
      if (cfg->model == ORC_OVERDAMPED) s.xi += z; else s.v += z;
      jumps += 1.0; kP++;
      orc_philox_call(seed, g, STREAM_POISSON, kP, w);
      rP = -log(orc_u01(w[0])) / p->lambda;
      z = -p->zeta * log(orc_u01(w[1]));
    }
    if (has_D && rD <= 0.0) { /* flip (eq. 13-14, :151-157); next sojourn ~ Exp(rate of leaving the new state) */
      d = 1 - d;
      jumps += 1.0; kD++;
      orc_philox_call(seed, g, STREAM_DICH, kD, w);
      rD = -log(orc_u01(w[0])) / mu_leave(p, d);
    }
    fold(&s, L);
    if (rem <= 0.0) {
      n++; rem = dt;
      if (trace && n <= trace_steps) { trace[2 * (n - 1)] = unfolded(&s, L); trace[2 * (n - 1) + 1] = s.v; }
      if (n == cfg->n_discard) snap = s;
    }
  }
  double Leff = (L > 0.0) ? L : 0.0;
  double span = (double)(n_steps - cfg->n_discard) * dt;
  out[ORC_OUT_XT] = unfolded(&s, L);
  out[ORC_OUT_VT] = s.v;
  /* eq. (30): (x(t_f) - x(t_i)) / (t_f - t_i), differences taken on (wraps, xi) separately */
  out[ORC_OUT_VBAR] = ((double)(s.wraps - snap.wraps) * Leff + (s.xi - snap.xi)) / span;
  out[ORC_OUT_JUMPS] = jumps;
  out[ORC_OUT_SUBSTEPS] = (double)m;
  out[ORC_OUT_XTI] = unfolded(&snap, L);
}

/* ------------------------------------------------------------------------------------------------
 * Paper-literal scheme (NEXT row f1): constant step dt, Alg. 2 three-point increment (:239-259, eq. 25),
 * Alg. 3 grid-quantised Poisson countdown (:270-291), Alg. 4 dichotomous countdown (:305-343), and Alg. 1
 * exactly as printed: increments d eta, d Gamma enter line 6 only (:234).  Over-damped only.
 * Readings: [.] in Alg. 3/4 is floor (A2); first countdowns drawn before step 0 (A3); uniform number n
 * of the Gaussian stream is word n%4 of call n/4; Poisson call k: w0 -> countdown before kick k, w1 ->
 * amplitude of kick k; dichotomous call k: w0 -> countdown of sojourn k.
 * ---------------------------------------------------------------------------------------------- */
static double exp_variate_literal(uint32_t w, double scale) { return -scale * log(1.0 - orc_u01(w)); } /* -ln(1-phi) */

static void path_paper_literal(const orc_config *cfg, const orc_params *p, uint64_t g, int64_t n_steps, double dt,
                               uint64_t seed, double *out, double *trace, int64_t trace_steps) {
  const double L = orc_period(cfg->potential);
  const int has_P = p->lambda > 0.0, has_D = p->mu_a > 0.0;
  pos_t s; int d;
  init_path(cfg, p, seed, g, L, &s, &d);
  uint32_t w[4], wg[4] = {0, 0, 0, 0};
  uint32_t kP = 0, kD = 0;
  double sP = 0.0, sD = 0.0, z = 0.0, jumps = 0.0;
  if (has_P) {
    orc_philox_call(seed, g, STREAM_POISSON, kP, w);
    sP = floor(exp_variate_literal(w[0], 1.0 / p->lambda) / dt);   /* Alg. 3 line 5 */
    z = exp_variate_literal(w[1], p->zeta);                        /* Alg. 3 line 7 */
  }
  if (has_D) {
    orc_philox_call(seed, g, STREAM_DICH, kD, w);
    sD = floor(exp_variate_literal(w[0], 1.0 / mu_leave(p, d)) / dt);
  }
  const double G = sqrt(2.0 * p->D);                               /* Alg. 2 line 1 */
  const double a = p->lambda * p->zeta;                            /* eq. (6); Alg. 3 line 1: sqrt(lambda D_P) */
  pos_t snap = s;
  for (int64_t n = 0; n < n_steps; ++n) {
    /* Alg. 2 */
    if ((n & 3) == 0) orc_philox_call(seed, g, STREAM_GAUSS, (uint32_t)(n >> 2), wg);
    double phi = orc_u01(wg[n & 3]);
    double dxi;
    if (phi <= 1.0 / 6.0) dxi = -G * sqrt(3.0 * dt);
    else if (phi > 1.0 / 6.0 && phi <= 1.0 / 3.0) dxi = G * sqrt(3.0 * dt);
    else dxi = 0.0;
    /* Alg. 3 */
    double deta = 0.0;
    if (has_P) {
      if (sP <= 0.0) {
        deta = z - a * dt;
        jumps += 1.0; kP++;
        orc_philox_call(seed, g, STREAM_POISSON, kP, w);
        sP = floor(exp_variate_literal(w[0], 1.0 / p->lambda) / dt);
        z = exp_variate_literal(w[1], p->zeta);
      } else {
        sP -= 1.0;
        deta = -a * dt;
      }
    }
    /* Alg. 4 */
    double dGam = 0.0;
    if (has_D) {
      if (sD <= 0.0) {
        d = 1 - d;
        jumps += 1.0; kD++;
        orc_philox_call(seed, g, STREAM_DICH, kD, w);
        sD = floor(exp_variate_literal(w[0], 1.0 / mu_leave(p, d)) / dt);
      } else {
        sD -= 1.0;
      }
      dGam = (d ? p->Fb : -p->Fa) * dt;
    }
    /* Alg. 1 as printed; the static load F (not in the paper) rides with -V' */
    double x = s.xi;
    double F1 = orc_minus_dV(p, cfg->potential, x) + p->F;
    double xb = x + F1 * dt + dxi;
    double F2 = orc_minus_dV(p, cfg->potential, xb) + p->F;
    xb = x + 0.5 * (F1 + F2) * dt + dxi;
    F2 = orc_minus_dV(p, cfg->potential, xb) + p->F;
    s.xi = x + 0.5 * (F1 + F2) * dt + dxi + deta + dGam;
    fold(&s, L);
    if (trace && n + 1 <= trace_steps) { trace[2 * n] = unfolded(&s, L); trace[2 * n + 1] = 0.0; }
    if (n + 1 == cfg->n_discard) snap = s;
  }
  double span = (double)(n_steps - cfg->n_discard) * dt;
  out[ORC_OUT_XT] = unfolded(&s, L);
  out[ORC_OUT_VT] = 0.0;
  out[ORC_OUT_VBAR] = ((double)(s.wraps - snap.wraps) * L + (s.xi - snap.xi)) / span;
  out[ORC_OUT_JUMPS] = jumps;
  out[ORC_OUT_SUBSTEPS] = (double)n_steps;
  out[ORC_OUT_XTI] = unfolded(&snap, L);
}

/* ------------------------------------------------------------------------------------------------
 * Dynamic step size control from chi (NEXT row f4).  PAPER.md:237: "The difference chi = xbar_{n+1} - x_{n+1} between
 * these values provides information about the local approximation error.  This quantity can be utilized to introduce a
 * dynamic time step size control".  The paper gives no controller; reading R14:
 *   - a grid step dt is covered by intervals of length dt 2^-k, k = 0..K (K = adapt_levels), each aligned to a multiple
 *     of its own length, so every grid point n dt is hit exactly and t_i, t_f, the trace stay where they were;
 *   - an interval is integrated as in the jump-adapted scheme (sub-steps end on the kicks and flips inside it; one
 *     Gaussian, number m = running sub-step count, per sub-step); chi of a sub-step is Alg. 1's predictor (line 4)
 *     minus its corrector (line 6);
 *   - no step is ever rejected (its noise has been drawn; redoing it with a finer step would need a Brownian bridge
 *     to keep the law): the largest |chi| of an interval sets the length of the NEXT one: halve (k+1) if it
 *     exceeds tol, double (k-1) if it is below tol/8 and the next interval would still be aligned, else keep.
 * Every path starts at k = 0.  tol = +inf reproduces the jump-adapted scheme; tol = 0 the same scheme at dt 2^-K.
 * Over-damped only (Alg. 1 is the over-damped scheme).
 * ---------------------------------------------------------------------------------------------- */
static void path_adaptive(const orc_config *cfg, const orc_params *p, uint64_t g, int64_t n_steps, double dt,
                          uint64_t seed, double *out, double *trace, int64_t trace_steps) {
  const double L = orc_period(cfg->potential);
  const int has_P = p->lambda > 0.0, has_D = p->mu_a > 0.0;
  const int K = cfg->adapt_levels;
  const int64_t TPC = (int64_t)1 << K; /* ticks per grid step */
  pos_t s; int d;
  init_path(cfg, p, seed, g, L, &s, &d);
  uint32_t w[4];
  uint32_t kP = 0, kD = 0;
  double rP = INFINITY, rD = INFINITY, z = 0.0;
  if (has_P) {
    orc_philox_call(seed, g, STREAM_POISSON, kP, w);
    rP = -log(orc_u01(w[0])) / p->lambda;
    z = -p->zeta * log(orc_u01(w[1]));
  }
  if (has_D) {
    orc_philox_call(seed, g, STREAM_DICH, kD, w);
    rD = -log(orc_u01(w[0])) / mu_leave(p, d);
  }
  uint64_t m = 0; double jumps = 0.0;
  double gblk[4] = {0, 0, 0, 0};
  pos_t snap = s;
  int k = 0;
  for (int64_t n = 0; n < n_steps; ++n) {
    int64_t tick = 0;
    while (tick < TPC) {
      const int64_t wd = TPC >> k;           /* interval width in ticks */
      const double H = ldexp(dt, -k);        /* its length, exactly dt 2^-k */
      double rem = H, chi_max = 0.0;
      while (rem > 0.0) {
        double h = rem;
        if (has_P && rP < h) h = rP;
        if (has_D && rD < h) h = rD;
        if ((m & 3u) == 0) orc_gauss_block(seed, g, (uint32_t)(m >> 2), gblk);
        double gn = gblk[m & 3u];
        m++;
        double st[5];
        double xn = orc_substep_overdamped(p, cfg->potential, d, s.xi, h, gn, st);
        double chi = fabs(st[3] - xn);       /* predictor (line 4) minus corrector (line 6) */
        if (chi > chi_max) chi_max = chi;
        s.xi = xn;
        rem -= h;
        if (has_P) rP -= h;
        if (has_D) rD -= h;
        if (has_P && rP <= 0.0) {
          s.xi += z;
          jumps += 1.0; kP++;
          orc_philox_call(seed, g, STREAM_POISSON, kP, w);
          rP = -log(orc_u01(w[0])) / p->lambda;
          z = -p->zeta * log(orc_u01(w[1]));
        }
        if (has_D && rD <= 0.0) {
          d = 1 - d;
          jumps += 1.0; kD++;
          orc_philox_call(seed, g, STREAM_DICH, kD, w);
          rD = -log(orc_u01(w[0])) / mu_leave(p, d);
        }
        fold(&s, L);
      }
      tick += wd;
      if (chi_max > cfg->adapt_tol && k < K) k += 1;
      else if (chi_max < 0.125 * cfg->adapt_tol && k > 0 && (tick % (2 * wd)) == 0) k -= 1;
    }
    if (trace && n + 1 <= trace_steps) { trace[2 * n] = unfolded(&s, L); trace[2 * n + 1] = 0.0; }
    if (n + 1 == cfg->n_discard) snap = s;
  }
  double span = (double)(n_steps - cfg->n_discard) * dt;
  out[ORC_OUT_XT] = unfolded(&s, L);
  out[ORC_OUT_VT] = 0.0;
  out[ORC_OUT_VBAR] = ((double)(s.wraps - snap.wraps) * L + (s.xi - snap.xi)) / span;
  out[ORC_OUT_JUMPS] = jumps;
  out[ORC_OUT_SUBSTEPS] = (double)m;
  out[ORC_OUT_XTI] = unfolded(&snap, L);
}

/* ------------------------------------------------------------------------------------------------ */
static int g_threads_used = 1;
int orc_threads_used(void) { return g_threads_used; }

int orc_simulate(const orc_config *cfg, const orc_params *params, int32_t n_points, int64_t n_paths,
                 int64_t n_steps, double dt, uint64_t seed, const int64_t *ids, int64_t n_ids,
                 double *out_paths, double *trace, int64_t trace_paths, int64_t trace_steps, int32_t threads) {
  if (!cfg || !params || !out_paths || n_points <= 0 || n_paths <= 0 || n_steps <= 0 || !(dt > 0.0)) return -1;
  if (cfg->n_discard < 0 || cfg->n_discard >= n_steps) return -1;
  if (cfg->scheme == ORC_SCHEME_PAPER_LITERAL && cfg->model != ORC_OVERDAMPED) return -2;
  if (cfg->scheme == ORC_SCHEME_ADAPTIVE && cfg->model != ORC_OVERDAMPED) return -2;
  if (cfg->scheme == ORC_SCHEME_ADAPTIVE && (cfg->adapt_levels < 0 || cfg->adapt_levels > 20 || !(cfg->adapt_tol >= 0.0))) return -1;
  if (cfg->potential < 0 || cfg->potential > ORC_POT_QUAD) return -1;
  int64_t total = ids ? n_ids : (int64_t)n_points * n_paths;
  if (total <= 0) return -1;
  for (int64_t i = 0; ids && i < total; ++i)
    if (ids[i] < 0 || ids[i] >= (int64_t)n_points * n_paths) return -1;
#ifdef _OPENMP
  int nt = threads > 0 ? threads : omp_get_max_threads();
  if ((int64_t)nt > total) nt = (int)total;
  g_threads_used = nt;
#else
  int nt = 1; (void)threads;
  g_threads_used = 1;
#endif
  /* each path is independent: any split over threads gives the same numbers */
#pragma omp parallel for schedule(dynamic, 4) num_threads(nt)
  for (int64_t i = 0; i < total; ++i) {
    uint64_t g = (uint64_t)(ids ? ids[i] : i);
    const orc_params *p = &params[g / (uint64_t)n_paths];
    double *tr = (trace && i < trace_paths) ? trace + i * trace_steps * 2 : NULL;
    if (cfg->scheme == ORC_SCHEME_PAPER_LITERAL)
      path_paper_literal(cfg, p, g, n_steps, dt, seed, out_paths + i * ORC_OUT_STRIDE, tr, trace_steps);
    else if (cfg->scheme == ORC_SCHEME_ADAPTIVE)
      path_adaptive(cfg, p, g, n_steps, dt, seed, out_paths + i * ORC_OUT_STRIDE, tr, trace_steps);
    else
      path_jump_adapted(cfg, p, g, n_steps, dt, seed, out_paths + i * ORC_OUT_STRIDE, tr, trace_steps);
  }
  return 0;
}

/* R9  ensemble statistics: two passes in index order (mean; then unbiased variance). */
void orc_reduce(const double *out_paths, int64_t n, orc_stats *st) {
  memset(st, 0, sizeof(*st));
  if (n <= 0) return;
  double sv = 0, sx = 0, sj = 0, ss = 0;
  for (int64_t i = 0; i < n; ++i) {
    const double *r = out_paths + i * ORC_OUT_STRIDE;
    sv += r[ORC_OUT_VBAR]; sx += r[ORC_OUT_XT]; sj += r[ORC_OUT_JUMPS]; ss += r[ORC_OUT_SUBSTEPS];
  }
  double mv = sv / (double)n, mx = sx / (double)n;
  double qv = 0, qx = 0;
  for (int64_t i = 0; i < n; ++i) {
    const double *r = out_paths + i * ORC_OUT_STRIDE;
    qv += (r[ORC_OUT_VBAR] - mv) * (r[ORC_OUT_VBAR] - mv);
    qx += (r[ORC_OUT_XT] - mx) * (r[ORC_OUT_XT] - mx);
  }
  st->n = (double)n;
  st->mean_v = mv; st->mean_xT = mx;
  st->var_v = (n > 1) ? qv / (double)(n - 1) : 0.0;
  st->var_xT = (n > 1) ? qx / (double)(n - 1) : 0.0;
  st->mean_jumps = sj / (double)n;
  st->mean_substeps = ss / (double)n;
}
