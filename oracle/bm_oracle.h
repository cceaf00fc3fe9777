/*
 * oracle/bm_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle for the hot path of arXiv 1409.4923 (Spiechowicz, Kostur,
 * Machura): ensemble Monte Carlo integration of Brownian-motor Langevin equations with the
 * jump-adapted weak-order-2.0 predictor-corrector scheme.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may use it.  It shares no code with the
 * CUDA path (own Philox, own Box-Muller, own stepper, own struct declarations).
 *
 * Citations are PAPER.md:<line> (+ equation / algorithm) or DESIGN.md reading Rn where the
 * paper is silent.  See DESIGN.md section 3 for the readings.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): ATen's philox_engine (library routine), OU closed
 * form of the scheme, weak order 2 on OU, free motion, Poisson cumulants, dichotomous
 * autocovariance, jump-adaptation invariance, Stratonovich formula, equipartition, eq. (21)-(23).
 * Full-length ensemble values on configs C0..C4 themselves: PARITY UNPINNED by the paper (it prints
 * no numbers for them); they are pinned only through the closed forms above.
 */
#ifndef BM_ORACLE_H
#define BM_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* One parameter point.  16 doubles.  (Declared independently of include/bm.h on purpose.) */
typedef struct {
  double A1, A2;        /* SINE2: V(x)=A1 sin(2 pi x)+A2 sin(4 pi x), L=1.  PWL: A1 scales eq.(2). QUAD: V=A1 x^2/2 */
  double F;             /* static load */
  double D;             /* Gaussian intensity: overdamped sqrt(2D) dW (eq. 9-10); inertial D := gamma*Q */
  double lambda, zeta;  /* Poisson rate (eq. 4) and mean amplitude (eq. 5); bias -lambda*zeta (eq. 3, 6) */
  double Fa, Fb;        /* dichotomous states -Fa, +Fb (eq. 13) */
  double mu_a, mu_b;    /* rates of leaving -Fa, +Fb (eq. 14) */
  double gamma, amp, omega; /* inertial: friction, drive amplitude, drive angular frequency */
  double x0_fixed;      /* >= 0: x0 = x0_fixed; < 0: x0 ~ U[0,L) */
  double v0_lo, v0_hi;  /* inertial: v0 ~ U[v0_lo, v0_hi] */
} orc_params;

enum { ORC_OVERDAMPED = 0, ORC_INERTIAL = 1 };
enum { ORC_POT_SINE2 = 0, ORC_POT_PWL = 1, ORC_POT_QUAD = 2 };
enum { ORC_SCHEME_JUMP_ADAPTED = 0, ORC_SCHEME_PAPER_LITERAL = 1, ORC_SCHEME_ADAPTIVE = 2 };

typedef struct {
  int32_t model;      /* ORC_OVERDAMPED / ORC_INERTIAL */
  int32_t potential;  /* ORC_POT_* */
  int32_t scheme;     /* ORC_SCHEME_* */
  int32_t reserved;
  int64_t n_discard;  /* grid steps before t_i (eq. 30) */
  /* ORC_SCHEME_ADAPTIVE only (reading R14): tolerance on |chi| = |xbar_{n+1} - x_{n+1}| and the number
   * of times the step dt may be halved */
  double adapt_tol;
  int32_t adapt_levels;
  int32_t reserved2;
} orc_config;

/* per-path record: 6 doubles */
enum { ORC_OUT_XT = 0, ORC_OUT_VT = 1, ORC_OUT_VBAR = 2, ORC_OUT_JUMPS = 3, ORC_OUT_SUBSTEPS = 4, ORC_OUT_XTI = 5,
       ORC_OUT_STRIDE = 6 };

typedef struct { double n, mean_v, var_v, mean_xT, var_xT, mean_jumps, mean_substeps, rsv; } orc_stats;

/* R1: Philox4x32-10 (Salmon et al. SC'11). ctr[4], key[2] -> out[4]. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* R2: the keyed call used by the method: key=(seed lo,hi), ctr=(idx, stream, g lo, g hi). */
void orc_philox_call(uint64_t seed, uint64_t g, uint32_t stream, uint32_t idx, uint32_t out[4]);
/* R3: u(w) = (w+0.5) 2^-32 in (0,1). */
double orc_u01(uint32_t w);
/* R3: Box-Muller block b of path g: 4 standard normals (Gaussian numbers 4b..4b+3). */
void orc_gauss_block(uint64_t seed, uint64_t g, uint32_t b, double out[4]);
/* Gaussian number m of path g (block m/4, component m%4). */
double orc_gauss(uint64_t seed, uint64_t g, uint64_t m);

/* Static drift a(x) of R6 for dichotomous state d (d<0: no dichotomous term). */
double orc_drift(const orc_params *p, int potential, double xi, int d);
/* -V'(x) only. */
double orc_minus_dV(const orc_params *p, int potential, double xi);
/* period L of the potential (0 for QUAD = no folding) */
double orc_period(int potential);

/* Alg. 1 as read in R6: one overdamped sub-step of length h with injected
 * standard normal g.  stages[5] = {F1, xbar1, F2, xbar2, F2'} (may be NULL).  Returns x_{n+1} (unfolded:
 * x is the folded coordinate, result may leave [0,L)). */
double orc_substep_overdamped(const orc_params *p, int potential, int d, double x, double h, double g,
                              double stages[5]);
/* R7: one inertial sub-step from time t; xv[2] in/out. */
void orc_substep_inertial(const orc_params *p, int potential, int d, double t, double h, double g, double xv[2]);

/* Simulate the listed global path ids (g = point*n_paths + p).  ids == NULL: all n_points*n_paths paths,
 * n_ids ignored.  out_paths[n][ORC_OUT_STRIDE].  trace (optional): for the first trace_paths listed
 * ids, (x unfolded, v) after each of the first trace_steps grid steps: [trace_paths][trace_steps][2].
 * threads <= 0: all cores (OpenMP).  Returns 0, or <0 on invalid arguments. */
int orc_simulate(const orc_config *cfg, const orc_params *params, int32_t n_points, int64_t n_paths,
                 int64_t n_steps, double dt, uint64_t seed, const int64_t *ids, int64_t n_ids,
                 double *out_paths, double *trace, int64_t trace_paths, int64_t trace_steps, int32_t threads);

/* R9: two-pass mean / unbiased variance in index order over n records of out_paths. */
void orc_reduce(const double *out_paths, int64_t n, orc_stats *st);

int orc_threads_used(void);

#ifdef __cplusplus
}
#endif
#endif
