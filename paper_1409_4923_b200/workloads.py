"""Seeded synthetic workloads C0..C4 of BASELINE.json.

This module holds NONE of the method's arithmetic: it only builds parameter tables (plain float64 arrays in
the 16-column layout of `bm_params`, include/bm.h) and run sizes.  It is the one module that serves both the
CUDA path and the oracle's tests; it imports neither.

The paper uses no dataset: every workload is generated from parameters (PAPER.md:418-425 for its own runs).
"""
import math
from dataclasses import dataclass, field

import numpy as np

SEED = 14094923

# column order of bm_params (include/bm.h) == OrcParams (oracle/bm_oracle.h)
FIELDS = ("A1", "A2", "F", "D", "lambda", "zeta", "Fa", "Fb", "mu_a", "mu_b", "gamma", "amp", "omega",
          "x0_fixed", "v0_lo", "v0_hi")
COL = {n: i for i, n in enumerate(FIELDS)}

OVERDAMPED, INERTIAL = 0, 1
POT_SINE2, POT_PWL, POT_QUAD = 0, 1, 2
SCHEME_JUMP_ADAPTED, SCHEME_PAPER_LITERAL, SCHEME_ADAPTIVE = 0, 1, 2


def params_table(n_points=1, **kw):
    """(n_points,16) float64 table; each keyword is a scalar or a length-n_points array."""
    t = np.zeros((n_points, 16), dtype=np.float64)
    t[:, COL["x0_fixed"]] = -1.0
    for k, v in kw.items():
        k = "lambda" if k == "lambda_" else k
        t[:, COL[k]] = v
    return t


@dataclass
class Workload:
    name: str
    model: int
    params: np.ndarray          # (n_points,16)
    n_paths: int                # per point
    n_steps: int
    dt: float
    n_discard: int
    potential: int = POT_SINE2
    scheme: int = SCHEME_JUMP_ADAPTED
    seed: int = SEED
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def n_points(self):
        return self.params.shape[0]

    @property
    def path_steps(self):
        return self.n_points * self.n_paths * self.n_steps

    def scaled(self, n_paths=None, n_steps=None, n_discard=None, points=None):
        """Same physics at a reduced size (parity-test cases)."""
        p = self.params if points is None else np.ascontiguousarray(self.params[points])
        ns = self.n_steps if n_steps is None else n_steps
        nd = n_discard if n_discard is not None else (self.n_discard * ns) // self.n_steps
        return Workload(self.name + "-scaled", self.model, p, n_paths or self.n_paths, ns, self.dt, nd,
                        self.potential, self.scheme, self.seed, self.note, dict(self.extra))


DT_INERTIAL = (2.0 * math.pi / 4.9) / 400.0


def c0():
    """Overdamped Gaussian ratchet, 1024 paths x 1e4 steps, <v> over the 2nd half (BASELINE.json configs[0])."""
    return Workload("C0", OVERDAMPED, params_table(1, A1=1.0, A2=0.25, F=0.1, D=0.05), 1024, 10_000, 1e-3, 5_000)


def c1():
    """Overdamped ratchet + white Poissonian noise, 65536 paths x 1e5 steps (configs[1]); 10 % discarded (:423)."""
    return Workload("C1", OVERDAMPED, params_table(1, A1=1.0, A2=0.25, F=0.0, D=0.01, lambda_=2.0, zeta=0.3),
                    65_536, 100_000, 1e-3, 10_000)


def _inertial_point(n_points, f):
    g, Q = 0.9, 1e-3
    return params_table(n_points, A1=1.0, A2=0.0, F=f, D=g * Q, Fa=0.5, Fb=0.5, mu_a=1.0, mu_b=1.0, gamma=g,
                        amp=4.2, omega=4.9, v0_lo=-2.0, v0_hi=2.0)


def c2():
    """Inertial motor, dichotomous noise, 65536 paths x 500 periods x 400 steps (configs[2]); 10 % discarded."""
    return Workload("C2", INERTIAL, _inertial_point(1, 0.1), 65_536, 500 * 400, DT_INERTIAL, 50 * 400)


def c3():
    """Inertial dichotomous sweep, f over linspace(-0.5,0.5,256) x 1024 paths, 2000 periods, 500 discarded."""
    return Workload("C3", INERTIAL, _inertial_point(256, np.linspace(-0.5, 0.5, 256)), 1024, 2000 * 400,
                    DT_INERTIAL, 500 * 400)


def c4():
    """Poisson 2-D sweep: lambda over logspace(-1,2,128) x zeta over linspace(0.05,1,128), 4096 paths/point."""
    lam = np.logspace(-1.0, 2.0, 128)
    zet = np.linspace(0.05, 1.0, 128)
    L, Z = np.meshgrid(lam, zet, indexing="ij")     # point = i*128 + j
    return Workload("C4", OVERDAMPED, params_table(128 * 128, A1=1.0, A2=0.25, F=0.0, D=0.01,
                                                   lambda_=L.ravel(), zeta=Z.ravel()),
                    4096, 20_000, 1e-3, 2_000)


def m1():
    """The paper's own benchmark program `poisson` (Model I): piece-wise linear potential,
    white Poissonian noise a = 1.5, D_P = 1, D_G = 0, scheme as printed (Alg. 1-4), spp = 400; N = 131072 paths (the
    paper's speed-up saturates "around N = 1e5"), 4e4 steps = 100 characteristic times.  Context, not a BASELINE config."""
    a, DP = 1.5, 1.0
    zeta, lam = DP / a, a * a / DP
    return Workload("M1", OVERDAMPED, params_table(1, A1=1.0, D=0.0, lambda_=lam, zeta=zeta), 131_072, 40_000,
                    (1 / lam) / 400, 4_000, potential=POT_PWL, scheme=SCHEME_PAPER_LITERAL)


def m2():
    """The paper's program `dich` (Model II): dichotomous noise F_a = 3, F_b = 1.6, tau = 0.3, spp = 200."""
    Fa, Fb, tau = 3.0, 1.6, 0.3
    mu_a, mu_b = Fa / (tau * (Fa + Fb)), Fb / (tau * (Fa + Fb))
    return Workload("M2", OVERDAMPED, params_table(1, A1=1.0, D=0.0, Fa=Fa, Fb=Fb, mu_a=mu_a, mu_b=mu_b), 131_072,
                    40_000, min(1 / mu_a, 1 / mu_b) / 200, 4_000, potential=POT_PWL, scheme=SCHEME_PAPER_LITERAL)


def a1():
    """Dynamic step size control from chi on C1's physics: 65536 paths x 2e4 grid
    steps of 1e-3, each halved up to 4 times where |chi| exceeds 1e-5.  A bench case (fp64 only), not a BASELINE config."""
    w = c1()
    return Workload("A1", OVERDAMPED, w.params, w.n_paths, 20_000, w.dt, 2_000, scheme=SCHEME_ADAPTIVE,
                    extra=dict(adapt_tol=1e-5, adapt_levels=4))


CONFIGS = {"C0": c0, "C1": c1, "C2": c2, "C3": c3, "C4": c4, "M1": m1, "M2": m2, "A1": a1}
