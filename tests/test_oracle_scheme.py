"""Pins for the oracle's predictor-corrector stepper (R6, R7; Alg. 1).  CPU only.

P2  single sub-steps recomputed in 50-digit arithmetic; D=0 reduces to the Heun-then-trapezoid iteration.
P3  Ornstein-Uhlenbeck closed form of the 3-stage scheme itself: x' = R x + S dxi,
        R = 1 - z + z^2/2 - z^3/4,  S = 1 - z/2 + z^2/4,  z = theta h
    (plain Heun would give R = 1 - z + z^2/2, S = 1 - z/2: the cubic term tells the third stage is there).
P4  weak order 2: |x0 R^n - x0 exp(-theta T)| falls by 4 per halving of dt.
P11 inertial: linear damped driven ODE closed form, order 2; OU closed form of the (x,v) map.
"""
import math

import mpmath as mp
import numpy as np
import pytest

from paper_1409_4923_b200.workloads import SEED


def _golden_rows(name):
    import os
    rows = []
    with open(os.path.join(os.path.dirname(__file__), "golden", name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append([float(t) for t in line.split()])
    return rows


def test_p2_worked_steps_golden(orc):
    """tests/golden/worked_substeps.txt: Alg. 1 stage values worked out by hand in 50-digit arithmetic."""
    for A1, A2, F, D, lam, zeta, x, h, g, F1, xb1, F2, xb2, F2c, xn in _golden_rows("worked_substeps.txt"):
        p = orc.make_params(A1=A1, A2=A2, F=F, D=D, lambda_=lam, zeta=zeta)
        got_xn, st = orc.substep_overdamped(p, orc.POT_SINE2, -1, x, h, g)
        for a, e in zip(st + (got_xn,), (F1, xb1, F2, xb2, F2c, xn)):
            assert abs(a - e) <= 2e-14 * max(1.0, abs(e))


def test_p2_deterministic_reduces_to_heun_trapezoid(orc):
    """D=0: x1 = x + h f(x); x2 = x + h/2 (f(x)+f(x1)); x' = x + h/2 (f(x)+f(x2)), f = -V'+F, in mpmath."""
    mp.mp.dps = 40
    A1, A2, F = 0.7, -0.3, 0.2

    def f(x):
        return -(2 * mp.pi * A1 * mp.cos(2 * mp.pi * x) + 4 * mp.pi * A2 * mp.cos(4 * mp.pi * x)) + F
    p = orc.make_params(A1=A1, A2=A2, F=F, D=0.0)
    for x0, h in ((0.1, 1e-3), (0.73, 5e-3), (0.4999, 2e-2)):
        x = mp.mpf(x0); hh = mp.mpf(h)
        x1 = x + hh * f(x)
        x2 = x + hh / 2 * (f(x) + f(x1))
        x3 = x + hh / 2 * (f(x) + f(x2))
        got, _ = orc.substep_overdamped(p, orc.POT_SINE2, -1, x0, h, 1.2345)   # g irrelevant at D=0
        assert abs(got - float(x3)) < 1e-15


def test_p3_ou_single_step_linear_map(orc):
    theta, D = 2.0, 0.3
    p = orc.make_params(A1=theta, D=D, x0_fixed=0.0)
    for h in (0.04, 0.01, 0.25):
        z = theta * h
        R = 1 - z + z * z / 2 - z ** 3 / 4
        S = 1 - z / 2 + z * z / 4
        for x, g in ((1.0, 0.0), (0.0, 1.0), (-0.7, 0.9), (2.5, -1.3)):
            got, _ = orc.substep_overdamped(p, orc.POT_QUAD, -1, x, h, g)
            assert abs(got - (R * x + S * math.sqrt(2 * D * h) * g)) < 1e-14
    # W3 of SURVEY.md section 8(c): z = 0.08 -> R = 0.923072, S = 0.9616 exactly
    z = 0.08
    assert abs((1 - z + z * z / 2 - z ** 3 / 4) - 0.923072) < 1e-15 and abs((1 - z / 2 + z * z / 4) - 0.9616) < 1e-15


def test_p3_p4_ou_deterministic_decay_and_order_two(orc):
    theta, x0, T = 1.5, 2.0, 2.0
    errs = []
    for n in (50, 100, 200, 400):
        h = T / n
        p = orc.params_array([dict(A1=theta, D=0.0, x0_fixed=x0)])
        out, _ = orc.simulate(p, 1, n, h, SEED, potential=orc.POT_QUAD)
        z = theta * h
        R = 1 - z + z * z / 2 - z ** 3 / 4
        assert abs(out[0, orc.OUT_XT] - x0 * R ** n) < 1e-13
        errs.append(abs(out[0, orc.OUT_XT] - x0 * math.exp(-theta * T)))
    ratios = [errs[i] / errs[i + 1] for i in range(3)]
    for r in ratios:
        assert 3.7 < r < 4.3, ratios
    # leading error term x0 e^{-theta T} T theta^3 h^2 / 12
    h = T / 400
    assert abs(errs[-1] / (x0 * math.exp(-theta * T) * T * theta ** 3 * h * h / 12) - 1) < 0.05


def test_p3_p4_ou_moments_monte_carlo(orc):
    """E[x_n] = x0 R^n, Var_n = 2 D h S^2 (1-R^{2n})/(1-R^2); the scheme's variance converges at order 2."""
    theta, D, x0, T, N = 1.0, 0.5, 1.5, 1.0, 20000
    n = 20
    h = T / n
    p = orc.params_array([dict(A1=theta, D=D, x0_fixed=x0)])
    out, _ = orc.simulate(p, N, n, h, SEED, potential=orc.POT_QUAD)
    x = out[:, orc.OUT_XT]
    z = theta * h
    R = 1 - z + z * z / 2 - z ** 3 / 4
    S = 1 - z / 2 + z * z / 4
    var_n = 2 * D * h * S * S * (1 - R ** (2 * n)) / (1 - R * R)
    assert abs(x.mean() - x0 * R ** n) < 4 * math.sqrt(var_n / N)
    assert abs(x.var(ddof=1) - var_n) < 4 * var_n * math.sqrt(2 / (N - 1))
    # Gaussian increments -> x_n exactly Gaussian: kurtosis 3
    k = ((x - x.mean()) ** 4).mean() / x.var() ** 2
    assert abs(k - 3) < 4 * math.sqrt(24 / N)
    # closed-form variance of the scheme vs exact OU variance: order 2 in h
    exact = D / theta * (1 - math.exp(-2 * theta * T))
    e = []
    for nn in (80, 160, 320):
        hh = T / nn
        zz = theta * hh
        RR = 1 - zz + zz * zz / 2 - zz ** 3 / 4
        SS = 1 - zz / 2 + zz * zz / 4
        e.append(abs(2 * D * hh * SS * SS * (1 - RR ** (2 * nn)) / (1 - RR * RR) - exact))
    assert 3.6 < e[0] / e[1] < 4.4 and 3.6 < e[1] / e[2] < 4.4


def test_p11_inertial_linear_ode_closed_form(orc):
    """V=0, D=0: x'' + gamma x' = amp cos(omega t) + F has an elementary solution; scheme error ~ h^2."""
    gam, amp, om, F, x0, v0, T = 0.9, 4.2, 4.9, 0.3, 0.2, -1.0, 3.0
    # particular: v_p(t) = F/gam + a cos(om t) + b sin(om t), a = amp gam/(gam^2+om^2), b = amp om/(gam^2+om^2)
    a = amp * gam / (gam * gam + om * om)
    b = amp * om / (gam * gam + om * om)
    c = v0 - F / gam - a
    vT = F / gam + a * math.cos(om * T) + b * math.sin(om * T) + c * math.exp(-gam * T)
    xT = x0 + F / gam * T + a / om * math.sin(om * T) - b / om * (math.cos(om * T) - 1) + c / gam * (1 - math.exp(-gam * T))
    errs = []
    for n in (300, 600, 1200):
        p = orc.params_array([dict(F=F, gamma=gam, amp=amp, omega=om, x0_fixed=x0, v0_lo=v0, v0_hi=v0)])
        out, _ = orc.simulate(p, 1, n, T / n, SEED, model=orc.INERTIAL)
        errs.append((abs(out[0, orc.OUT_XT] - xT), abs(out[0, orc.OUT_VT] - vT)))
    for i in range(2):
        for k in range(2):
            assert 3.5 < errs[i][k] / errs[i + 1][k] < 4.5, errs
    assert errs[-1][0] < 1e-4 and errs[-1][1] < 1e-4


def test_p11_inertial_single_step_in_high_precision(orc):
    mp.mp.dps = 40
    par = dict(A1=1.0, A2=0.0, F=0.1, D=0.9e-3, Fa=0.5, Fb=0.5, mu_a=1.0, mu_b=1.0, gamma=0.9, amp=4.2, omega=4.9)
    p = orc.make_params(**par)

    def A(x, v, t, d):
        return (v, -mp.mpf(par["gamma"]) * v - 2 * mp.pi * mp.cos(2 * mp.pi * x) + mp.mpf(par["amp"]) * mp.cos(mp.mpf(par["omega"]) * t)
                + mp.mpf(par["F"]) + (mp.mpf(par["Fb"]) if d else -mp.mpf(par["Fa"])))
    for x0, v0, t0, h0, g0, d in ((0.3, 1.1, 0.0, 3.2e-3, 0.4, 1), (0.95, -1.7, 12.5, 1.1e-3, -2.0, 0)):
        x, v, t, h, g = (mp.mpf(s) for s in (x0, v0, t0, h0, g0))
        nv = mp.sqrt(2 * mp.mpf(par["D"]) * h) * g
        a1 = A(x, v, t, d)
        xb, vb = x + a1[0] * h, v + a1[1] * h + nv
        a2 = A(xb, vb, t + h, d)
        xb, vb = x + (a1[0] + a2[0]) * h / 2, v + (a1[1] + a2[1]) * h / 2 + nv
        a2 = A(xb, vb, t + h, d)
        xe, ve = x + (a1[0] + a2[0]) * h / 2, v + (a1[1] + a2[1]) * h / 2 + nv
        gx, gv = orc.substep_inertial(p, orc.POT_SINE2, d, t0, h0, g0, x0, v0)
        assert abs(gx - float(xe)) < 1e-15 and abs(gv - float(ve)) < 2e-15


def test_p11_drive_time_inside_a_split_grid_step(orc):
    """Reading R5 / SURVEY O7: a sub-step that starts inside a grid step sees the drive at t = n dt + tau, not at n dt.
    The linear driven ODE of the test above with Poisson kicks of amplitude ZERO (lambda > 0, zeta = 0): the kicks split
    grid steps (jump-adapted grid) but move nothing, so every path must still follow the closed form at
    order 2 and stay within O(dt^2) of the unsplit run.  A drive evaluated at the start of the grid step instead of the
    start of the sub-step is an O(dt) error per split and breaks both."""
    gam, amp, om, F, x0, v0, T, lam = 0.9, 4.2, 4.9, 0.3, 0.2, -1.0, 3.0, 40.0
    a = amp * gam / (gam * gam + om * om)
    b = amp * om / (gam * gam + om * om)
    c = v0 - F / gam - a
    vT = F / gam + a * math.cos(om * T) + b * math.sin(om * T) + c * math.exp(-gam * T)
    xT = x0 + F / gam * T + a / om * math.sin(om * T) - b / om * (math.cos(om * T) - 1) + c / gam * (1 - math.exp(-gam * T))
    n_paths = 64
    errs = []
    for n in (300, 600, 1200):
        base = dict(F=F, gamma=gam, amp=amp, omega=om, x0_fixed=x0, v0_lo=v0, v0_hi=v0)
        split, _ = orc.simulate(orc.params_array([dict(base, lambda_=lam, zeta=0.0)]), n_paths, n, T / n, SEED,
                                model=orc.INERTIAL)
        plain, _ = orc.simulate(orc.params_array([base]), 1, n, T / n, SEED, model=orc.INERTIAL)
        assert split[:, orc.OUT_JUMPS].min() >= 60            # ~120 kicks per path: most grid steps near them are split
        assert np.all(split[:, orc.OUT_SUBSTEPS] == n + split[:, orc.OUT_JUMPS])
        ex = np.abs(split[:, orc.OUT_XT] - xT).max()
        ev = np.abs(split[:, orc.OUT_VT] - vT).max()
        errs.append((ex, ev))
        # splitting a step changes the result only at the order of the scheme's own error
        e0 = max(abs(plain[0, orc.OUT_XT] - xT), abs(plain[0, orc.OUT_VT] - vT))
        assert ex < 3 * e0 and ev < 3 * e0, (n, ex, ev, e0)
    for i in range(2):
        for k in range(2):
            # order 2 or better (the share of split steps, lambda dt = 0.4 / 0.2 / 0.1, falls with dt; an O(dt) error
            # of the drive time would give a ratio of 2 and errors sixty times larger)
            assert 3.3 < errs[i][k] / errs[i + 1][k] < 7.0, errs
    assert errs[-1][0] < 2e-5 and errs[-1][1] < 2e-5
