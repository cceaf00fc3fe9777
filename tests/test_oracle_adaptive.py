"""Pins for the oracle's dynamic step size control from chi = xbar - x (DESIGN.md
reading R14).  CPU only.

A1  tol = +inf never refines: the scheme IS the jump-adapted scheme, bit for bit, whatever noise sources are on.
A2  tol = 0 refines at every interval down to the finest level: for the deterministic linear drift the result is the
    product of the scheme's own amplification factors R(theta h) over the step sequence the controller must take
    (dt, dt/2, dt/4, ... , then dt 2^-K for ever; every interval aligned) -- computed here independently.
A3  the controller: for the deterministic linear drift chi = theta^3 h^3 x / 4 exactly (Alg. 1 worked out by hand), so
    the step sequence can be replayed here from the rule "halve above tol, double below tol/8 if aligned"; the oracle's
    sub-step count and x(T) must agree with the replay.
A4  efficiency: tol/8 halves every step of that sequence, so the global error against exp(-theta T) falls by 4
    (the scheme is of order 2), while the number of sub-steps doubles.
A5  the law is not biased by the control: the Stratonovich current of a tilted smooth potential (textbook quadrature)
    is met within 4 standard errors with steps that really vary.
"""
import math

import numpy as np
import pytest

from paper_1409_4923_b200.workloads import SEED


def R(z):
    return 1 - z + z * z / 2 - z ** 3 / 4


def test_a1_infinite_tolerance_is_the_jump_adapted_scheme(orc):
    p = orc.params_array([dict(A1=1.0, A2=0.25, F=0.1, D=0.05, lambda_=3.0, zeta=0.3, Fa=0.4, Fb=0.7, mu_a=2.0, mu_b=3.0)])
    a, ta = orc.simulate(p, 64, 400, 2e-3, SEED, n_discard=40, trace_paths=8, trace_steps=400)
    b, tb = orc.simulate(p, 64, 400, 2e-3, SEED, n_discard=40, trace_paths=8, trace_steps=400,
                         scheme=orc.SCHEME_ADAPTIVE, adapt_tol=float("inf"), adapt_levels=7)
    assert np.array_equal(a, b) and np.array_equal(ta[:, :, 0], tb[:, :, 0])
    with pytest.raises(ValueError):
        orc.simulate(p, 4, 10, 1e-3, SEED, model=orc.INERTIAL, scheme=orc.SCHEME_ADAPTIVE, adapt_tol=1e-3, adapt_levels=3)


def test_a2_zero_tolerance_walks_down_to_the_finest_level(orc):
    theta, x0, dt, n, K = 1.3, 2.0, 0.05, 12, 4
    p = orc.params_array([dict(A1=theta, D=0.0, x0_fixed=x0)])
    out, _ = orc.simulate(p, 1, n, dt, SEED, potential=orc.POT_QUAD, scheme=orc.SCHEME_ADAPTIVE, adapt_tol=0.0, adapt_levels=K)
    # the sequence the rule dictates: one interval per level on the way down, then the finest level
    x, k, steps = x0, 0, 0
    for cell in range(n):
        tick, TPC = 0, 1 << K
        while tick < TPC:
            x *= R(theta * dt / (1 << k))
            steps += 1
            tick += TPC >> k
            if k < K:
                k += 1
    assert out[0, orc.OUT_SUBSTEPS] == steps
    assert abs(out[0, orc.OUT_XT] - x) <= 1e-13 * abs(x)


def replay_linear(theta, x0, dt, n, K, tol):
    """The controller replayed on the deterministic linear drift, where chi = theta^3 h^3 x / 4 (worked by hand from
    Alg. 1: xbar1 - xbar2 = -theta^2 h^2 x / 2, chi = (h/2)(-theta)(xbar1 - xbar2))."""
    x, k, steps = x0, 0, 0
    for cell in range(n):
        tick, TPC = 0, 1 << K
        while tick < TPC:
            h = dt / (1 << k)
            w = TPC >> k
            chi = abs(theta ** 3 * h ** 3 * x / 4)
            x *= R(theta * h)
            steps += 1
            tick += w
            if chi > tol and k < K:
                k += 1
            elif chi < tol / 8 and k > 0 and tick % (2 * w) == 0:
                k -= 1
    return x, steps


def test_a3_controller_follows_the_rule(orc):
    theta, x0, dt, n, K = 2.0, 3.0, 0.08, 40, 6
    p = orc.params_array([dict(A1=theta, D=0.0, x0_fixed=x0)])
    seen = set()
    for tol in (3e-3, 1e-4, 2e-6):
        out, _ = orc.simulate(p, 1, n, dt, SEED, potential=orc.POT_QUAD, scheme=orc.SCHEME_ADAPTIVE, adapt_tol=tol,
                              adapt_levels=K)
        x, steps = replay_linear(theta, x0, dt, n, K, tol)
        assert out[0, orc.OUT_SUBSTEPS] == steps, (tol, out[0, orc.OUT_SUBSTEPS], steps)
        assert abs(out[0, orc.OUT_XT] - x) <= 1e-12 * abs(x)
        seen.add(steps)
    assert len(seen) == 3 and min(seen) > n          # the step really varies, and differs between the tolerances


def test_a4_an_eighth_of_the_tolerance_quarters_the_error(orc):
    """Measured on x(T)/x(t_s), t_s two grid steps in, so that the walk down from the first full step (every path starts
    at level 0) does not enter: exact value exp(-theta (T - t_s))."""
    theta, x0, dt, n, K = 1.0, 1.0, 0.25, 16, 12
    exact = math.exp(-theta * dt * (n - 2))
    p = orc.params_array([dict(A1=theta, D=0.0, x0_fixed=x0)])
    errs, subs = [], []
    for tol in (1e-5, 1e-5 / 8, 1e-5 / 64, 1e-5 / 512):
        out, tr = orc.simulate(p, 1, n, dt, SEED, potential=orc.POT_QUAD, scheme=orc.SCHEME_ADAPTIVE, adapt_tol=tol,
                               adapt_levels=K, trace_paths=1, trace_steps=n)
        errs.append(abs(tr[0, n - 1, 0] / tr[0, 1, 0] - exact))
        subs.append(out[0, orc.OUT_SUBSTEPS])
    for i in range(3):
        assert 3.4 < errs[i] / errs[i + 1] < 4.6, errs
        assert 1.8 < subs[i + 1] / subs[i] < 2.2, subs


def test_a5_stratonovich_current_with_varying_steps(orc):
    from test_oracle_physics import stratonovich_velocity
    A1, A2, F, D = 0.2, 0.05, 0.3, 0.1
    v_th = stratonovich_velocity(A1, A2, F, D)
    p = orc.params_array([dict(A1=A1, A2=A2, F=F, D=D)])
    N, n, dt = 4096, 3000, 1.6e-2
    out, _ = orc.simulate(p, N, n, dt, SEED, n_discard=300, scheme=orc.SCHEME_ADAPTIVE, adapt_tol=2e-5, adapt_levels=5)
    v = out[:, orc.OUT_VBAR]
    se = v.std(ddof=1) / math.sqrt(N)
    sub = out[:, orc.OUT_SUBSTEPS]
    assert 1.5 * n < sub.mean() < 20 * n and sub.std() > 0          # refined, not pinned to either end, path-dependent
    assert abs(v.mean() - v_th) < 4 * se, (v.mean(), v_th, se)
