"""Determinism / partition pins (P12) and the paper-literal scheme (Alg. 1-4 as printed; NEXT row f1).  CPU only."""
import math

import numpy as np
import pytest

from paper_1409_4923_b200 import workloads as W
from paper_1409_4923_b200.workloads import SEED


def test_p12_thread_count_and_subset_independence(orc):
    w = W.c1()
    a, _ = orc.simulate(w.params, 96, 500, w.dt, SEED, n_discard=50, threads=1)
    b, _ = orc.simulate(w.params, 96, 500, w.dt, SEED, n_discard=50, threads=5)
    assert np.array_equal(a, b)
    ids = np.array([95, 3, 17, 64])
    c, _ = orc.simulate(w.params, 96, 500, w.dt, SEED, n_discard=50, ids=ids)
    assert np.array_equal(c, a[ids])


def test_p12_global_path_id_decides_the_words(orc):
    """Path g = point*n_paths + p sees the same words whatever the (n_points, n_paths) split is."""
    one = W.params_table(1, A1=1.0, A2=0.25, D=0.01, lambda_=2.0, zeta=0.3)
    four = np.repeat(one, 4, axis=0)
    a, _ = orc.simulate(one, 64, 300, 1e-3, SEED)
    b, _ = orc.simulate(four, 16, 300, 1e-3, SEED)
    assert np.array_equal(a, b)


def test_reduce_two_pass(orc):
    rng = np.random.default_rng(0)
    rec = rng.normal(size=(1000, 6)) + 5.0
    st = orc.reduce(rec)
    assert st["n"] == 1000
    assert abs(st["mean_v"] - rec[:, 2].mean()) < 1e-14 and abs(st["var_v"] - rec[:, 2].var(ddof=1)) < 1e-13
    assert abs(st["mean_xT"] - rec[:, 0].mean()) < 1e-14 and abs(st["var_xT"] - rec[:, 0].var(ddof=1)) < 1e-13
    assert abs(st["mean_jumps"] - rec[:, 3].mean()) < 1e-14


def test_vbar_is_eq30(orc):
    """eq. (30): vbar = (x(t_f) - x(t_i))/(t_f - t_i), t_i = n_discard dt."""
    w = W.c0()
    out, tr = orc.simulate(w.params, 8, 400, w.dt, SEED, n_discard=100, trace_paths=8, trace_steps=400)
    x_ti = tr[:, 99, 0]
    assert np.allclose(out[:, orc.OUT_XTI], x_ti, atol=1e-15)
    assert np.allclose(out[:, orc.OUT_VBAR], (out[:, orc.OUT_XT] - x_ti) / (300 * w.dt), atol=1e-12)
    assert np.allclose(tr[:, -1, 0], out[:, orc.OUT_XT], atol=0)


def test_invalid_arguments_rejected(orc):
    w = W.c0()
    with pytest.raises(ValueError):
        orc.simulate(w.params, 8, 10, w.dt, SEED, n_discard=10)
    with pytest.raises(ValueError):
        orc.simulate(w.params, 8, 10, -1.0, SEED)
    with pytest.raises(ValueError):
        orc.simulate(w.params, 8, 10, w.dt, SEED, model=orc.INERTIAL, scheme=orc.SCHEME_PAPER_LITERAL)


# ---- paper-literal scheme ---------------------------------------------------------------------------------

def test_literal_alg2_three_point_moments(orc):
    """eq. (25): P(+-G sqrt(3 dt)) = 1/6, P(0) = 2/3 -> moments 0, 2 D dt, 0, 3 (2 D dt)^2."""
    D, dt, N = 0.3, 0.01, 60000
    p = orc.params_array([dict(D=D, x0_fixed=0.5)])
    out, _ = orc.simulate(p, N, 1, dt, SEED, scheme=orc.SCHEME_PAPER_LITERAL)
    y = out[:, orc.OUT_XT] - 0.5
    s = math.sqrt(2 * D) * math.sqrt(3 * dt)
    vals = np.unique(np.round(y / s).astype(int))
    assert set(vals) == {-1, 0, 1} and np.allclose(y / s, np.round(y / s), atol=1e-12)
    for k, pk in ((-1, 1 / 6), (0, 2 / 3), (1, 1 / 6)):
        assert abs((np.round(y / s) == k).mean() - pk) < 4 * math.sqrt(pk * (1 - pk) / N)


def test_literal_alg3_countdown_is_grid_quantised(orc):
    """Alg. 3 with [.] = floor: V=0, D=0 -> every kick lands on a grid step and the gap between
    kicks k-1 and k is floor(W_k/dt)+1 steps, W_k = -ln(1-phi)/lambda from stream-2 call k word 0."""
    lam, zeta, dt, n = 3.0, 0.5, 0.05, 200
    p = orc.params_array([dict(lambda_=lam, zeta=zeta, x0_fixed=0.0)])
    out, tr = orc.simulate(p, 16, n, dt, SEED, scheme=orc.SCHEME_PAPER_LITERAL, trace_paths=16, trace_steps=n)
    for g in range(16):
        x = np.concatenate([[0.0], tr[g, :, 0]])
        inc = np.diff(x) + lam * zeta * dt                      # kick amplitude or 0
        steps = np.nonzero(inc > 1e-12)[0]
        # replay
        exp_steps, exp_z, s, k = [], [], None, 0
        w = orc.philox_call(SEED, g, 2, 0)
        s = math.floor(-math.log(1 - (w[0] + 0.5) / 2 ** 32) / lam / dt)
        z = -zeta * math.log(1 - (w[1] + 0.5) / 2 ** 32)
        for i in range(n):
            if s <= 0:
                exp_steps.append(i); exp_z.append(z)
                k += 1
                w = orc.philox_call(SEED, g, 2, k)
                s = math.floor(-math.log(1 - (w[0] + 0.5) / 2 ** 32) / lam / dt)
                z = -zeta * math.log(1 - (w[1] + 0.5) / 2 ** 32)
            else:
                s -= 1
        assert list(steps) == exp_steps
        assert np.allclose(inc[steps], exp_z, atol=1e-12)
        assert out[g, orc.OUT_JUMPS] == len(exp_steps)


def test_literal_model_I_reproduces_paper_validation(orc):
    """PAPER.md:418-423 (Fig. 3a): spp = 400, 1024 paths, 10 % discarded, D_G = 0; <v> -> 2 J_I of eq. (21a)."""
    from test_oracle_physics import J_model_I
    a, DP = 1.5, 1.0
    zeta, lam = DP / a, a * a / DP
    p = orc.params_array([dict(A1=1.0, D=0.0, lambda_=lam, zeta=zeta)])
    n = 40000                                                   # 100 characteristic times (paper: 1000)
    out, _ = orc.simulate(p, 1024, n, (1 / lam) / 400, SEED, potential=orc.POT_PWL,
                          scheme=orc.SCHEME_PAPER_LITERAL, n_discard=n // 10)
    v = out[:, orc.OUT_VBAR]
    se = v.std(ddof=1) / math.sqrt(v.size)
    assert abs(v.mean() - 2 * J_model_I(a, DP)) < 4 * se + 0.01, (v.mean(), 2 * J_model_I(a, DP), se)


def test_literal_model_II_reproduces_paper_validation(orc):
    """PAPER.md:425 (Fig. 3b): spp = 200 of the shorter sojourn time; <v> -> 2 J_II (eq. 21b with reading R12)."""
    from test_oracle_physics import J_model_II
    Fa, Fb, tau = 3.0, 1.6, 0.3
    mu_a, mu_b = Fa / (tau * (Fa + Fb)), Fb / (tau * (Fa + Fb))
    p = orc.params_array([dict(A1=1.0, D=0.0, Fa=Fa, Fb=Fb, mu_a=mu_a, mu_b=mu_b)])
    n = 40000
    out, _ = orc.simulate(p, 1024, n, min(1 / mu_a, 1 / mu_b) / 200, SEED, potential=orc.POT_PWL,
                          scheme=orc.SCHEME_PAPER_LITERAL, n_discard=n // 10)
    v = out[:, orc.OUT_VBAR]
    se = v.std(ddof=1) / math.sqrt(v.size)
    assert abs(v.mean() - 2 * J_model_II(Fa, Fb, tau)) < 4 * se + 0.01, (v.mean(), 2 * J_model_II(Fa, Fb, tau), se)


def test_absorbing_dichotomous_state_closed_form_and_negative_rate(orc):
    """include/bm.h (bm_params.mu_b): a non-positive rate of leaving +Fb makes that state absorbing.  With mu_a > 0 the
    stationary weight of +Fb is then 1: every path starts there and never flips, so without Gaussian noise the path in
    the harmonic potential is the ODE x' = -A1 x + Fb with x(t) = Fb/A1 + (x0 - Fb/A1) e^{-A1 t} (the weak order 2.0
    scheme is the second-order Heun-type ODE scheme there).  A NEGATIVE mu_b must not give negative waiting times: it
    is the same absorbing state, bit for bit -- in all three schemes."""
    A1, Fb, x0, T, n = 1.7, 0.9, -0.4, 2.0, 400
    def table(mu_b):
        return W.params_table(1, A1=A1, D=0.0, Fa=0.6, Fb=Fb, mu_a=2.0, mu_b=mu_b, x0_fixed=x0 + 10.0)
    exact = Fb / A1 + (x0 + 10.0 - Fb / A1) * math.exp(-A1 * T)
    # (the scheme as printed keeps the constant forces out of the predictor lines: first order in dt for this ODE)
    for scheme, tol, kw in ((W.SCHEME_JUMP_ADAPTED, 2e-5, {}), (W.SCHEME_PAPER_LITERAL, 5e-3, {}),
                            (W.SCHEME_ADAPTIVE, 2e-5, dict(adapt_tol=1e-6, adapt_levels=3))):
        zero, _ = orc.simulate(table(0.0), 8, n, T / n, SEED, potential=W.POT_QUAD, scheme=scheme, **kw)
        neg, _ = orc.simulate(table(-3.0), 8, n, T / n, SEED, potential=W.POT_QUAD, scheme=scheme, **kw)
        assert np.array_equal(zero, neg)
        assert np.all(zero[:, orc.OUT_JUMPS] == 0)
        assert np.abs(zero[:, orc.OUT_XT] - exact).max() < tol * abs(exact), (scheme, zero[0, orc.OUT_XT], exact)
    # and the other way round the state is left: mu_b > 0 flips
    both, _ = orc.simulate(table(5.0), 64, n, T / n, SEED, potential=W.POT_QUAD)
    assert both[:, orc.OUT_JUMPS].mean() > 2
