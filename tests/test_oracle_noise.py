"""Pins for the oracle's noise sources and jump scheduler (R3-R5, R8).  CPU only.

P5  free motion V=0: x(T)-x0-FT ~ N(0, 2DT) exactly, for any sub-step pattern (eq. 9, :129).
P6  white Poissonian noise at V=0: compensated mean, variance (2D+2 lambda zeta^2)T (eq. 7-8, :120-125),
    third cumulant 6 lambda zeta^3 T, kick count ~ Poisson(lambda T) (eq. 4, :107).
P7  dichotomous noise: stationary law, autocovariance Fa Fb exp(-(mu_a+mu_b)|t|) (eq. 15-17, :161-171).
P8  jump-adaptation invariance: at V=0, D=0 the result does not depend on dt at all, and equals an independent
    replay of the kick sequence from the raw Philox words.
"""
import math

import numpy as np
import pytest
from scipy import stats

from paper_1409_4923_b200.workloads import SEED


def test_p5_free_motion_is_exactly_gaussian(orc):
    F, D, T, n, N = 0.7, 0.3, 2.0, 40, 20000
    # zeta=0 kicks split the steps at random times without moving the particle: variance must still be 2DT
    for lam in (0.0, 5.0):
        p = orc.params_array([dict(F=F, D=D, lambda_=lam, zeta=0.0, x0_fixed=0.25)])
        out, _ = orc.simulate(p, N, n, T / n, SEED)
        y = out[:, orc.OUT_XT] - 0.25 - F * T
        assert abs(y.mean()) < 4 * math.sqrt(2 * D * T / N)
        assert abs(y.var(ddof=1) - 2 * D * T) < 4 * 2 * D * T * math.sqrt(2 / (N - 1))
        assert stats.kstest(y / math.sqrt(2 * D * T), "norm").pvalue > 1e-3
        if lam > 0:
            assert abs(out[:, orc.OUT_JUMPS].mean() - lam * T) < 4 * math.sqrt(lam * T / N)
            assert np.all(out[:, orc.OUT_SUBSTEPS] >= n + out[:, orc.OUT_JUMPS] - 1)


def test_p5_random_x0_is_uniform(orc):
    p = orc.params_array([dict(D=0.0)])
    out, _ = orc.simulate(p, 20000, 1, 1e-9, SEED)
    assert stats.kstest(out[:, orc.OUT_XT], "uniform").pvalue > 1e-3


def test_p6_poisson_cumulants(orc):
    F, D, lam, zeta, T, n, N = 0.2, 0.05, 3.0, 0.4, 4.0, 80, 40000
    p = orc.params_array([dict(F=F, D=D, lambda_=lam, zeta=zeta, x0_fixed=0.0)])
    out, _ = orc.simulate(p, N, n, T / n, SEED)
    y = out[:, orc.OUT_XT] - F * T
    var = (2 * D + 2 * lam * zeta ** 2) * T
    k3 = 6 * lam * zeta ** 3 * T
    k4 = 24 * lam * zeta ** 4 * T
    assert abs(y.mean()) < 4 * math.sqrt(var / N)                       # compensator -lambda*zeta (eq. 3, 6)
    assert abs(y.var(ddof=1) - var) < 4 * math.sqrt((k4 + 2 * var * var) / N)
    m3 = ((y - y.mean()) ** 3).mean()
    # var(m3) ~ (mu6 - mu3^2 - 6 mu4 mu2 + 9 mu2^3)/N ; estimate mu6, mu4 from the sample itself
    c = y - y.mean()
    se3 = math.sqrt(max(((c ** 6).mean() - m3 ** 2 - 6 * (c ** 4).mean() * c.var() + 9 * c.var() ** 3), 0) / N)
    assert abs(m3 - k3) < 4 * se3
    j = out[:, orc.OUT_JUMPS]
    assert abs(j.mean() - lam * T) < 4 * math.sqrt(lam * T / N)
    assert abs(j.var(ddof=1) - lam * T) < 4 * math.sqrt((lam * T + 2 * (lam * T) ** 2) / N)
    # Poisson law itself (eq. 4): chi-square on the kick-count histogram
    kmax = 30
    obs = np.bincount(j.astype(int), minlength=kmax + 1)[:kmax + 1]
    exp = N * stats.poisson.pmf(np.arange(kmax + 1), lam * T)
    sel = exp > 20
    chi2 = ((obs[sel] - exp[sel]) ** 2 / exp[sel]).sum()
    assert chi2 < stats.chi2.ppf(0.9999, sel.sum() - 1)


def test_p6_inertial_kicks_go_to_velocity(orc):
    """R7: in the inertial model a kick z changes v (eta enters the force equation); V=0, D=0, gamma>0:
    long-time <v> = F/gamma (compensated noise has zero mean)."""
    gam, F, lam, zeta, T, n, N = 2.0, 0.5, 4.0, 0.3, 6.0, 600, 8000
    p = orc.params_array([dict(F=F, gamma=gam, lambda_=lam, zeta=zeta, x0_fixed=0.0, v0_lo=F / gam, v0_hi=F / gam)])
    out, _ = orc.simulate(p, N, n, T / n, SEED, model=orc.INERTIAL)
    v = out[:, orc.OUT_VT]
    # stationary variance of shot-noise driven OU velocity: lambda E[z^2] / (2 gamma) = lambda zeta^2 / gamma
    sd = math.sqrt(lam * zeta ** 2 / gam)
    assert abs(v.mean() - F / gam) < 4 * sd / math.sqrt(N)
    assert abs(v.var(ddof=1) / (lam * zeta ** 2 / gam) - 1) < 0.08


def test_p7_dichotomous_integral_variance_and_flip_count(orc):
    Fa, Fb, mu_a, T, n, N = 3.0, 1.5, 2.0, 5.0, 100, 20000
    mu_b = mu_a * Fb / Fa * 1.0            # zero mean needs Fa mu_b = Fb mu_a
    mu_b = Fb * mu_a / Fa
    tau = 1.0 / (mu_a + mu_b)
    p = orc.params_array([dict(Fa=Fa, Fb=Fb, mu_a=mu_a, mu_b=mu_b, x0_fixed=0.0)])
    out, _ = orc.simulate(p, N, n, T / n, SEED)
    y = out[:, orc.OUT_XT]
    var = 2 * Fa * Fb * tau * (T - tau * (1 - math.exp(-T / tau)))
    assert abs(y.mean()) < 4 * math.sqrt(var / N)
    k4 = ((y - y.mean()) ** 4).mean()
    assert abs(y.var(ddof=1) - var) < 4 * math.sqrt((k4 - y.var() ** 2) / N)
    # flips per unit time in the stationary state: 2 mu_a mu_b/(mu_a+mu_b)
    rate = 2 * mu_a * mu_b / (mu_a + mu_b)
    j = out[:, orc.OUT_JUMPS]
    assert abs(j.mean() - rate * T) < 4 * j.std() / math.sqrt(N)


def test_p7_dichotomous_autocovariance(orc):
    """C2's noise: sigma=0.5, mu=1 each way -> <G(t)G(s)> = sigma^2 exp(-2 mu |t-s|).  Increments of a free
    particle I_n = int_{t_n}^{t_n+dt} G give Cov(I_0,I_k) = sigma^2 tau^2 e^{-k dt/tau}(e^{dt/tau}-1)(1-e^{-dt/tau})."""
    sig, mu, dt, n, N = 0.5, 1.0, 0.1, 200, 4000
    tau = 1 / (2 * mu)
    p = orc.params_array([dict(Fa=sig, Fb=sig, mu_a=mu, mu_b=mu, x0_fixed=0.0)])
    out, tr = orc.simulate(p, N, n, dt, SEED, trace_paths=N, trace_steps=n)
    x = np.concatenate([np.zeros((N, 1)), tr[:, :, 0]], axis=1)
    inc = np.diff(x, axis=1)                                  # (N, n)
    assert abs(inc.mean()) < 4 * inc.std() / math.sqrt(inc.size / 10)
    # stationary start: P(+Fb) = mu_a/(mu_a+mu_b) = 1/2 already in the first step
    first = inc[:, 0]
    assert abs((first > 0).mean() - 0.5) < 4 * 0.5 / math.sqrt(N)
    for k in (1, 2, 5, 10):
        prod = (inc[:, :-k] * inc[:, k:]).mean(axis=1)
        theory = sig ** 2 * tau ** 2 * math.exp(-k * dt / tau) * (math.exp(dt / tau) - 1) * (1 - math.exp(-dt / tau))
        assert abs(prod.mean() - theory) < 4 * prod.std(ddof=1) / math.sqrt(N), (k, prod.mean(), theory)
    # variance of one increment: 2 sigma^2 tau (dt - tau (1 - e^{-dt/tau}))
    v1 = (inc ** 2).mean(axis=1)
    th = 2 * sig ** 2 * tau * (dt - tau * (1 - math.exp(-dt / tau)))
    assert abs(v1.mean() - th) < 4 * v1.std(ddof=1) / math.sqrt(N)


def test_p7_asymmetric_stationary_law(orc):
    Fa, Fb, mu_a, mu_b = 2.0, 0.5, 1.0, 4.0        # P(+Fb) = mu_a/(mu_a+mu_b) = 0.2 (from eq. 14)
    N = 20000
    p = orc.params_array([dict(Fa=Fa, Fb=Fb, mu_a=mu_a, mu_b=mu_b, x0_fixed=0.0)])
    out, tr = orc.simulate(p, N, 300, 0.01, SEED, trace_paths=N, trace_steps=300)
    # velocity over the last tiny step is -Fa or +Fb (unless a flip fell inside it)
    dx = (tr[:, -1, 0] - tr[:, -2, 0]) / 0.01
    up = np.isclose(dx, Fb, atol=1e-9).mean()
    dn = np.isclose(dx, -Fa, atol=1e-9).mean()
    assert abs(up - 0.2) < 4 * math.sqrt(0.16 / N) + 0.02 and abs(dn - 0.8) < 4 * math.sqrt(0.16 / N) + 0.02
    # <Gamma> = (Fb mu_a - Fa mu_b)/(mu_a+mu_b) = -1.5: mean displacement
    T = 3.0
    se = out[:, orc.OUT_XT].std() / math.sqrt(N)
    assert abs(out[:, orc.OUT_XT].mean() - (-1.5) * T) < 4 * se


def test_p8_jump_adaptation_invariance_and_word_replay(orc):
    F, lam, zeta, T, N = 0.3, 2.5, 0.35, 4.0, 64
    res = []
    for n in (10, 20, 160):
        p = orc.params_array([dict(F=F, D=0.0, lambda_=lam, zeta=zeta, x0_fixed=0.5)])
        out, _ = orc.simulate(p, N, n, T / n, SEED)
        res.append(out)
    for r in res[1:]:
        assert np.array_equal(r[:, orc.OUT_JUMPS], res[0][:, orc.OUT_JUMPS])
        assert np.abs(r[:, orc.OUT_XT] - res[0][:, orc.OUT_XT]).max() < 1e-12
    # independent replay from the raw words (stream 2; call k: w0 -> waiting time before kick k, w1 -> amplitude)
    for g in range(N):
        t, x, k, nj = 0.0, 0.5 + (F - lam * zeta) * T, 0, 0
        while True:
            w = orc.philox_call(SEED, g, 2, k)
            t += -math.log((w[0] + 0.5) / 2 ** 32) / lam
            if t > T:
                break
            x += -zeta * math.log((w[1] + 0.5) / 2 ** 32)
            nj += 1
            k += 1
        assert res[0][g, orc.OUT_JUMPS] == nj
        assert abs(res[0][g, orc.OUT_XT] - x) < 1e-12


def test_p8_flip_times_replay(orc):
    """D=0, V=0, dichotomous only: x(T) = sum of (+Fb or -Fa) x sojourn lengths replayed from stream-3 words."""
    Fa, Fb, mu_a, mu_b, T, N = 1.0, 2.0, 1.5, 0.7, 5.0, 64
    p = orc.params_array([dict(Fa=Fa, Fb=Fb, mu_a=mu_a, mu_b=mu_b, x0_fixed=0.0)])
    out, _ = orc.simulate(p, N, 50, T / 50, SEED)
    for g in range(N):
        w = orc.philox_call(SEED, g, 0, 0)
        d = 1 if (w[2] + 0.5) / 2 ** 32 < mu_a / (mu_a + mu_b) else 0
        t, x, k = 0.0, 0.0, 0
        while True:
            s = -math.log((orc.philox_call(SEED, g, 3, k)[0] + 0.5) / 2 ** 32) / (mu_b if d else mu_a)
            val = Fb if d else -Fa
            if t + s >= T:
                x += val * (T - t)
                break
            x += val * s
            t += s
            d = 1 - d
            k += 1
        assert out[g, orc.OUT_JUMPS] == k
        assert abs(out[g, orc.OUT_XT] - x) < 1e-12


def test_r4_initial_velocity_is_uniform_and_independent(orc):
    """Reading R4: v0 = v0_lo + (v0_hi - v0_lo) u(w1) of init-stream call 0 -- uniform on [v0_lo, v0_hi] and independent
    of x0 (word 0) and of the initial dichotomous state d (word 2).  A force-free, friction-free particle keeps v0 and
    moves by v0 dt in one step, so OUT_VT is v0 and OUT_XT - v0 dt is x0; with the two dichotomous forces switched on
    (no flips within the step, no friction) v(dt) - v0 = +Fb dt or -Fa dt reads off d."""
    from scipy import stats as st
    N, lo, hi, dt = 20000, -2.0, 2.0, 1e-6
    free = orc.params_array([dict(v0_lo=lo, v0_hi=hi)])
    out, _ = orc.simulate(free, N, 1, dt, SEED, model=orc.INERTIAL)
    v0 = out[:, orc.OUT_VT]
    x0 = out[:, orc.OUT_XT] - v0 * dt
    assert v0.min() >= lo and v0.max() <= hi
    assert st.kstest((v0 - lo) / (hi - lo), "uniform").statistic < 1.63 / math.sqrt(N)      # 1 % critical value
    assert abs(v0.mean() - 0.5 * (lo + hi)) < 4 * (hi - lo) / math.sqrt(12 * N)
    assert abs(v0.var() - (hi - lo) ** 2 / 12) < 4 * (hi - lo) ** 2 / 12 * math.sqrt(0.8 / N)   # kurtosis 1.8
    assert st.kstest(x0, "uniform").statistic < 1.63 / math.sqrt(N)
    assert abs(np.corrcoef(v0, x0)[0, 1]) < 4 / math.sqrt(N)
    # rank correlation too: a monotone but non-linear dependence would show here
    assert abs(st.spearmanr(v0, x0).statistic) < 4 / math.sqrt(N)
    dich = orc.params_array([dict(v0_lo=lo, v0_hi=hi, Fa=1.0, Fb=1.0, mu_a=1e-9, mu_b=3e-9)])
    out2, _ = orc.simulate(dich, N, 1, dt, SEED, model=orc.INERTIAL)
    assert np.all(out2[:, orc.OUT_JUMPS] == 0)
    d = np.sign(out2[:, orc.OUT_VT] - v0)                       # +1: state +Fb, -1: state -Fa
    assert np.all(np.abs(np.abs(out2[:, orc.OUT_VT] - v0) - dt) < 1e-12)
    assert abs((d > 0).mean() - 0.25) < 4 * math.sqrt(0.25 * 0.75 / N)      # P(+Fb) = mu_a / (mu_a + mu_b)
    assert abs(np.corrcoef(v0, d)[0, 1]) < 4 / math.sqrt(N)
    assert abs(np.corrcoef(x0, d)[0, 1]) < 4 / math.sqrt(N)
