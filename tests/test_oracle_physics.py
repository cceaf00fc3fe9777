"""Physics pins for the oracle.  CPU only.

P9   additive Gaussian white noise alone cannot induce a current.
P10  tilted smooth periodic potential + Gaussian noise: Stratonovich's formula (textbook; numerical quadrature).
P11  inertial free particle: <v> -> F/gamma, Var v -> Q = D/gamma (equipartition).
P14  the paper's own validation: <v> = L J with J from eq. (21a)/(21b), (22), (23) on the
     piece-wise linear potential of eq. (2) at D_G = 0.  Eq. (21b)/(22) as extracted has beta+ and beta- swapped
     (reading R12): beta_pm = exp(1/((Fa -+ 1)(Fb +- 1) tau)); the adiabatic limit tau -> infinity,
     <v> -> (Fb-Fa)/(Fa Fb), fixes the sign.
"""
import math

import numpy as np
import pytest
from scipy import integrate

from paper_1409_4923_b200.workloads import SEED


def _vbar(orc, out):
    v = out[:, orc.OUT_VBAR]
    return v.mean(), v.std(ddof=1) / math.sqrt(v.size)


def test_p9_no_current_from_equilibrium_noise(orc):
    p = orc.params_array([dict(A1=0.2, A2=0.05, F=0.0, D=0.1)])
    out, _ = orc.simulate(p, 2048, 10000, 4e-3, SEED, n_discard=1000)
    m, se = _vbar(orc, out)
    assert abs(m) < 4 * se and se < 0.02


def stratonovich_velocity(A1, A2, F, D):
    """<v> = L D (1 - e^{-LF/D}) / int_0^L dx int_x^{x+L} dy exp((U(y)-U(x))/D),  U = V - F x, L = 1."""
    def U(x):
        return A1 * math.sin(2 * math.pi * x) + A2 * math.sin(4 * math.pi * x) - F * x
    den, _ = integrate.dblquad(lambda y, x: math.exp((U(y) - U(x)) / D), 0.0, 1.0, lambda x: x, lambda x: x + 1.0,
                               epsabs=1e-10, epsrel=1e-10)
    return D * (1 - math.exp(-F / D)) / den


def test_p10_stratonovich_formula(orc):
    assert abs(stratonovich_velocity(0.0, 0.0, 0.3, 0.1) - 0.3) < 1e-9      # V=0 -> <v> = F
    A1, A2, F, D = 0.2, 0.05, 0.3, 0.1
    v_th = stratonovich_velocity(A1, A2, F, D)
    assert 0.05 < v_th < 0.29
    p = orc.params_array([dict(A1=A1, A2=A2, F=F, D=D)])
    out, _ = orc.simulate(p, 4096, 12000, 4e-3, SEED, n_discard=1200)
    m, se = _vbar(orc, out)
    assert se < 0.004
    assert abs(m - v_th) < 4 * se, (m, v_th, se)


def test_p11_inertial_equipartition(orc):
    gam, Q, F = 0.9, 0.5, 0.4
    p = orc.params_array([dict(F=F, D=gam * Q, gamma=gam, x0_fixed=0.0, v0_lo=-1.0, v0_hi=1.0)])
    N = 20000
    out, _ = orc.simulate(p, N, 1000, 0.01, SEED, model=orc.INERTIAL)
    v = out[:, orc.OUT_VT]
    assert abs(v.mean() - F / gam) < 4 * math.sqrt(Q / N) + 1e-3
    assert abs(v.var(ddof=1) - Q) < 4 * Q * math.sqrt(2 / N) + 1e-3


def J_model_I(a, DP):
    ap = math.exp(a / (DP * (a - 1)))
    am = math.exp(a / (DP * (a + 1)))
    return (ap - am) / ((ap - 1) * (am - 1)) / (4 * DP)


def J_model_II(Fa, Fb, tau):
    DD = Fa * Fb * tau
    bp = math.exp(1 / ((Fa - 1) * (Fb + 1) * tau))
    bm = math.exp(1 / ((Fa + 1) * (Fb - 1) * tau))
    return (bp - bm) / ((bp - 1) * (bm - 1)) / (4 * DD)


def test_p14_closed_form_limits():
    # D_P -> infinity: <v> -> 1/a (adiabatic: speeds a+1, a-1 over the two unit-slope segments)
    assert abs(2 * J_model_I(1.5, 1e4) - 1 / 1.5) < 1e-3
    assert abs(2 * J_model_I(1.5, 1.0) - 0.581987) < 1e-6
    assert abs(2 * J_model_I(2.5, 0.5) - 0.278192) < 1e-6
    assert abs(2 * J_model_II(3.0, 1.1, 1e5) - (1.1 - 3.0) / 3.3) < 1e-3


@pytest.mark.parametrize("a,DP", [(1.5, 1.0), (2.5, 0.5)])
def test_p14_model_I_velocity_vs_eq21a(orc, a, DP):
    """Model I: eq. (1)-(8); a = lambda zeta, D_P = lambda zeta^2; <v> = 2 J_I (eq. 23)."""
    zeta, lam = DP / a, a * a / DP
    p = orc.params_array([dict(A1=1.0, D=0.0, lambda_=lam, zeta=zeta)])
    n = 30000
    dt = (1 / lam) / 100
    out, _ = orc.simulate(p, 1024, n, dt, SEED, potential=orc.POT_PWL, n_discard=n // 10)
    m, se = _vbar(orc, out)
    th = 2 * J_model_I(a, DP)
    assert se < 0.02
    assert abs(m - th) < 4 * se + 0.004, (m, th, se)


@pytest.mark.parametrize("Fb,tau", [(1.1, 1.0), (1.6, 0.3)])
def test_p14_model_II_velocity_vs_eq21b(orc, Fb, tau):
    """Model II: eq. (12)-(17) with Fa mu_b = Fb mu_a; <v> = 2 J_II (eq. 21b with R12's beta, eq. 23)."""
    Fa = 3.0
    mu_a = Fa / (tau * (Fa + Fb))
    mu_b = Fb / (tau * (Fa + Fb))
    p = orc.params_array([dict(A1=1.0, D=0.0, Fa=Fa, Fb=Fb, mu_a=mu_a, mu_b=mu_b)])
    n = 30000
    dt = min(1 / mu_a, 1 / mu_b) / 100
    out, _ = orc.simulate(p, 1024, n, dt, SEED, potential=orc.POT_PWL, n_discard=n // 10)
    m, se = _vbar(orc, out)
    th = 2 * J_model_II(Fa, Fb, tau)
    assert th < 0 and se < 0.03
    assert abs(m - th) < 4 * se + 0.004, (m, th, se)
