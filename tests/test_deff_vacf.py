"""Row f3, second part: effective diffusion D_eff = Var x / (2 t) and the velocity autocorrelation of the
stationary state, from checkpoints of a chunked run (bm_state_moments).

CPU part: the oracle's two observable functions (plain definitions on its traces) are pinned by closed forms --
V = 0 with Gaussian and Poissonian noise spreads as Var x = (2 D + 2 lambda zeta^2) t (eq. 7-8), so
D_eff = D + lambda zeta^2 at every t; the velocity of a free inertial particle is an Ornstein-Uhlenbeck process with
stationary autocovariance Q exp(-gamma |t|) (D = gamma Q).
GPU part: bm_state_moments on the checkpoints of the CUDA run against the oracle's functions on the same workload."""
import math

import numpy as np
import pytest

from paper_1409_4923_b200 import workloads as W


def test_oracle_deff_of_free_poisson_diffusion(orc):
    D, lam, zeta, dt, n_steps, N = 0.03, 4.0, 0.2, 5e-3, 400, 12000
    p = orc.params_array([dict(D=D, lambda_=lam, zeta=zeta, x0_fixed=0.25)])
    _, tr = orc.simulate(p, N, n_steps, dt, W.SEED, trace_paths=N, trace_steps=n_steps)
    want = D + lam * zeta * zeta
    for i0, i in ((1, 101), (50, 400), (200, 400)):
        got = orc.deff_from_trace(tr, i0, i, dt)
        # the increments are sums of a Gaussian and a compound-Poisson part: kurtosis of dx is 3 + kappa4/var^2
        T = (i - i0) * dt
        k4 = 24 * lam * zeta ** 4 * T
        se = math.sqrt((2 + k4 / (2 * want * T) ** 2) / N) * want
        assert abs(got - want) < 4 * se, (i0, i, got, want, se)
    assert abs(want - D) > 20 * se          # the Poissonian part is visible: dropping it fails the test


def test_oracle_vacf_of_free_inertial_particle(orc):
    gam, Q, dt, N = 1.5, 0.4, 4e-3, 20000
    p = orc.params_array([dict(gamma=gam, D=gam * Q, v0_lo=-1.0, v0_hi=1.0, x0_fixed=0.0)])
    i0 = int(6.0 / gam / dt)                            # e^-12 of the initial variance left
    lags = [0, int(0.5 / gam / dt), int(1.0 / gam / dt), int(2.0 / gam / dt)]
    n_steps = i0 + lags[-1]
    _, tr = orc.simulate(p, N, n_steps, dt, W.SEED, model=orc.INERTIAL, trace_paths=N, trace_steps=n_steps)
    for lag in lags:
        got = orc.vacf_from_trace(tr, i0, i0 + lag)
        want = Q * math.exp(-gam * lag * dt)
        se = math.sqrt((Q * Q + want * want) / N)
        assert abs(got - want) < 4 * se + 2e-3 * Q, (lag, got, want, se)      # + the scheme's O(dt^2) error
    # and the diffusion of the position: D_eff -> Q / gamma for t >> 1/gamma
    i1 = i0 + lags[-1]
    T = (i1 - i0) * dt
    want = Q / gam * (1 - (1 - math.exp(-gam * T)) / (gam * T))       # Var dx = 2 (Q/gamma) (T - (1 - e^{-gamma T})/gamma)
    got = orc.deff_from_trace(tr, i0, i1, dt)
    assert abs(got - want) < 4 * want * math.sqrt(2 / N) + 2e-3 * want


def gpu_moments(B, w, prec, cuts):
    """Checkpoints of a chunked CUDA run at the grid steps `cuts`; moments of each against the first."""
    import torch
    cfg = B.config_for(w, prec)
    dev = torch.device("cuda:0")
    params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
    stats = torch.zeros((w.n_points, 8), dtype=torch.float64, device=dev)
    state = torch.zeros(B.bm_state_bytes(cfg, w.n_points, w.n_paths), dtype=torch.uint8, device=dev)
    out = torch.zeros((w.n_points, B.BM_MOM_STRIDE), dtype=torch.float64, device=dev)
    ref, res, b = None, [], 0
    for c in cuts:
        B.bm_simulate_chunk(cfg, params, w.n_points, w.n_paths, w.n_steps, w.dt, w.seed, b, c - b, state, stats)
        b = c
        if ref is None:
            ref = state.clone()
        B.bm_state_moments(cfg, w.n_points, w.n_paths, state, out, ref_state=ref)
        torch.cuda.synchronize()
        res.append(out.cpu().numpy().copy())
    return res


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name", ["C2-like", "C1-like", "literal"])
def test_gpu_state_moments_match_oracle(orc, name, prec):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_4923_b200 import binding as B
    w = {"C2-like": W.c2().scaled(n_paths=1500, n_steps=2400, points=None),
         "C1-like": W.Workload("c1s", W.OVERDAMPED, W.params_table(2, A1=1.0, A2=0.25, D=0.01, lambda_=[2.0, 20.0], zeta=0.3), 777,
                               2400, 1e-3, 240),
         "literal": W.Workload("lit", W.OVERDAMPED, W.params_table(1, A1=1.0, D=0.05, lambda_=2.25, zeta=2 / 3), 640, 2400, 2e-3, 240,
                               potential=W.POT_PWL, scheme=W.SCHEME_PAPER_LITERAL)}[name]
    cuts = [800, 1200, 1600, 2400]                      # multiples of BM_CHUNK_ALIGN
    got = gpu_moments(B, w, B.BM_F64 if prec == "f64" else B.BM_F32, cuts)
    N = w.n_paths
    for pt in range(w.n_points):
        ids = pt * N + np.arange(N)
        paths, tr = orc.simulate(w.params, N, w.n_steps, w.dt, w.seed, model=w.model, potential=w.potential, scheme=w.scheme,
                                 n_discard=w.n_discard, ids=ids, trace_paths=N, trace_steps=w.n_steps)
        for k, c in enumerate(cuts):
            g = got[k][pt]
            x, v = tr[:, c - 1, 0], tr[:, c - 1, 1]
            assert g[B.BM_MOM_N] == N
            if k == 0:
                assert g[B.BM_MOM_VAR_DX] == 0 and g[B.BM_MOM_MEAN_DX] == 0
                continue
            deff_o = orc.deff_from_trace(tr, cuts[0], c, w.dt)
            cov_o = orc.vacf_from_trace(tr, cuts[0], c)
            deff_g = g[B.BM_MOM_VAR_DX] / (2 * (c - cuts[0]) * w.dt)
            if prec == "f64" and w.model == W.OVERDAMPED:
                # the same paths to ~1e-12: the moments agree far below any statistical error
                assert abs(g[B.BM_MOM_MEAN_X] - x.mean()) <= 1e-9 * (1 + abs(x.mean()))
                assert abs(g[B.BM_MOM_VAR_X] - x.var(ddof=1)) <= 1e-8 * x.var(ddof=1)
                assert abs(deff_g - deff_o) <= 1e-8 * deff_o
            else:
                # fp32 (other normals, R13) and the chaotic inertial model: the same law, not the same paths
                se_x = math.sqrt(2.0 * x.var(ddof=1) / N)
                assert abs(g[B.BM_MOM_MEAN_X] - x.mean()) <= 4 * se_x
                dx = x - tr[:, cuts[0] - 1, 0]
                m2, m4 = dx.var(), ((dx - dx.mean()) ** 4).mean()
                se_d = math.sqrt(2.0 * max(m4 - m2 * m2, 0.0) / N) / (2 * (c - cuts[0]) * w.dt)
                assert abs(deff_g - deff_o) <= 4 * se_d, (name, prec, pt, c, deff_g, deff_o, se_d)
                if w.model == W.INERTIAL:
                    v0 = tr[:, cuts[0] - 1, 1]
                    se_c = math.sqrt(2.0 * (v0.var() * v.var() + cov_o ** 2) / N)
                    assert abs(g[B.BM_MOM_COV_V0V] - cov_o) <= 4 * se_c, (c, g[B.BM_MOM_COV_V0V], cov_o, se_c)
                    assert abs(g[B.BM_MOM_VAR_V] - v.var(ddof=1)) <= 4 * v.var() * math.sqrt(4.0 / N) * 2
            if w.model == W.OVERDAMPED:
                assert g[B.BM_MOM_VAR_V] == 0 and g[B.BM_MOM_COV_V0V] == 0
    if prec == "f64" and w.model == W.INERTIAL:
        # first 1000 steps of the inertial model agree per path (1e-10): a checkpoint inside that window agrees tightly
        g1 = gpu_moments(B, w, B.BM_F64, [400, 800])[1][0]
        _, tr = orc.simulate(w.params, N, 800, w.dt, w.seed, model=w.model, n_discard=0, trace_paths=N, trace_steps=800)
        assert abs(g1[B.BM_MOM_COV_V0V] - orc.vacf_from_trace(tr, 400, 800)) <= 1e-8 * tr[:, 399, 1].var()
        assert abs(g1[B.BM_MOM_VAR_DX] / (2 * 400 * w.dt) - orc.deff_from_trace(tr, 400, 800, w.dt)) <= 1e-8 * g1[B.BM_MOM_VAR_DX]


@pytest.mark.gpu
def test_gpu_state_moments_are_reproducible_and_check_arguments(orc):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_4923_b200 import binding as B
    w = W.c2().scaled(n_paths=1000, n_steps=800)
    a = gpu_moments(B, w, B.BM_F32, [400, 800])
    b = gpu_moments(B, w, B.BM_F32, [400, 800])
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    cfg = B.config_for(w, B.BM_F32)
    out = torch.zeros((1, B.BM_MOM_STRIDE), dtype=torch.float64, device="cuda")
    small = torch.zeros(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.BmError) as e:
        B.bm_state_moments(cfg, 1, w.n_paths, small, out)
    assert e.value.status == B.BM_ERR_WORKSPACE
