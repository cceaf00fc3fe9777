"""Every jump-adapted kernel the library can launch, against the oracle: the noise combinations BASELINE.json's five
configs do not reach.  Over-damped model with dichotomous noise at smooth V (Model II, eq. 12), with
Poissonian and dichotomous noise together and with all three sources (eq. 24: the scheduler takes the
minimum over both jump clocks, ties apply the kick first), asymmetric rates and forces; the inertial model with
Poissonian kicks (v += z, reading R7); parameter points whose dichotomous rates are zero; dense events (several per
grid cell).  fp64: per path |dx| <= 1e-8 (1 + |x|) with equal event and sub-step counts (over-damped), (x, v) within
1e-10 relative over the first 1000 grid steps (inertial); fp32: 3 combined standard errors, event counts per path."""
import math

import numpy as np
import pytest

from paper_1409_4923_b200 import workloads as W
from parity_util import assert_3se, assert_counts_close, assert_few_ill_conditioned, ill_conditioned, oracle_run

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_4923_b200 import binding
    binding.lib()
    return binding


def od_case(mask, dense=False, n_paths=777, n_steps=6000):
    """Over-damped ratchet at the smooth potential of C0/C1 with the sources of `mask` (1 Gaussian, 2 Poisson, 4 dich.)."""
    kw = dict(A1=1.0, A2=0.25, F=0.05)
    if mask & 1:
        kw["D"] = 0.02
    if mask & 2:
        kw.update(lambda_=60.0 if dense else 2.5, zeta=0.04 if dense else 0.25)
    if mask & 4:
        kw.update(Fa=0.7, Fb=1.3, mu_a=45.0 if dense else 2.0, mu_b=80.0 if dense else 3.5)
    dt = 5e-3 if dense else 2e-3      # dense: lambda dt = 0.3, mu dt = 0.2-0.4: several events in one grid cell are common
    return W.Workload(f"od-mask{mask}{'-dense' if dense else ''}", W.OVERDAMPED, W.params_table(1, **kw), n_paths,
                      n_steps, dt, n_steps // 10)


OD_CASES = [(4, False), (5, False), (6, False), (7, False), (6, True), (7, True), (3, True)]


@pytest.mark.parametrize("mask,dense", OD_CASES)
def test_overdamped_noise_combinations_fp64_per_path(B, orc, mask, dense):
    w = od_case(mask, dense)
    assert B.noise_mask(w.params) == mask
    stats, paths, _ = B.run_workload(w, B.BM_F64, want_paths=True)
    ref, _ = oracle_run(orc, w)
    assert np.array_equal(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS]), "event counts differ"
    assert np.array_equal(paths[:, B.BM_OUT_SUBSTEPS], ref[:, orc.OUT_SUBSTEPS]), "sub-step counts differ"
    assert ref[:, orc.OUT_JUMPS].mean() > (1000 if dense else 20)
    dx = np.abs(paths[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT])
    over = np.nonzero(dx > 1e-8 * (1 + np.abs(ref[:, orc.OUT_XT])))[0]
    if over.size:
        ill = ill_conditioned(orc, w, over)
        assert ill.all(), f"{int((~ill).sum())} well-conditioned paths beyond 1e-8(1+|x|), max {dx[over[~ill]].max():.3e}"
        assert_few_ill_conditioned(int(ill.sum()), dx.size, w.name)
    else:
        o = orc.reduce(ref)
        assert abs(stats[0, 1] - o["mean_v"]) <= 1e-9 * abs(o["mean_v"]) + 1e-13
        assert abs(stats[0, 4] - o["var_xT"]) <= 1e-9 * o["var_xT"]
    assert abs(stats[0, 5] - ref[:, orc.OUT_JUMPS].mean()) < 1e-9


@pytest.mark.parametrize("gauss", ["W16", "W32"])
@pytest.mark.parametrize("mask,dense", OD_CASES)
def test_overdamped_noise_combinations_fp32(B, orc, mask, dense, gauss):
    w = od_case(mask, dense, n_paths=2048 + 13, n_steps=4000)
    _, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True, gauss=B.BM_GAUSS_W32 if gauss == "W32" else B.BM_GAUSS_AUTO)
    ref, _ = oracle_run(orc, w)
    assert_3se(paths, ref, B.BM_OUT_VBAR, f"{w.name} fp32 <v>")
    assert_3se(paths, ref, B.BM_OUT_XT, f"{w.name} fp32 x(T)")
    assert_counts_close(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS], w.name)
    assert np.array_equal(paths[:, B.BM_OUT_SUBSTEPS], w.n_steps + paths[:, B.BM_OUT_JUMPS])


def inertial_case(mask, n_paths, n_steps, dense=False):
    """The motor of C2 with Poissonian kicks in the velocity (R7) added to, or instead of, the dichotomous force."""
    kw = dict(A1=1.0, F=0.1, gamma=0.9, amp=4.2, omega=4.9, v0_lo=-2.0, v0_hi=2.0)
    if mask & 1:
        kw["D"] = 0.9e-3
    if mask & 2:
        kw.update(lambda_=40.0 if dense else 1.5, zeta=0.1 if dense else 0.6)
    if mask & 4:
        kw.update(Fa=0.4, Fb=0.7, mu_a=30.0 if dense else 1.2, mu_b=55.0 if dense else 0.8)
    return W.Workload(f"in-mask{mask}", W.INERTIAL, W.params_table(1, **kw), n_paths, n_steps, W.DT_INERTIAL, n_steps // 10)


@pytest.mark.parametrize("mask,dense", [(2, False), (3, False), (7, False), (3, True), (7, True), (4, False)])
def test_inertial_kicks_fp64_trace(B, orc, mask, dense):
    w = inertial_case(mask, 384 + 5, 1200, dense)
    stats, paths, trace = B.run_workload(w, B.BM_F64, want_paths=True, trace_steps=1000, trace_paths=w.n_paths)
    ref, rtrace = oracle_run(orc, w, trace_paths=w.n_paths, trace_steps=1000)
    rel = np.abs(trace - rtrace) / np.maximum(1.0, np.abs(rtrace))
    assert rel.max() <= 1e-10, f"{w.name}: trace deviates by {rel.max():.3e}"
    assert np.array_equal(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS])
    assert np.array_equal(paths[:, B.BM_OUT_SUBSTEPS], ref[:, orc.OUT_SUBSTEPS])
    assert ref[:, orc.OUT_JUMPS].mean() > (100 if dense else 2)
    if mask & 2:    # a kick changes v, not x: v(t) is discontinuous, x(t) is not -- the largest one-step change of x is
        # |v| dt, of v it is a kick
        assert np.abs(np.diff(trace[:, :, 1], axis=1)).max() > 0.3
        assert np.abs(np.diff(trace[:, :, 0], axis=1)).max() < 0.2


@pytest.mark.parametrize("mask,dense", [(3, False), (7, False), (7, True)])
def test_inertial_kicks_fp32(B, orc, mask, dense):
    w = inertial_case(mask, 2048, 12000, dense)
    _, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True)
    ref, _ = oracle_run(orc, w)
    assert_3se(paths, ref, B.BM_OUT_VBAR, f"{w.name} fp32 <v>")
    assert_3se(paths, ref, B.BM_OUT_VT, f"{w.name} fp32 v(T)")
    assert_counts_close(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS], w.name)


def test_sweep_points_with_zero_dichotomous_rates(B, orc):
    """mu_a = 0 at a point of a sweep switches the dichotomous source off there (Gamma = 0, as the oracle); mu_b = 0 with
    mu_a > 0 makes +Fb absorbing.  All kernels: jump-adapted fp64 / fp32 and the paper-literal scheme."""
    params = W.params_table(4, A1=1.0, A2=0.25, D=0.02, Fa=0.6, Fb=0.9, mu_a=np.array([0.0, 2.0, 2.0, 0.0]),
                            mu_b=np.array([0.0, 3.0, 0.0, 3.0]))
    for scheme in (W.SCHEME_JUMP_ADAPTED, W.SCHEME_PAPER_LITERAL):
        w = W.Workload("mu0", W.OVERDAMPED, params, 160, 1500, 2e-3, 0, scheme=scheme)
        ref, _ = oracle_run(orc, w)
        assert np.all(ref[:160, orc.OUT_JUMPS] == 0) and np.all(ref[480:, orc.OUT_JUMPS] == 0)
        assert np.all(ref[320:480, orc.OUT_JUMPS] <= 1) and ref[160:320, orc.OUT_JUMPS].mean() > 3
        s64, p64, _ = B.run_workload(w, B.BM_F64, want_paths=True)
        assert np.array_equal(p64[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS])
        assert np.abs(p64[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT]).max() < 1e-9
        s32, p32, _ = B.run_workload(w, B.BM_F32, want_paths=True, gauss=B.BM_GAUSS_W32)
        assert np.abs(p32[:, B.BM_OUT_JUMPS] - ref[:, orc.OUT_JUMPS]).max() <= (1 if scheme == W.SCHEME_JUMP_ADAPTED else 2)
        assert np.all(p32[:160, B.BM_OUT_JUMPS] == 0) and np.all(p32[480:, B.BM_OUT_JUMPS] == 0)
        # points 0 and 3 (source off: Gaussian noise only) and paths of point 2 that sit in the absorbing state follow
        # the oracle path by path in fp32 as well (same words for the same purpose, W32)
        quiet = ref[:, orc.OUT_JUMPS] == 0
        assert np.abs(p32[quiet, B.BM_OUT_XT] - ref[quiet, orc.OUT_XT]).max() < 2e-2
        assert np.median(np.abs(p32[quiet, B.BM_OUT_XT] - ref[quiet, orc.OUT_XT])) < 2e-4


def test_negative_rate_of_leaving_fb_is_the_absorbing_state_in_every_kernel(B, orc):
    """bm.h: "mu_b <= 0 with mu_a > 0 makes +Fb absorbing".  bm_simulate does not check parameter values (device
    pointer), so a negative mu_b reaches the kernels: it must behave as mu_b = 0 bit for bit -- an infinite sojourn, not a
    negative waiting time -- in the fp64, fp32, paper-literal and adaptive kernels, and as the oracle."""
    def table(mu_b):
        return W.params_table(2, A1=1.0, A2=0.25, D=0.02, Fa=0.6, Fb=0.9, mu_a=np.array([2.0, 40.0]), mu_b=mu_b)
    cases = [(W.SCHEME_JUMP_ADAPTED, B.BM_F64, {}), (W.SCHEME_JUMP_ADAPTED, B.BM_F32, {}),
             (W.SCHEME_PAPER_LITERAL, B.BM_F64, {}), (W.SCHEME_PAPER_LITERAL, B.BM_F32, {}),
             (W.SCHEME_ADAPTIVE, B.BM_F64, dict(adapt_tol=1e-5, adapt_levels=3))]
    for scheme, prec, extra in cases:
        def run(mu_b):
            w = W.Workload("mub", W.OVERDAMPED, table(mu_b), 200, 800, 2e-3, 0, scheme=scheme, extra=dict(extra))
            return w, B.run_workload(w, prec, want_paths=True)
        w0, (s0, p0, _) = run(0.0)
        _, (sn, pn, _) = run(np.array([-3.0, -0.5]))
        assert np.array_equal(p0.view(np.uint64), pn.view(np.uint64)), (scheme, prec)
        assert np.array_equal(s0.view(np.uint64), sn.view(np.uint64)), (scheme, prec)
        assert np.all(p0[:, B.BM_OUT_JUMPS] == 0) and np.all(p0[:, B.BM_OUT_SUBSTEPS] >= 800)
        if prec == B.BM_F64:
            ref, _ = orc.simulate(table(np.array([-3.0, -0.5])), 200, 800, 2e-3, w0.seed, scheme=scheme, **extra)
            assert np.abs(p0[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT]).max() < 1e-9
            assert np.array_equal(p0[:, B.BM_OUT_SUBSTEPS], ref[:, orc.OUT_SUBSTEPS])


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_chunked_ragged_ensemble_of_several_waves(B, prec):
    """Row f2 at a size where the grid does not fit on the device at once and the last warp is ragged: the lanes past
    the end of the ensemble must not take part in anything (they once re-read path 0's checkpoint while its owner was
    overwriting it).  Dense kicks so that most warps take the event path within the run."""
    import torch
    n_paths = 200001 if prec == "f32" else 60001
    w = W.Workload("ragged", W.OVERDAMPED, W.params_table(1, A1=1.0, A2=0.25, D=0.01, lambda_=50.0, zeta=0.1), n_paths, 64,
                   1e-3, 8)
    p = B.BM_F32 if prec == "f32" else B.BM_F64
    s0, p0, _ = B.run_workload(w, p, want_paths=True)
    cfg = B.config_for(w, p)
    dev = torch.device("cuda:0")
    params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
    for rep in range(2):
        stats = torch.zeros((1, 8), dtype=torch.float64, device=dev)
        paths = torch.zeros((n_paths, B.BM_OUT_STRIDE), dtype=torch.float64, device=dev)
        state = torch.zeros(B.bm_state_bytes(cfg, 1, n_paths), dtype=torch.uint8, device=dev)
        for b in range(0, 64, 16):
            B.bm_simulate_chunk(cfg, params, 1, n_paths, 64, w.dt, w.seed, b, 16, state, stats, paths)
        torch.cuda.synchronize()
        assert np.array_equal(paths.cpu().numpy(), p0), f"{prec}: chunked run differs from the single launch (rep {rep})"
        assert np.array_equal(stats.cpu().numpy(), s0)
    assert p0[:, B.BM_OUT_JUMPS].mean() > 2.5


@pytest.mark.parametrize("name", ["C1", "C2", "od-all", "in-all-dense"])
def test_fp64_two_paths_per_thread_give_the_same_paths(B, name):
    """bm_config.paths_per_thread = 2 (fp64 kernels: two independent chains per thread) is the same computation per path
    as one per thread; only the reduction tree of the statistics changes.  Also for a chunked run and a ragged end."""
    import torch
    w = {"C1": lambda: W.c1().scaled(n_paths=777, n_steps=3000), "C2": lambda: W.c2().scaled(n_paths=333, n_steps=2400),
         "od-all": lambda: od_case(7, True, n_paths=300, n_steps=800), "in-all-dense": lambda: inertial_case(7, 300, 800, True)}[name]()
    s1, p1, _ = B.run_workload(w, B.BM_F64, want_paths=True, paths_per_thread=1)
    s2, p2, _ = B.run_workload(w, B.BM_F64, want_paths=True, paths_per_thread=2)
    assert np.array_equal(p1[:, [B.BM_OUT_JUMPS, B.BM_OUT_SUBSTEPS]], p2[:, [B.BM_OUT_JUMPS, B.BM_OUT_SUBSTEPS]])
    assert np.abs(p1 - p2).max() <= 1e-13 * (1 + np.abs(p1).max()), np.abs(p1 - p2).max()
    assert np.allclose(s1, s2, rtol=1e-12, atol=1e-13)
    _, p3, _ = B.run_workload(w, B.BM_F64, want_paths=True, paths_per_thread=2, block_threads=64)
    assert np.array_equal(p2, p3)
    cfg = B.config_for(w, B.BM_F64, paths_per_thread=2)
    dev = torch.device("cuda:0")
    params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
    stats = torch.zeros((1, 8), dtype=torch.float64, device=dev)
    paths = torch.zeros((w.n_paths, B.BM_OUT_STRIDE), dtype=torch.float64, device=dev)
    state = torch.zeros(B.bm_state_bytes(cfg, 1, w.n_paths), dtype=torch.uint8, device=dev)
    for b in range(0, w.n_steps, 800):
        B.bm_simulate_chunk(cfg, params, 1, w.n_paths, w.n_steps, w.dt, w.seed, b, min(800, w.n_steps - b), state, stats, paths)
    torch.cuda.synchronize()
    assert np.array_equal(paths.cpu().numpy(), p2) and np.array_equal(stats.cpu().numpy(), s2)


def test_paths_per_thread_is_an_fp64_option(B):
    import torch
    w = W.c1().scaled(n_paths=64, n_steps=16)
    params = torch.from_numpy(np.ascontiguousarray(w.params)).cuda()
    stats = torch.zeros((1, 8), dtype=torch.float64, device="cuda")
    for kw in (dict(prec=B.BM_F32), dict(prec=B.BM_F64, potential=B.BM_POT_PWL), dict(prec=B.BM_F64, scheme=B.BM_SCHEME_PAPER_LITERAL)):
        c = B.make_config(**{**dict(noise=3, paths_per_thread=2), **kw})
        with pytest.raises(B.BmError) as e:
            B.bm_simulate(c, params, 1, w.n_paths, w.n_steps, w.dt, w.seed, stats)
        assert e.value.status == B.BM_ERR_UNSUPPORTED
