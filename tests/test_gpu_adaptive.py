"""Row f4: dynamic step size control from chi = xbar - x (reading R14) --
the CUDA kernel (BM_SCHEME_ADAPTIVE, fp64) against the oracle per path: the same sub-step sequence (every halve / double
decision taken alike, both sides in fp64), the same events, x(T) within 1e-8 (1 + |x|), ensemble <v> within 1e-9."""
import numpy as np
import pytest

from paper_1409_4923_b200 import workloads as W
from parity_util import ill_conditioned

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_4923_b200 import binding
    binding.lib()
    return binding


def adaptive(w, tol, levels):
    return W.Workload(w.name + "-adaptive", w.model, w.params, w.n_paths, w.n_steps, w.dt, w.n_discard, w.potential,
                      W.SCHEME_ADAPTIVE, w.seed, extra=dict(adapt_tol=tol, adapt_levels=levels))


CASES = {
    "C0": lambda: adaptive(W.c0().scaled(n_paths=333, n_steps=2000), 2e-6, 5),
    "C1": lambda: adaptive(W.Workload("c1", W.OVERDAMPED, W.params_table(1, A1=1.0, A2=0.25, D=0.01, lambda_=2.0, zeta=0.3), 300,
                                      1500, 4e-3, 150), 1e-5, 6),
    "all-sources-sweep": lambda: adaptive(W.Workload("all", W.OVERDAMPED,
                                                     W.params_table(3, A1=1.0, A2=0.25, F=0.05, D=[0.02, 0.0, 0.05], lambda_=[2.5, 8.0, 0.0],
                                                                    zeta=0.25, Fa=0.7, Fb=1.3, mu_a=[2.0, 0.0, 9.0], mu_b=3.5),
                                                     130, 1200, 5e-3, 120), 3e-5, 4),
    "OU": lambda: adaptive(W.Workload("ou", W.OVERDAMPED, W.params_table(1, A1=2.0, D=0.3, x0_fixed=1.5), 256, 200, 0.08, 0,
                                      potential=W.POT_QUAD), 1e-4, 6),
}


@pytest.mark.parametrize("name", list(CASES))
def test_adaptive_scheme_fp64_matches_oracle_per_path(B, orc, name):
    w = CASES[name]()
    stats, paths, trace = B.run_workload(w, B.BM_F64, want_paths=True, trace_steps=64, trace_paths=32)
    ref, rtrace = orc.simulate(w.params, w.n_paths, w.n_steps, w.dt, w.seed, potential=w.potential, scheme=orc.SCHEME_ADAPTIVE,
                               n_discard=w.n_discard, adapt_tol=w.extra["adapt_tol"], adapt_levels=w.extra["adapt_levels"],
                               trace_paths=32, trace_steps=64)
    assert np.array_equal(paths[:, B.BM_OUT_SUBSTEPS], ref[:, orc.OUT_SUBSTEPS]), "a step-size decision was taken differently"
    assert np.array_equal(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS])
    sub = ref[:, orc.OUT_SUBSTEPS] - ref[:, orc.OUT_JUMPS]
    assert sub.min() > w.n_steps and np.unique(sub).size > 8            # refined, and differently from path to path
    dx = np.abs(paths[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT])
    over = np.nonzero(dx > 1e-8 * (1 + np.abs(ref[:, orc.OUT_XT])))[0]
    assert over.size == 0, f"{over.size} paths beyond 1e-8(1+|x|), max {dx.max():.3e}"
    assert np.abs(trace[:, :, 0] - rtrace[:, :, 0]).max() <= 1e-10 * (1 + np.abs(rtrace[:, :, 0]).max())
    for pt in range(w.n_points):
        o = orc.reduce(ref[pt * w.n_paths:(pt + 1) * w.n_paths])
        assert abs(stats[pt, 1] - o["mean_v"]) <= 1e-9 * abs(o["mean_v"]) + 1e-12
        assert abs(stats[pt, 6] - o["mean_substeps"]) <= 1e-12 * o["mean_substeps"]


def test_adaptive_scheme_limits_and_unsupported_combinations(B, orc):
    import torch
    base = W.Workload("c1", W.OVERDAMPED, W.params_table(1, A1=1.0, A2=0.25, D=0.01, lambda_=2.0, zeta=0.3), 200, 600, 2e-3, 60)
    _, fixed, _ = B.run_workload(base, B.BM_F64, want_paths=True)
    _, never, _ = B.run_workload(adaptive(base, float("inf"), 6), B.BM_F64, want_paths=True)
    assert np.array_equal(fixed[:, [B.BM_OUT_JUMPS, B.BM_OUT_SUBSTEPS]], never[:, [B.BM_OUT_JUMPS, B.BM_OUT_SUBSTEPS]])
    assert np.abs(fixed - never).max() <= 1e-12          # tol = inf: the jump-adapted scheme (another kernel, same arithmetic)
    w = adaptive(base, 1e-5, 4)
    params = torch.from_numpy(np.ascontiguousarray(w.params)).cuda()
    stats = torch.zeros((1, 8), dtype=torch.float64, device="cuda")
    for kw, want in ((dict(prec=B.BM_F32), B.BM_ERR_UNSUPPORTED), (dict(model=B.BM_INERTIAL), B.BM_ERR_UNSUPPORTED),
                     (dict(adapt_levels=21), B.BM_ERR_INVALID_ARG), (dict(adapt_tol=-1.0), B.BM_ERR_INVALID_ARG),
                     (dict(adapt_tol=float("nan")), B.BM_ERR_INVALID_ARG)):
        cfg = B.make_config(**{**dict(prec=B.BM_F64, scheme=B.BM_SCHEME_ADAPTIVE, noise=3, n_discard=60, adapt_tol=1e-5, adapt_levels=4), **kw})
        with pytest.raises(B.BmError) as e:
            B.bm_simulate(cfg, params, 1, w.n_paths, w.n_steps, w.dt, w.seed, stats)
        assert e.value.status == want, kw
    cfg = B.config_for(w, B.BM_F64)
    state = torch.zeros(B.bm_state_bytes(cfg, 1, w.n_paths), dtype=torch.uint8, device="cuda")
    with pytest.raises(B.BmError) as e:
        B.bm_simulate_chunk(cfg, params, 1, w.n_paths, w.n_steps, w.dt, w.seed, 0, 64, state, stats)
    assert e.value.status == B.BM_ERR_UNSUPPORTED
