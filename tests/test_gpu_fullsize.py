"""fp32 parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (default block size, default
Gaussian assignment, no per-path output): the GPU runs the whole workload, the oracle computes a sample of its paths
one by one, and the ensemble statistics of the GPU (n, mean, variance per point from the on-device reduction) must
agree with the oracle's sample within 3 combined standard errors.  Properties that hold at any size ride along."""
import math

import numpy as np
import pytest

from paper_1409_4923_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_4923_b200 import binding
    binding.lib()
    return binding


def oracle_sample(orc, w, ids):
    out, _ = orc.simulate(w.params, w.n_paths, w.n_steps, w.dt, w.seed, model=w.model, potential=w.potential,
                          scheme=w.scheme, n_discard=w.n_discard, ids=np.asarray(ids, dtype=np.int64))
    return out


def check_point(stats_row, ref, orc, what):
    n, mv, vv = stats_row[0], stats_row[1], stats_row[2]
    v = ref[:, orc.OUT_VBAR]
    se = math.hypot(math.sqrt(vv / n), v.std(ddof=1) / math.sqrt(v.size))
    assert abs(mv - v.mean()) <= 3 * se, f"{what}: <v> gpu {mv:.6f} vs oracle sample {v.mean():.6f}, 3 SE = {3 * se:.2e}"
    c = v - v.mean()
    se_var_o = math.sqrt(max((c ** 4).mean() - (c ** 2).mean() ** 2, 0.0) / v.size)
    se_var_g = vv * math.sqrt(2.0 / n) * 2.0           # generous normal-theory bound for the large ensemble
    assert abs(vv - v.var(ddof=1)) <= 3 * math.hypot(se_var_o, se_var_g), f"{what}: Var v {vv:.3e} vs {v.var(ddof=1):.3e}"
    x = ref[:, orc.OUT_XT]
    se_x = math.hypot(math.sqrt(stats_row[4] / n), x.std(ddof=1) / math.sqrt(x.size))
    assert abs(stats_row[3] - x.mean()) <= 3 * se_x, f"{what}: <x(T)> {stats_row[3]:.4f} vs {x.mean():.4f}"


def test_c1_full_size_fp32(B, orc):
    w = W.c1()
    stats, _, _ = B.run_workload(w, B.BM_F32)
    assert stats[0, 0] == w.n_paths
    ids = np.sort(np.random.default_rng(11).choice(w.n_paths, 2048, replace=False))
    check_point(stats[0], oracle_sample(orc, w, ids), orc, "C1 full fp32")
    lamT = 2.0 * w.n_steps * w.dt
    assert abs(stats[0, 5] - lamT) < 5 * math.sqrt(lamT / w.n_paths)            # Poisson count law
    assert abs(stats[0, 6] - (w.n_steps + stats[0, 5])) < 1e-6                  # sub-steps = grid steps + events


def test_c2_full_size_fp32(B, orc):
    w = W.c2()
    stats, _, _ = B.run_workload(w, B.BM_F32)
    assert stats[0, 0] == w.n_paths
    ids = np.sort(np.random.default_rng(12).choice(w.n_paths, 768, replace=False))
    check_point(stats[0], oracle_sample(orc, w, ids), orc, "C2 full fp32")
    muT = 1.0 * w.n_steps * w.dt
    assert abs(stats[0, 5] - muT) < 5 * math.sqrt(muT / w.n_paths)              # flips: Poisson process of rate mu


def test_c3_full_size_fp32_sampled_points(B, orc):
    w = W.c3()
    stats, _, _ = B.run_workload(w, B.BM_F32)
    assert np.all(stats[:, 0] == w.n_paths)
    for pt in (0, 128, 255):
        ids = pt * w.n_paths + np.arange(1024)       # the whole point: 1024 paths
        check_point(stats[pt], oracle_sample(orc, w, ids), orc, f"C3 full fp32 point {pt}")
    # flips per path at every point: a Poisson process of rate mu = 1 over T = 2000 periods (5 SE)
    muT = 1.0 * w.n_steps * w.dt
    assert np.all(np.abs(stats[:, 5] - muT) < 5 * math.sqrt(muT / w.n_paths))
    # the sweep is antisymmetric up to the ratchet bias: <v> increases with the load f on average
    assert stats[-32:, 1].mean() > stats[:32, 1].mean()


def test_c4_full_size_fp32_sampled_points(B, orc):
    w = W.c4()
    stats, _, _ = B.run_workload(w, B.BM_F32)
    assert stats.shape == (16384, 8) and np.all(stats[:, 0] == w.n_paths)
    for pt in (0, 37 * 128 + 90, 64 * 128 + 64, 127 * 128 + 127, 127 * 128):
        ids = pt * w.n_paths + np.arange(1024)
        check_point(stats[pt], oracle_sample(orc, w, ids), orc, f"C4 full fp32 point {pt}")
    # kick counts follow lambda T at every point of the lattice (T = 20)
    lam = w.params[:, W.COL["lambda"]]
    assert np.all(np.abs(stats[:, 5] - 20.0 * lam) < 6 * np.sqrt(20.0 * lam / w.n_paths) + 1e-9)
