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


def test_c1_full_size_fp32(B, orc, c1_full_oracle):
    """Against the oracle on ALL 65 536 paths (the same words per path on both sides for the kicks, other words for the
    normals: W16 against the oracle's W32), so that the combined standard error is that of two full ensembles and a
    systematic fp32 bias of 1.7 % of sigma(vbar) is already 3 SE."""
    w = W.c1()
    stats, _, _ = B.run_workload(w, B.BM_F32)
    assert stats[0, 0] == w.n_paths
    assert c1_full_oracle.shape[0] == w.n_paths
    check_point(stats[0], c1_full_oracle, orc, "C1 full fp32")
    lamT = 2.0 * w.n_steps * w.dt
    assert abs(stats[0, 5] - lamT) < 5 * math.sqrt(lamT / w.n_paths)            # Poisson count law
    assert abs(stats[0, 6] - (w.n_steps + stats[0, 5])) < 1e-6                  # sub-steps = grid steps + events


def test_c2_full_size_fp32(B, orc):
    w = W.c2()
    stats, _, _ = B.run_workload(w, B.BM_F32)
    assert stats[0, 0] == w.n_paths
    ids = np.sort(np.random.default_rng(12).choice(w.n_paths, 4096, replace=False))
    check_point(stats[0], oracle_sample(orc, w, ids), orc, "C2 full fp32")
    muT = 1.0 * w.n_steps * w.dt
    assert abs(stats[0, 5] - muT) < 5 * math.sqrt(muT / w.n_paths)              # flips: Poisson process of rate mu


_SWEEPS = {}


def sweep(B, name, prec, seed_shift=0, keep_points=()):
    """One full-size run of a sweep config (cached per module): (stats, {point: per-path records of that point}).  The
    per-path output of the whole sweep stays on the device; only the points asked for are copied to the host."""
    key = (name, prec, seed_shift)
    if key not in _SWEEPS:
        import torch
        w = W.CONFIGS[name]()
        cfg = B.config_for(w, prec)
        dev = torch.device("cuda:0")
        params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
        stats = torch.zeros((w.n_points, 8), dtype=torch.float64, device=dev)
        paths = (torch.empty((w.n_points * w.n_paths, B.BM_OUT_STRIDE), dtype=torch.float64, device=dev)
                 if keep_points else None)
        B.bm_simulate(cfg, params, w.n_points, w.n_paths, w.n_steps, w.dt, w.seed + seed_shift, stats, paths)
        torch.cuda.synchronize()
        kept = {pt: paths[pt * w.n_paths:(pt + 1) * w.n_paths].cpu().numpy() for pt in keep_points}
        del paths
        _SWEEPS[key] = (stats.cpu().numpy(), kept)
    return _SWEEPS[key]


def z_scores(s32, s64):
    """(<v>_32 - <v>_64) / SE per point, from the on-device statistics of two INDEPENDENT ensembles (different seeds)."""
    se = np.sqrt(s32[:, 2] / s32[:, 0] + s64[:, 2] / s64[:, 0])
    return (s32[:, 1] - s64[:, 1]) / se


def test_c3_full_size_fp32_sampled_points(B, orc):
    w = W.c3()
    stats, _ = sweep(B, "C3", B.BM_F32)
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
    stats, _ = sweep(B, "C4", B.BM_F32)
    assert stats.shape == (16384, 8) and np.all(stats[:, 0] == w.n_paths)
    for pt in (0, 37 * 128 + 90, 64 * 128 + 64, 127 * 128 + 127, 127 * 128):
        ids = pt * w.n_paths + np.arange(1024)
        check_point(stats[pt], oracle_sample(orc, w, ids), orc, f"C4 full fp32 point {pt}")
    # kick counts follow lambda T at every point of the lattice (T = 20)
    lam = w.params[:, W.COL["lambda"]]
    assert np.all(np.abs(stats[:, 5] - 20.0 * lam) < 6 * np.sqrt(20.0 * lam / w.n_paths) + 1e-9)


# ---- every point of the sweeps: fp32 against the fp64 kernels, the fp64 kernels against the oracle ------------------
# The oracle can afford a few points of a sweep; the fp64 GPU kernels can afford all of them (C3: 4 s, C4: 15 s).  So the
# fp64 sweep is anchored to the oracle at chosen points (per path for the over-damped C4, statistically for the chaotic
# inertial C3) and every point of the fp32 sweep is then compared with the fp64 sweep of an INDEPENDENT ensemble
# (seed + 1: with the same seed the kick times would be common to both and z would not have unit variance): a launch-map or
# event-form error that hits a band of points shows up as |z| > 5 there or lifts the mean of z^2 above 1.

C4_ANCHORS = [i * 128 + j for i in (0, 60, 96, 97, 98, 99, 120, 127) for j in (3, 120)]   # lambda dt = 0.02 lies between i = 97 and 98


def test_c4_every_point_fp32_against_fp64(B, orc):
    w = W.c4()
    s32, _ = sweep(B, "C4", B.BM_F32)
    s64, kept = sweep(B, "C4", B.BM_F64, seed_shift=1, keep_points=tuple(C4_ANCHORS))
    # the anchor: the fp64 sweep follows the oracle path by path at 16 points on both sides of the CELLS / LANES split
    from parity_util import assert_few_ill_conditioned, ill_conditioned
    n_chk, n_ill = 256, 0
    w1 = W.Workload("C4+1", w.model, w.params, w.n_paths, w.n_steps, w.dt, w.n_discard, seed=w.seed + 1)
    for pt in C4_ANCHORS:
        ids = pt * w.n_paths + np.arange(n_chk)
        ref = oracle_sample(orc, w1, ids)
        got = kept[pt][:n_chk]
        assert np.array_equal(got[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS]), f"point {pt}: kick counts differ"
        assert np.array_equal(got[:, B.BM_OUT_SUBSTEPS], ref[:, orc.OUT_SUBSTEPS]), f"point {pt}: sub-step counts differ"
        dx = np.abs(got[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT])
        over = np.nonzero(dx > 1e-8 * (1 + np.abs(ref[:, orc.OUT_XT])))[0]
        if over.size:
            ill = ill_conditioned(orc, w1, ids[over])
            assert ill.all(), f"point {pt}: {int((~ill).sum())} well-conditioned paths beyond 1e-8(1+|x|), max {dx[over[~ill]].max():.3e}"
            n_ill += int(ill.sum())
    assert_few_ill_conditioned(n_ill, 65536, f"C4 fp64 anchors ({len(C4_ANCHORS)} points x {n_chk} paths)")
    # every point
    z = z_scores(s32, s64)
    assert np.all(np.isfinite(z))
    worst = int(np.argmax(np.abs(z)))
    assert np.abs(z).max() < 5.0, f"point {worst}: z = {z[worst]:.2f} (<v> fp32 {s32[worst, 1]:.5f}, fp64 {s64[worst, 1]:.5f})"
    assert abs((z ** 2).mean() - 1.0) < 0.1, f"mean z^2 = {(z ** 2).mean():.3f} over {z.size} points"
    assert abs(z.mean()) < 5.0 / math.sqrt(z.size), f"mean z = {z.mean():.4f}: a bias common to the points"
    # and by bands of the lattice (rows of constant lambda, 128 points each): no band stands out
    zz = (z.reshape(128, 128) ** 2).mean(axis=1)
    assert np.abs(zz - 1.0).max() < 6.0 * math.sqrt(2.0 / 128), f"row {int(np.argmax(np.abs(zz - 1)))}: mean z^2 = {zz.max():.2f}"
    # same kick statistics in both precisions at every point (independent ensembles: 6 SE of the difference)
    lam = w.params[:, W.COL["lambda"]]
    assert np.all(np.abs(s32[:, 5] - s64[:, 5]) < 6 * np.sqrt(2 * 20.0 * lam / w.n_paths) + 1e-9)


def test_c3_every_point_fp32_against_fp64(B, orc):
    w = W.c3()
    s32, _ = sweep(B, "C3", B.BM_F32)
    s64, _ = sweep(B, "C3", B.BM_F64, seed_shift=1)
    w1 = W.Workload("C3+1", w.model, w.params, w.n_paths, w.n_steps, w.dt, w.n_discard, seed=w.seed + 1)
    for pt in (40, 200):                             # the anchor: fp64 statistics against the oracle's at two points
        ids = pt * w.n_paths + np.arange(512)
        check_point(s64[pt], oracle_sample(orc, w1, ids), orc, f"C3 full fp64 point {pt}")
    z = z_scores(s32, s64)
    assert np.all(np.isfinite(z))
    worst = int(np.argmax(np.abs(z)))
    assert np.abs(z).max() < 5.0, f"point {worst}: z = {z[worst]:.2f} (<v> fp32 {s32[worst, 1]:.5f}, fp64 {s64[worst, 1]:.5f})"
    assert abs((z ** 2).mean() - 1.0) < 0.3, f"mean z^2 = {(z ** 2).mean():.3f} over {z.size} points"      # 256 points: SE 0.09
    assert abs(z.mean()) < 5.0 / math.sqrt(z.size), f"mean z = {z.mean():.4f}: a bias common to the points"
