"""The two forms of the fp32 over-damped path kernel (bm_config.event_mode; jump adaptation; the divergence
PAPER.md:412 leaves open): CELLS (all lanes of a warp in the same grid cell) and LANES (per-lane clocks in a sliding
window).  They perform the same operations per path, so (1) every per-path output and every statistic must agree BIT
FOR BIT between CELLS, LANES and AUTO (AUTO picks per parameter point), on sweeps that mix sparse and dense points,
switched-off sources, all noise combinations, the three potentials, the Gaussian assignments, ragged ensembles, and in
chunked runs; (2) the LANES form goes against the fp64 oracle like every other kernel (3 combined standard errors, event
counts per path)."""
import numpy as np
import pytest

from paper_1409_4923_b200 import workloads as W
from parity_util import assert_3se, assert_counts_close, oracle_run

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_4923_b200 import binding
    binding.lib()
    return binding


def sweep_poisson(n_paths=300, n_steps=2000):
    lam = np.array([0.0, 0.1, 1.0, 5.0, 19.0, 21.0, 60.0, 100.0, 400.0, 3000.0])     # lambda dt from 0 to 3 events per cell
    tab = W.params_table(len(lam), A1=1.0, A2=0.25, F=0.0, D=0.01, lambda_=lam, zeta=0.3)
    return W.Workload("poisson-sweep", W.OVERDAMPED, tab, n_paths, n_steps, 1e-3, 203)


def sweep_all_sources():
    tab = W.params_table(5, A1=1.0, A2=0.25, F=0.05, D=0.02, lambda_=[0, 30, 80, 200, 4], zeta=0.2,
                         Fa=[0.5, 0.8, 0.3, 0.5, 0.6], Fb=[0.5, 0.4, 0.6, 0.5, 0.2], mu_a=[50, 0, 20, 300, 3],
                         mu_b=[30, 5, 0, 300, 9])
    return W.Workload("all-sources", W.OVERDAMPED, tab, 257, 1500, 1e-3, 100)


def sweep_dich_no_gauss():
    tab = W.params_table(3, A1=1.0, A2=0.25, D=0.0, Fa=0.7, Fb=0.4, mu_a=[40, 100, 2], mu_b=[60, 20, 1])
    return W.Workload("dich", W.OVERDAMPED, tab, 130, 1204, 1e-3, 0)


def sweep_pwl():
    tab = W.params_table(3, A1=1.0, D=[0.0, 0.05, 0.05], lambda_=[50, 150, 3], zeta=0.4)
    return W.Workload("pwl", W.OVERDAMPED, tab, 200, 1000, 1e-3, 56, potential=W.POT_PWL)


def sweep_quad():
    tab = W.params_table(2, A1=2.0, D=0.1, lambda_=[80, 2], zeta=0.1, x0_fixed=0.25)
    return W.Workload("quad", W.OVERDAMPED, tab, 96, 800, 1e-3, 80, potential=W.POT_QUAD)


CASES = [("poisson", sweep_poisson, {}), ("poisson-w32", sweep_poisson, {"gauss": "W32"}),
         ("poisson-w16p", sweep_poisson, {"gauss": "W16P"}), ("poisson-fma", sweep_poisson, {"sincos": "FMA"}),
         ("poisson-b64", sweep_poisson, {"block_threads": 64}), ("poisson-b512", sweep_poisson, {"block_threads": 512}),
         ("all", sweep_all_sources, {}), ("dich", sweep_dich_no_gauss, {}), ("pwl", sweep_pwl, {}), ("quad", sweep_quad, {})]


def run(B, w, mode, opts):
    kw = {}
    if "gauss" in opts:
        kw["gauss"] = getattr(B, "BM_GAUSS_" + opts["gauss"])
    if "sincos" in opts:
        kw["sincos"] = getattr(B, "BM_SINCOS_" + opts["sincos"])
    if "block_threads" in opts:
        kw["block_threads"] = opts["block_threads"]
    stats, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True, event_mode=mode, **kw)
    return stats, paths


@pytest.mark.parametrize("name,make,opts", CASES, ids=[c[0] for c in CASES])
def test_cells_lanes_auto_agree_bit_for_bit(B, name, make, opts):
    w = make()
    sc, pc = run(B, w, B.BM_EVENTS_CELLS, opts)
    sl, pl = run(B, w, B.BM_EVENTS_LANES, opts)
    sa, pa = run(B, w, B.BM_EVENTS_AUTO, opts)
    assert pc[:, B.BM_OUT_JUMPS].sum() > 0
    bad = np.flatnonzero((pc.view(np.uint64) != pl.view(np.uint64)).any(axis=1))
    assert bad.size == 0, f"{name}: {bad.size} paths differ between CELLS and LANES, first {bad[:4]}"
    assert np.array_equal(sc.view(np.uint64), sl.view(np.uint64))
    assert np.array_equal(pc.view(np.uint64), pa.view(np.uint64)) and np.array_equal(sc.view(np.uint64), sa.view(np.uint64))


def test_lanes_dense_events_take_the_careful_path(B):
    """lambda dt = 3: most blocks of 8 cells hold more events of a lane than its ring of 8, so the LANES form falls back
    to the all-lanes-together cell-by-cell path; still the same results."""
    tab = W.params_table(2, A1=1.0, A2=0.25, D=0.01, lambda_=[3000.0, 1500.0], zeta=0.01, Fa=0.3, Fb=0.3, mu_a=[0, 700], mu_b=[0, 900])
    w = W.Workload("very-dense", W.OVERDAMPED, tab, 70, 600, 1e-3, 60)
    sc, pc = run(B, w, B.BM_EVENTS_CELLS, {})
    sl, pl = run(B, w, B.BM_EVENTS_LANES, {})
    assert pc[:, B.BM_OUT_JUMPS].mean() > 1500
    assert np.array_equal(pc.view(np.uint64), pl.view(np.uint64)) and np.array_equal(sc.view(np.uint64), sl.view(np.uint64))


def test_lanes_chunked_run_is_bit_identical(B):
    import torch
    w = sweep_poisson(n_paths=161, n_steps=1203)
    s0, p0 = run(B, w, B.BM_EVENTS_CELLS, {})
    for mode in (B.BM_EVENTS_LANES, B.BM_EVENTS_AUTO):
        cfg = B.config_for(w, B.BM_F32, event_mode=mode)
        dev = torch.device("cuda:0")
        params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
        stats = torch.zeros((w.n_points, 8), dtype=torch.float64, device=dev)
        paths = torch.zeros((w.n_points * w.n_paths, B.BM_OUT_STRIDE), dtype=torch.float64, device=dev)
        state = torch.zeros(B.bm_state_bytes(cfg, w.n_points, w.n_paths), dtype=torch.uint8, device=dev)
        edges = [0, 8, 200, 208, 600, 1200, w.n_steps]           # around t_i = 203 and a ragged last chunk
        for b, e in zip(edges[:-1], edges[1:]):
            B.bm_simulate_chunk(cfg, params, w.n_points, w.n_paths, w.n_steps, w.dt, w.seed, b, e - b, state, stats, paths)
        torch.cuda.synchronize()
        assert np.array_equal(paths.cpu().numpy().view(np.uint64), p0.view(np.uint64))
        assert np.array_equal(stats.cpu().numpy().view(np.uint64), s0.view(np.uint64))


def od_case(mask, dense, n_paths=2048 + 13, n_steps=4000):
    kw = dict(A1=1.0, A2=0.25, F=0.05)
    if mask & 1:
        kw["D"] = 0.02
    if mask & 2:
        kw.update(lambda_=60.0 if dense else 2.5, zeta=0.04 if dense else 0.25)
    if mask & 4:
        kw.update(Fa=0.7, Fb=1.3, mu_a=45.0 if dense else 2.0, mu_b=80.0 if dense else 3.5)
    dt = 5e-3 if dense else 2e-3
    return W.Workload(f"od-mask{mask}{'-dense' if dense else ''}", W.OVERDAMPED, W.params_table(1, **kw), n_paths,
                      n_steps, dt, n_steps // 10)


@pytest.mark.parametrize("mask,dense", [(2, True), (3, True), (3, False), (4, True), (5, True), (6, True), (7, True), (7, False)])
def test_lanes_form_against_the_oracle(B, orc, mask, dense):
    w = od_case(mask, dense)
    _, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True, event_mode=B.BM_EVENTS_LANES)
    ref, _ = oracle_run(orc, w)
    assert_3se(paths, ref, B.BM_OUT_VBAR, f"{w.name} fp32 LANES <v>")
    assert_3se(paths, ref, B.BM_OUT_XT, f"{w.name} fp32 LANES x(T)")
    assert_counts_close(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS], w.name)
    assert np.array_equal(paths[:, B.BM_OUT_SUBSTEPS], w.n_steps + paths[:, B.BM_OUT_JUMPS])


def test_c4_top_corner_full_length_lanes(B, orc):
    """The points of C4 that AUTO gives to the LANES form (lambda dt > 0.02), at C4's full length and path count per point,
    against an oracle sample: 3 combined standard errors and the Poisson count law."""
    c4 = W.c4()
    pts = [127 * 128 + 127, 127 * 128 + 3, 110 * 128 + 64]
    w = c4.scaled(points=pts)
    lam = w.params[:, W.COL["lambda"]]
    assert (lam * w.dt > 0.02).all()
    stats, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True)
    n_or = 256
    for k in range(len(pts)):
        ids = np.arange(k * w.n_paths, k * w.n_paths + n_or)
        ref, _ = oracle_run(orc, w, ids=ids)
        mine = paths[k * w.n_paths:(k + 1) * w.n_paths]
        assert_3se(mine, ref, B.BM_OUT_VBAR, f"C4 point {pts[k]} <v>")
        mean_count = lam[k] * w.n_steps * w.dt
        assert abs(mine[:, B.BM_OUT_JUMPS].mean() - mean_count) <= 5 * np.sqrt(mean_count / w.n_paths)
        assert_counts_close(mine[:n_or, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS], f"C4 point {pts[k]}")


def test_event_mode_argument_errors(B):
    import torch
    w = W.c1().scaled(n_paths=64, n_steps=64)
    params = torch.from_numpy(np.ascontiguousarray(w.params)).cuda()
    stats = torch.zeros((1, 8), dtype=torch.float64, device="cuda")

    def rc(cfg, wl=w):
        try:
            B.bm_simulate(cfg, params, 1, wl.n_paths, wl.n_steps, wl.dt, wl.seed, stats)
        except B.BmError as e:
            return e.status
        torch.cuda.synchronize()
        return B.BM_OK

    assert rc(B.config_for(w, B.BM_F32, event_mode=B.BM_EVENTS_LANES)) == B.BM_OK
    assert rc(B.config_for(w, B.BM_F64, event_mode=B.BM_EVENTS_LANES)) == B.BM_ERR_UNSUPPORTED
    assert rc(B.config_for(W.c0().scaled(n_paths=64, n_steps=64), B.BM_F32, event_mode=B.BM_EVENTS_CELLS)) == B.BM_ERR_UNSUPPORTED
    bad = B.config_for(w, B.BM_F32)
    bad.event_mode = 3
    assert B.bm_workspace_bytes(bad, 1, 64) == 0


def test_per_point_step_length_decides_the_form(B, orc):
    """bm_simulate_dt: the event mode of a point follows lambda times ITS step length.  The same kick rate at dt = 2e-4
    (0.008 events per cell: CELLS) and at dt = 2e-3 (0.08: LANES) in one call; AUTO = CELLS = LANES bit for bit, and each
    point against the oracle run at its own dt."""
    import torch
    dev = torch.device("cuda:0")
    n_paths, n_steps = 1024 + 7, 3000
    params = W.params_table(3, A1=1.0, A2=0.25, F=0.02, D=0.01, lambda_=40.0, zeta=0.1)
    dts = np.array([2e-4, 2e-3, 1e-3])
    out = {}
    for mode in (B.BM_EVENTS_AUTO, B.BM_EVENTS_CELLS, B.BM_EVENTS_LANES):
        cfg = B.make_config(prec=B.BM_F32, noise=3, n_discard=300, event_mode=mode)
        st = torch.zeros((3, 8), dtype=torch.float64, device=dev)
        pa = torch.zeros((3 * n_paths, B.BM_OUT_STRIDE), dtype=torch.float64, device=dev)
        B.bm_simulate_dt(cfg, torch.from_numpy(params).to(dev), torch.from_numpy(dts).to(dev), 3, n_paths, n_steps, W.SEED, st, pa)
        torch.cuda.synchronize()
        out[mode] = (st.cpu().numpy(), pa.cpu().numpy())
    for mode in (B.BM_EVENTS_CELLS, B.BM_EVENTS_LANES):
        assert np.array_equal(out[mode][1].view(np.uint64), out[B.BM_EVENTS_AUTO][1].view(np.uint64))
        assert np.array_equal(out[mode][0].view(np.uint64), out[B.BM_EVENTS_AUTO][0].view(np.uint64))
    paths = out[B.BM_EVENTS_AUTO][1]
    for k in range(3):
        # path g of point k of the sweep = path g of a one-point run whose table has k rows before it: ids select it
        w = W.Workload("dtp", W.OVERDAMPED, params, n_paths, n_steps, float(dts[k]), 300)
        ids = np.arange(k * n_paths, (k + 1) * n_paths)
        ref, _ = oracle_run(orc, w, ids=ids)
        mine = paths[k * n_paths:(k + 1) * n_paths]
        assert_3se(mine, ref, B.BM_OUT_VBAR, f"point {k} (dt = {dts[k]}) <v>")
        assert_counts_close(mine[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS], f"point {k}")
