"""GPU tests of the boundary: edge cases, error codes, determinism, the reduction, the host-pointer entry."""
import ctypes as C
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


def test_error_codes(B):
    import torch
    w = W.c0().scaled(n_paths=64, n_steps=10)
    cfg = B.config_for(w, B.BM_F64)
    params = torch.from_numpy(w.params).cuda()
    stats = torch.zeros((1, 8), dtype=torch.float64, device="cuda")
    ws = torch.zeros(B.bm_workspace_bytes(cfg, 1, 64), dtype=torch.uint8, device="cuda")
    L = B.lib()

    def call(cfg=cfg, n_points=1, n_paths=64, n_steps=10, dt=1e-3, params=params, stats=stats, ws=ws, wsb=None,
             trace=None):
        return L.bm_simulate(C.byref(cfg), params.data_ptr() if params is not None else None, n_points, n_paths,
                             n_steps, dt, 1, stats.data_ptr() if stats is not None else None, None, trace,
                             ws.data_ptr() if ws is not None else None, ws.numel() if wsb is None else wsb, None)
    assert call() == B.BM_OK
    assert call(n_paths=0) == B.BM_ERR_INVALID_ARG
    assert call(n_steps=0) == B.BM_ERR_INVALID_ARG
    assert call(dt=0.0) == B.BM_ERR_INVALID_ARG
    assert call(dt=float("nan")) == B.BM_ERR_INVALID_ARG
    assert call(params=None) == B.BM_ERR_INVALID_ARG
    assert call(stats=None) == B.BM_ERR_INVALID_ARG
    assert call(wsb=8) == B.BM_ERR_WORKSPACE
    assert call(ws=None, wsb=0) == B.BM_ERR_WORKSPACE
    bad = B.config_for(w, B.BM_F64); bad.n_discard = 10
    assert call(cfg=bad) == B.BM_ERR_INVALID_ARG
    bad = B.config_for(w, B.BM_F64); bad.block_threads = 48
    assert call(cfg=bad) == B.BM_ERR_INVALID_ARG
    bad = B.config_for(w, B.BM_F64); bad.model = 7
    assert call(cfg=bad) == B.BM_ERR_INVALID_ARG
    uns = B.config_for(w, B.BM_F64); uns.model = B.BM_INERTIAL; uns.potential = B.BM_POT_PWL
    assert call(cfg=uns) == B.BM_ERR_UNSUPPORTED
    tr = B.config_for(w, B.BM_F32); tr.trace_steps = 4; tr.trace_paths = 4
    assert call(cfg=tr, trace=stats.data_ptr()) == B.BM_ERR_UNSUPPORTED
    assert B.bm_workspace_bytes(cfg, 0, 64) == 0
    torch.cuda.synchronize()


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("n_paths", [1, 31, 33, 129, 300])
def test_ragged_path_counts_and_reduction(B, prec, n_paths):
    """Ragged tails: block-partial + grid-pass reduction equals a two-pass numpy reduction of out_paths."""
    pr = B.BM_F32 if prec == "f32" else B.BM_F64
    base = W.c4().scaled(n_paths=n_paths, n_steps=300, points=[5, 77 * 128 + 3, 127 * 128 + 127])
    stats, paths, _ = B.run_workload(base, pr, want_paths=True)
    for pt in range(3):
        sl = paths[pt * n_paths:(pt + 1) * n_paths]
        assert stats[pt, 0] == n_paths
        assert abs(stats[pt, 1] - sl[:, B.BM_OUT_VBAR].mean()) <= 1e-13 * max(1, abs(sl[:, B.BM_OUT_VBAR].mean()))
        assert abs(stats[pt, 3] - sl[:, B.BM_OUT_XT].mean()) <= 1e-13 * max(1, abs(sl[:, B.BM_OUT_XT].mean()))
        if n_paths > 1:
            assert abs(stats[pt, 2] - sl[:, B.BM_OUT_VBAR].var(ddof=1)) <= 1e-10 * sl[:, B.BM_OUT_VBAR].var(ddof=1)
            assert abs(stats[pt, 4] - sl[:, B.BM_OUT_XT].var(ddof=1)) <= 1e-10 * sl[:, B.BM_OUT_XT].var(ddof=1)
        else:
            assert stats[pt, 2] == 0 and stats[pt, 4] == 0
        assert abs(stats[pt, 5] - sl[:, B.BM_OUT_JUMPS].mean()) < 1e-12
        assert abs(stats[pt, 6] - sl[:, B.BM_OUT_SUBSTEPS].mean()) < 1e-9


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_bitwise_determinism_and_stream_independence(B, prec):
    import torch
    pr = B.BM_F32 if prec == "f32" else B.BM_F64
    w = W.c1().scaled(n_paths=700, n_steps=800)
    a = B.run_workload(w, pr, want_paths=True)
    b = B.run_workload(w, pr, want_paths=True)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        c = B.run_workload(w, pr, want_paths=True)
    assert np.array_equal(a[0], c[0]) and np.array_equal(a[1], c[1])


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_paths_do_not_depend_on_grid_shape(B, prec):
    """RNG contract: path g sees the same words whatever the block size or the (points x paths) split is."""
    pr = B.BM_F32 if prec == "f32" else B.BM_F64
    one = W.c1().scaled(n_paths=512, n_steps=600)
    _, p128, _ = B.run_workload(one, pr, want_paths=True, block_threads=128)
    _, p64, _ = B.run_workload(one, pr, want_paths=True, block_threads=64)
    _, p256, _ = B.run_workload(one, pr, want_paths=True, block_threads=256)
    assert np.array_equal(p128, p64) and np.array_equal(p128, p256)
    four = W.Workload("split", one.model, np.repeat(one.params, 4, axis=0), 128, one.n_steps, one.dt, one.n_discard)
    _, p4, _ = B.run_workload(four, pr, want_paths=True)
    assert np.array_equal(p128, p4)


def test_n_discard_zero_and_sweep_with_disabled_points(B, orc):
    """lambda = 0 at some points of a Poisson sweep: that point must behave as if the source were off."""
    params = W.params_table(3, A1=1.0, A2=0.25, D=0.02, lambda_=np.array([0.0, 3.0, 0.0]), zeta=0.4)
    w = W.Workload("mixed", W.OVERDAMPED, params, 160, 500, 1e-3, 0)
    stats, paths, _ = B.run_workload(w, B.BM_F64, want_paths=True)
    ref, _ = orc.simulate(w.params, w.n_paths, w.n_steps, w.dt, w.seed, n_discard=0)
    assert np.abs(paths[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT]).max() < 1e-9
    assert np.array_equal(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS])
    assert stats[0, 5] == 0 and stats[2, 5] == 0 and stats[1, 5] > 0
    # fp32 with the oracle's word assignment (W32): a path follows the oracle's until its first kick (R13 gives
    # the sub-step that ends at a kick its own normal), so the jump-free points agree path by path and the kicked
    # point agrees for the paths without a kick; the kick counts are those of the same Poisson words
    s32, p32, _ = B.run_workload(w, B.BM_F32, want_paths=True, gauss=B.BM_GAUSS_W32)
    assert s32[0, 5] == 0 and s32[2, 5] == 0 and s32[1, 5] > 0
    quiet = ref[:, orc.OUT_JUMPS] == 0
    assert quiet.sum() > 2 * w.n_paths
    assert np.abs(p32[quiet, B.BM_OUT_XT] - ref[quiet, orc.OUT_XT]).max() < 5e-3
    assert np.abs(p32[:, B.BM_OUT_JUMPS] - ref[:, orc.OUT_JUMPS]).max() <= 1


def test_noise_source_off_ignores_parameters(B):
    w = W.c1().scaled(n_paths=64, n_steps=200)
    cfg_stats, p_on, _ = B.run_workload(w, B.BM_F64, want_paths=True)
    w_off = W.Workload("off", w.model, w.params.copy(), 64, 200, w.dt, w.n_discard)
    w_off.params[:, W.COL["lambda"]] = 0.0
    _, p_ref, _ = B.run_workload(w_off, B.BM_F64, want_paths=True)
    # run the lambda>0 table with the Poisson bit cleared: must equal the lambda=0 run
    import torch
    cfg = B.config_for(w, B.BM_F64)
    cfg.noise = B.BM_NOISE_GAUSS
    params = torch.from_numpy(w.params).cuda()
    stats = torch.zeros((1, 8), dtype=torch.float64, device="cuda")
    paths = torch.zeros((64, 6), dtype=torch.float64, device="cuda")
    B.bm_simulate(cfg, params, 1, 64, 200, w.dt, w.seed, stats, paths)
    torch.cuda.synchronize()
    assert np.array_equal(paths.cpu().numpy(), p_ref)
    assert not np.array_equal(p_on, p_ref)


def test_host_pointer_entry_matches_device_entry(B):
    w = W.c1().scaled(n_paths=300, n_steps=400)
    stats, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True)
    cfg = B.config_for(w, B.BM_F32)
    hs = np.zeros((1, 8))
    hp = np.zeros((300, 6))
    B.bm_simulate_host(cfg, np.ascontiguousarray(w.params), 1, 300, 400, w.dt, w.seed, hs, hp)
    assert np.array_equal(hs, stats) and np.array_equal(hp, paths)


def test_kernel_info_and_probe(B):
    import torch
    w = W.c1()
    info = B.bm_kernel_info(B.config_for(w, B.BM_F32), w.n_points, w.n_paths)
    assert 16 <= info["regs_per_thread"] <= 255 and info["blocks_per_sm"] >= 1 and info["sm_count"] >= 1
    assert info["launch_threads"] in (128, 256, 512)
    assert info["gauss"] == B.BM_GAUSS_W16                     # AUTO resolves to the variant measured faster
    w32 = B.bm_kernel_info(B.config_for(w, B.BM_F32, gauss=B.BM_GAUSS_W32), w.n_points, w.n_paths)
    assert w32["gauss"] == B.BM_GAUSS_W32 and w32["launch_threads"] == info["launch_threads"]
    assert B.bm_kernel_info(B.config_for(w, B.BM_F64), w.n_points, w.n_paths)["gauss"] == 0
    sink = torch.zeros(148 * 256, dtype=torch.float32, device="cuda")
    for op in range(B.BM_PROBE_COUNT):
        B.bm_pipe_probe(op, 4, 148, 256, sink)
    torch.cuda.synchronize()


@pytest.mark.parametrize("kind", ["f32", "f64", "literal-f32", "f32-inertial"])
def test_guard_bands_around_every_buffer_stay_intact(B, kind):
    """compute-sanitizer is closed on this GPU pool, so out-of-bounds writes are looked for with guard bands of our
    own: every device buffer a call may write (stats, per-path outputs, checkpoint state, workspace, histogram, moments)
    is carved out of one arena with 4 KiB of a canary pattern on both sides; ragged ensemble sizes, a multi-point sweep,
    single-launch and chunked runs; afterwards every canary byte must be untouched."""
    import torch
    dev = torch.device("cuda:0")
    n_points, n_paths, n_steps = 3, 333, 160
    if kind == "f32-inertial":
        w = W.Workload("g", W.INERTIAL, np.repeat(W.c2().params, n_points, axis=0), n_paths, n_steps, W.DT_INERTIAL, 16)
    else:
        w = W.c4().scaled(n_paths=n_paths, n_steps=n_steps, points=[5, 64 * 128 + 64, 127 * 128 + 127])
        if kind.startswith("literal"):
            w = W.Workload("g", W.OVERDAMPED, w.params, n_paths, n_steps, w.dt, 16, scheme=W.SCHEME_PAPER_LITERAL)
    prec = B.BM_F64 if kind == "f64" else B.BM_F32
    cfg = B.config_for(w, prec)
    GUARD, CANARY = 4096, 0xA5
    sizes = {"stats": n_points * 64, "paths": n_points * n_paths * B.BM_OUT_STRIDE * 8,
             "state": B.bm_state_bytes(cfg, n_points, n_paths), "ws": max(16, B.bm_workspace_bytes(cfg, n_points, n_paths)),
             "hist": n_points * 24 * 8, "mom": n_points * B.BM_MOM_STRIDE * 8}
    offs, total = {}, GUARD
    for k, sz in sizes.items():
        offs[k] = total
        total += (sz + 255) // 256 * 256 + GUARD
    arena = torch.full((total,), CANARY, dtype=torch.uint8, device=dev)
    view = {k: arena[offs[k]:offs[k] + sizes[k]] for k in sizes}
    for v in view.values():
        v.zero_()
    stats = view["stats"].view(torch.float64).view(n_points, 8)
    paths = view["paths"].view(torch.float64).view(n_points * n_paths, B.BM_OUT_STRIDE)
    hist = view["hist"].view(torch.int64).view(n_points, 24)
    mom = view["mom"].view(torch.float64).view(n_points, B.BM_MOM_STRIDE)
    params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
    B.bm_simulate(cfg, params, n_points, n_paths, n_steps, w.dt, w.seed, stats, paths, workspace=view["ws"])
    for b in range(0, n_steps, 40):
        B.bm_simulate_chunk(cfg, params, n_points, n_paths, n_steps, w.dt, w.seed, b, 40, view["state"], stats, paths, workspace=view["ws"])
        B.bm_state_histogram(cfg, n_points, n_paths, view["state"], 24, hist)
        B.bm_state_moments(cfg, n_points, n_paths, view["state"], mom)
    torch.cuda.synchronize()
    host = arena.cpu().numpy()
    mask = np.ones(total, dtype=bool)
    for k in sizes:
        mask[offs[k]:offs[k] + sizes[k]] = False
    assert np.all(host[mask] == CANARY), f"{int((host[mask] != CANARY).sum())} guard bytes overwritten"
    assert float(stats[0, 0]) == n_paths and int(hist.sum()) == n_points * n_paths * (n_steps // 40)
