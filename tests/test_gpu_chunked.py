"""Row f2: chunked launches / checkpoint-resume through bm_simulate_chunk.  A run cut into chunks --
with the state copied to the host and back between chunks -- must be BIT-identical to the single bm_simulate call."""
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


def single(B, w, prec):
    stats, paths, _ = B.run_workload(w, prec, want_paths=True)
    return stats, paths


def chunked(B, w, prec, cuts, through_host=True):
    import torch
    cfg = B.config_for(w, prec)
    dev = torch.device("cuda:0")
    params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
    stats = torch.full((w.n_points, 8), -7.0, dtype=torch.float64, device=dev)
    paths = torch.full((w.n_points * w.n_paths, B.BM_OUT_STRIDE), -7.0, dtype=torch.float64, device=dev)
    state = torch.zeros(B.bm_state_bytes(cfg, w.n_points, w.n_paths), dtype=torch.uint8, device=dev)
    edges = [0] + list(cuts) + [w.n_steps]
    for b, e in zip(edges[:-1], edges[1:]):
        B.bm_simulate_chunk(cfg, params, w.n_points, w.n_paths, w.n_steps, w.dt, w.seed, b, e - b, state, stats, paths)
        torch.cuda.synchronize()
        if e < w.n_steps:
            assert float(stats[0, 0]) == -7.0 and float(paths[0, 0]) == -7.0   # outputs belong to the last chunk
            if through_host:                                                    # the checkpoint: host round trip
                saved = state.cpu().numpy().copy()
                state = torch.zeros_like(state)
                state.copy_(torch.from_numpy(saved))
    return stats.cpu().numpy(), paths.cpu().numpy()


CASES = {
    "C1": lambda: W.c1().scaled(n_paths=333, n_steps=4003),                     # ragged paths, ragged end
    "C2": lambda: W.c2().scaled(n_paths=200, n_steps=2400),
    "C4": lambda: W.c4().scaled(n_paths=96, n_steps=1600, points=[5, 64 * 128 + 64, 127 * 128 + 127]),
    "lit": lambda: W.Workload("lit", W.OVERDAMPED,
                              W.params_table(1, A1=1.0, D=0.05, lambda_=2.25, zeta=2 / 3, Fa=0.4, Fb=0.8, mu_a=1.5, mu_b=3.0),
                              130, 2000, 1e-3, 200, potential=W.POT_PWL, scheme=W.SCHEME_PAPER_LITERAL),
}


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("name", list(CASES))
def test_chunked_run_is_bit_identical(B, name, prec):
    w = CASES[name]()
    p = B.BM_F32 if prec == "f32" else B.BM_F64
    s0, p0 = single(B, w, p)
    nd = w.n_discard
    cuts = sorted({8, 8 * (nd // 8), 8 * (nd // 8) + 8, 8 * (w.n_steps // 16), 8 * ((w.n_steps - 1) // 8)} - {0})
    cuts = [c for c in cuts if 0 < c < w.n_steps]
    s1, p1 = chunked(B, w, p, cuts)
    assert np.array_equal(p0, p1), f"{name}/{prec}: per-path outputs differ between one launch and {len(cuts) + 1} chunks"
    assert np.array_equal(s0, s1)
    s2, p2 = chunked(B, w, p, [8 * (w.n_steps // 24)], through_host=False)
    assert np.array_equal(p0, p2) and np.array_equal(s0, s2)


def test_chunk_argument_errors(B):
    import torch
    w = W.c0().scaled(n_paths=64, n_steps=64)
    cfg = B.config_for(w, B.BM_F32)
    params = torch.from_numpy(np.ascontiguousarray(w.params)).cuda()
    stats = torch.zeros((1, 8), dtype=torch.float64, device="cuda")
    state = torch.zeros(B.bm_state_bytes(cfg, 1, 64), dtype=torch.uint8, device="cuda")
    assert B.bm_state_bytes(cfg, 1, 64) == 16 * 8 * 64 and B.bm_state_bytes(cfg, 0, 64) == 0

    def rc(begin, count, st=state):
        try:
            B.bm_simulate_chunk(cfg, params, 1, 64, 64, w.dt, w.seed, begin, count, st, stats)
        except B.BmError as e:
            return e.status
        return B.BM_OK

    assert rc(0, 12) == B.BM_ERR_INVALID_ARG            # ends inside a Gaussian block
    assert rc(4, 60) == B.BM_ERR_INVALID_ARG            # starts inside one
    assert rc(8, 64) == B.BM_ERR_INVALID_ARG            # beyond the end
    assert rc(0, 0) == B.BM_ERR_INVALID_ARG
    assert rc(0, 8, state[:1024]) == B.BM_ERR_WORKSPACE
    assert rc(0, 64) == B.BM_OK                         # one chunk = the whole run
    torch.cuda.synchronize()
