"""Row f3: the stationary density p(x mod L) of eq. (19), as a histogram of the reduced
coordinate at the chunk boundaries of a chunked run (bm_state_histogram).

CPU part: the oracle's own histogram (from its trace output) is pinned by the Boltzmann density of an equilibrium
system (Gaussian noise only, no load): p(x) ~ exp(-V(x)/D), a textbook closed form.
GPU part: the CUDA histogram against the oracle's, bin by bin."""
import math

import numpy as np
import pytest
from scipy import integrate

from paper_1409_4923_b200 import workloads as W


def boltzmann_bins(A1, A2, D, n_bins):
    f = lambda x: math.exp(-(A1 * math.sin(2 * math.pi * x) + A2 * math.sin(4 * math.pi * x)) / D)
    w = np.array([integrate.quad(f, i / n_bins, (i + 1) / n_bins)[0] for i in range(n_bins)])
    return w / w.sum()


def test_oracle_histogram_matches_boltzmann_density(orc):
    A1, A2, D, n_bins = 0.2, 0.05, 0.1, 16
    p = orc.params_array([dict(A1=A1, A2=A2, F=0.0, D=D)])
    n_paths, n_steps = 512, 6000
    _, tr = orc.simulate(p, n_paths, n_steps, 4e-3, W.SEED, trace_paths=n_paths, trace_steps=n_steps)
    steps = np.arange(1200, n_steps + 1, 160)            # ~2.5 correlation times apart, after equilibration
    counts = orc.hist_from_trace(tr[:, :, 0], steps, 1.0, n_bins)
    n = counts.sum()
    assert n == n_paths * steps.size
    p_th = boltzmann_bins(A1, A2, D, n_bins)
    assert p_th.max() / p_th.min() > 5                   # the density is far from flat: the test can fail
    z = (counts / n - p_th) / np.sqrt(p_th * (1 - p_th) / n)
    assert np.abs(z).max() < 4.5, z
    assert (z ** 2).sum() < 2.5 * n_bins


@pytest.mark.gpu
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("name", ["C1", "C2", "literal"])
def test_gpu_state_histogram_matches_oracle(orc, name, prec):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1409_4923_b200 import binding as B
    w = {"C1": W.c1().scaled(n_paths=384, n_steps=2400),
         "C2": W.c2().scaled(n_paths=256, n_steps=2400),
         "literal": W.Workload("lit", W.OVERDAMPED, W.params_table(1, A1=1.0, D=0.05, lambda_=2.25, zeta=2 / 3), 320, 2400,
                               2e-3, 240, potential=W.POT_PWL, scheme=W.SCHEME_PAPER_LITERAL)}[name]
    period = 2.0 if w.potential == W.POT_PWL else 1.0
    n_bins, chunk = 24, 80
    p = B.BM_F64 if prec == "f64" else B.BM_F32
    cfg = B.config_for(w, p)
    dev = torch.device("cuda:0")
    params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
    stats = torch.zeros((1, 8), dtype=torch.float64, device=dev)
    state = torch.zeros(B.bm_state_bytes(cfg, 1, w.n_paths), dtype=torch.uint8, device=dev)
    counts = torch.zeros((1, n_bins), dtype=torch.int64, device=dev)
    sample_steps = []
    for b in range(0, w.n_steps, chunk):
        B.bm_simulate_chunk(cfg, params, 1, w.n_paths, w.n_steps, w.dt, w.seed, b, chunk, state, stats)
        if b + chunk > w.n_discard:
            B.bm_state_histogram(cfg, 1, w.n_paths, state, n_bins, counts)
            sample_steps.append(b + chunk)
    torch.cuda.synchronize()
    got = counts.cpu().numpy()[0]
    _, tr = orc.simulate(w.params, w.n_paths, w.n_steps, w.dt, w.seed, model=w.model, potential=w.potential,
                         scheme=w.scheme, n_discard=w.n_discard, trace_paths=w.n_paths, trace_steps=w.n_steps)
    ref = orc.hist_from_trace(tr[:, :, 0], sample_steps, period, n_bins)
    assert got.sum() == ref.sum() == w.n_paths * len(sample_steps)
    if prec == "f64" and name != "C2":
        # same paths to 1e-12: only a position within rounding of a bin edge can change bins
        assert np.abs(got - ref).sum() <= 4, (got, ref)
    else:
        # fp32 (other normals) and the chaotic inertial model: the same density, not the same paths
        pr = (ref + 0.5) / ref.sum()
        z = (got - ref) / np.sqrt(2 * ref.sum() * pr * (1 - pr) * 8)     # samples of a path are correlated: x8 variance
        assert np.abs(z).max() < 4.5, z
