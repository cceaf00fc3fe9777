"""CPU-side checks of the boundary: the C-ABI library loads and exports every symbol include/bm.h declares, the
struct layouts of the binding match the header, and host-side argument validation works without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1409_4923_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_1409_4923_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "bm.h")).read()
    return sorted(set(re.findall(r"BM_API\s+[\w\s\*]+?\b(bm_\w+)\s*\(", src)))


def test_header_symbols_are_exported(B):
    syms = declared_symbols()
    assert set(syms) == set(B.EXPORTS), (syms, B.EXPORTS)
    for s in syms:
        assert hasattr(B.lib(), s), s


def test_struct_layouts_match_header(B):
    assert C.sizeof(B.BmConfig) == 80
    assert len(W.FIELDS) == 16 and len(B.STATS_FIELDS) == 8
    hdr = open(os.path.join(ROOT, "include", "bm.h")).read()
    body = hdr[hdr.index("typedef struct {", hdr.index("One parameter point")):hdr.index("} bm_params;")]
    names = re.findall(r"\b([A-Za-z_]\w*)\s*[,;]", re.sub(r"/\*.*?\*/", "", body, flags=re.S))
    assert tuple(names) == W.FIELDS
    cbody = hdr[hdr.rindex("typedef struct {", 0, hdr.index("} bm_config;")):hdr.index("} bm_config;")]
    cnames = re.findall(r"\b(?:int32_t|int64_t|double)\s+([A-Za-z_]\w*)\s*;", re.sub(r"/\*.*?\*/", "", cbody, flags=re.S))
    assert cnames == [f[0] for f in B.BmConfig._fields_], cnames
    cfg = B.make_config()
    cfg.event_mode = 3                       # not a bm_event_mode
    assert B.bm_workspace_bytes(cfg, 1, 128) == 0


def test_version_and_status_strings(B):
    assert B.bm_version() == 210
    assert B.status_string(B.BM_OK) == "BM_OK" and B.status_string(B.BM_ERR_CUDA) == "BM_ERR_CUDA"
    assert B.status_string(99) == "BM_ERR_UNKNOWN"


def test_workspace_bytes_host_logic(B):
    cfg = B.make_config(prec=B.BM_F32)
    assert B.bm_workspace_bytes(cfg, 1, 128) == 64
    assert B.bm_workspace_bytes(cfg, 3, 129) == 3 * 2 * 64
    cfg.block_threads = 64
    assert B.bm_workspace_bytes(cfg, 1, 128) == 128
    cfg.block_threads = 50
    assert B.bm_workspace_bytes(cfg, 1, 128) == 0
    assert B.bm_workspace_bytes(B.make_config(), 0, 1) == 0 and B.bm_workspace_bytes(B.make_config(), 1, 0) == 0


def test_invalid_arguments_are_rejected_before_any_cuda_call(B):
    cfg = B.make_config()
    L = B.lib()
    p = np.zeros((1, 16)); st = np.zeros((1, 8))
    assert L.bm_simulate(C.byref(cfg), None, 1, 32, 10, 1e-3, 1, st.ctypes.data, None, None, None, 0, None) == B.BM_ERR_INVALID_ARG
    assert L.bm_simulate(C.byref(cfg), p.ctypes.data, 1, 32, 10, -1.0, 1, st.ctypes.data, None, None, None, 0, None) == B.BM_ERR_INVALID_ARG
    assert L.bm_simulate(C.byref(cfg), p.ctypes.data, 1, 32, 10, 1e-3, 1, st.ctypes.data, None, None, None, 0, None) == B.BM_ERR_WORKSPACE
    assert L.bm_philox_fill(1, 0, 0, 1, 0, 4, None, None) == B.BM_ERR_INVALID_ARG
    assert L.bm_gauss_fill(B.BM_F64, 0, 1, 0, 4, 2, 4, p.ctypes.data, None) == B.BM_ERR_INVALID_ARG   # m0 % 8 != 0


def test_host_entry_validates_parameter_values(B):
    """negative rates / intensities and non-positive amplitudes of a source that is on are
    BM_ERR_INVALID_ARG.  Only the HOST entry can see the values; it rejects them before any CUDA call."""
    st = np.zeros((1, 8))

    def rc(noise=7, model=B.BM_OVERDAMPED, **kw):
        base = dict(A1=1.0, D=0.01, lambda_=2.0, zeta=0.3, Fa=0.5, Fb=0.5, mu_a=1.0, mu_b=1.0, gamma=0.9)
        base.update(kw)
        cfg = B.make_config(noise=noise, model=model)
        try:
            B.bm_simulate_host(cfg, W.params_table(1, **base), 1, 32, 10, 1e-3, 1, st)
        except B.BmError as e:
            return e.status
        return B.BM_OK
    for bad in (dict(D=-1e-3), dict(lambda_=-1.0), dict(zeta=0.0), dict(zeta=-0.3), dict(mu_a=-1.0), dict(mu_b=-2.0),
                dict(Fa=0.0), dict(Fb=-0.5), dict(A1=float("nan")), dict(F=float("inf"))):
        assert rc(**bad) == B.BM_ERR_INVALID_ARG, bad
    assert rc(model=B.BM_INERTIAL, gamma=-0.1) == B.BM_ERR_INVALID_ARG
    assert rc(model=B.BM_INERTIAL, v0_lo=1.0, v0_hi=-1.0) == B.BM_ERR_INVALID_ARG
    # a source that is switched off ignores its parameters; a rate of zero switches a source off at that point
    import torch
    ok = B.BM_OK if torch.cuda.is_available() else B.BM_ERR_CUDA
    assert rc(noise=B.BM_NOISE_GAUSS, lambda_=-1.0, mu_a=-1.0) == ok
    assert rc(lambda_=0.0, zeta=0.0, mu_a=0.0, Fa=0.0) == ok


def test_step_count_limits(B):
    """The fp32 kernels count grid cells in 32 bits; the fp64 kernels index the Gaussian stream in a 32-bit counter word."""
    L = B.lib()
    p = np.zeros((1, 16)); st = np.zeros((1, 8))
    for prec, limit in ((B.BM_F32, 0x7FFFFFF0), (B.BM_F64, 1 << 33)):
        cfg = B.make_config(prec=prec)
        assert L.bm_simulate(C.byref(cfg), p.ctypes.data, 1, 32, limit + 1, 1e-3, 1, st.ctypes.data, None, None, None, 0, None) == B.BM_ERR_INVALID_ARG
        assert L.bm_simulate(C.byref(cfg), p.ctypes.data, 1, 32, limit, 1e-3, 1, st.ctypes.data, None, None, None, 0, None) == B.BM_ERR_WORKSPACE


def test_adaptive_step_count_limit_and_reserved_fields(B):
    """The adaptive scheme can take 2^adapt_levels sub-steps per grid step, all indexed by the same 32-bit counter word
    (bm.h, bm_simulate): n_steps * 2^adapt_levels <= 2^33.  paths_per_thread outside the fp64 jump-adapted kernels is
    BM_ERR_UNSUPPORTED and a non-zero rsv BM_ERR_INVALID_ARG, as bm.h says."""
    L = B.lib()
    p = np.zeros((1, 16)); st = np.zeros((1, 8))

    def rc(cfg, n_steps):
        return L.bm_simulate(C.byref(cfg), p.ctypes.data, 1, 32, n_steps, 1e-3, 1, st.ctypes.data, None, None, None, 0, None)
    for levels in (0, 7, 20):
        cfg = B.make_config(prec=B.BM_F64, scheme=B.BM_SCHEME_ADAPTIVE, adapt_tol=1e-5, adapt_levels=levels)
        limit = (1 << 33) >> levels
        assert rc(cfg, limit + 1) == B.BM_ERR_INVALID_ARG
        assert rc(cfg, limit) == B.BM_ERR_WORKSPACE            # past the argument checks
    for kw in (dict(prec=B.BM_F32, paths_per_thread=1), dict(prec=B.BM_F64, scheme=B.BM_SCHEME_PAPER_LITERAL, paths_per_thread=1),
               dict(prec=B.BM_F64, scheme=B.BM_SCHEME_ADAPTIVE, paths_per_thread=2)):
        assert rc(B.make_config(**kw), 10) == B.BM_ERR_UNSUPPORTED, kw
    assert rc(B.make_config(prec=B.BM_F64, paths_per_thread=1), 10) == B.BM_ERR_WORKSPACE
    cfg = B.make_config(); cfg.rsv = 1
    assert rc(cfg, 10) == B.BM_ERR_INVALID_ARG
    assert B.bm_workspace_bytes(cfg, 1, 32) == 0


def test_no_cpu_fallback_without_a_device(B):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    cfg = B.make_config()
    p = np.zeros((1, 16)); st = np.zeros((1, 8))
    with pytest.raises(B.BmError) as e:
        B.bm_simulate_host(cfg, p, 1, 32, 10, 1e-3, 1, st)
    assert e.value.status == B.BM_ERR_CUDA
    assert np.all(st == 0)


def test_noise_mask_and_workload_tables(B):
    assert B.noise_mask(W.c0().params) == B.BM_NOISE_GAUSS
    assert B.noise_mask(W.c1().params) == B.BM_NOISE_GAUSS | B.BM_NOISE_POISSON
    assert B.noise_mask(W.c3().params) == B.BM_NOISE_GAUSS | B.BM_NOISE_DICH
    w = W.c4()
    assert w.n_points == 16384 and w.path_steps == 16384 * 4096 * 20000
    assert abs(w.params[0, W.COL["lambda"]] - 0.1) < 1e-15 and abs(w.params[-1, W.COL["lambda"]] - 100) < 1e-12
    assert abs(w.params[1, W.COL["zeta"]] - (0.05 + 0.95 / 127)) < 1e-15     # point = i*128 + j, j = zeta index
    w3 = W.c3()
    assert w3.n_points == 256 and w3.params[0, W.COL["F"]] == -0.5 and w3.params[-1, W.COL["F"]] == 0.5
    assert abs(w3.dt - 3.2057067893773e-3) < 1e-15
    s = W.c1().scaled(n_paths=10, n_steps=1000)
    assert s.n_discard == 100
