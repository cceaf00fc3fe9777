"""Thin ctypes binding of include/bm.h: same names, argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libbm.so; PyTorch is used for device memory and streams.
There is no CPU fallback: if libbm.so is missing or cannot be loaded, every call raises.
"""
import ctypes as C
import os

import numpy as np

from . import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libbm.so")

BM_OK, BM_ERR_INVALID_ARG, BM_ERR_UNSUPPORTED, BM_ERR_WORKSPACE, BM_ERR_CUDA = range(5)
BM_OVERDAMPED, BM_INERTIAL = 0, 1
BM_F32, BM_F64 = 0, 1
BM_SINCOS_AUTO, BM_SINCOS_SFU, BM_SINCOS_FMA = 0, 1, 2
BM_POT_SINE2, BM_POT_PWL, BM_POT_QUAD = 0, 1, 2
BM_SCHEME_JUMP_ADAPTED, BM_SCHEME_PAPER_LITERAL, BM_SCHEME_ADAPTIVE = 0, 1, 2
BM_NOISE_GAUSS, BM_NOISE_POISSON, BM_NOISE_DICH = 1, 2, 4
BM_GAUSS_AUTO, BM_GAUSS_W32, BM_GAUSS_W16, BM_GAUSS_W16P = 0, 1, 2, 3
BM_EVENTS_AUTO, BM_EVENTS_CELLS, BM_EVENTS_LANES = 0, 1, 2
BM_OUT_XT, BM_OUT_VT, BM_OUT_VBAR, BM_OUT_JUMPS, BM_OUT_SUBSTEPS, BM_OUT_XTI, BM_OUT_STRIDE = 0, 1, 2, 3, 4, 5, 6
(BM_PROBE_FFMA, BM_PROBE_MUFU_COS, BM_PROBE_MUFU_LG2, BM_PROBE_MUFU_SQRT, BM_PROBE_IMAD_WIDE, BM_PROBE_LOP3,
 BM_PROBE_DFMA, BM_PROBE_I2F, BM_PROBE_FADD, BM_PROBE_MIX, BM_PROBE_COUNT) = range(11)

BM_STATE_SLOTS, BM_CHUNK_ALIGN = 16, 8
(BM_MOM_N, BM_MOM_MEAN_X, BM_MOM_VAR_X, BM_MOM_MEAN_V, BM_MOM_VAR_V, BM_MOM_MEAN_DX, BM_MOM_VAR_DX, BM_MOM_COV_V0V,
 BM_MOM_VAR_V0) = range(9)
BM_MOM_STRIDE = 10
BM_STATIC_SCRATCH_BYTES = 4 * 1024 * 1024
EXPORTS = ("bm_workspace_bytes", "bm_simulate", "bm_simulate_static", "bm_simulate_dt", "bm_state_bytes", "bm_simulate_chunk", "bm_state_histogram",
           "bm_state_moments", "bm_simulate_host", "bm_philox_fill", "bm_gauss_fill", "bm_box_muller_words", "bm_event_normal_words",
           "bm_kernel_info", "bm_pipe_probe", "bm_status_string", "bm_version")
STATS_FIELDS = ("n", "mean_v", "var_v", "mean_xT", "var_xT", "mean_jumps", "mean_substeps", "rsv")


class BmConfig(C.Structure):
    _fields_ = [("model", C.c_int32), ("prec", C.c_int32), ("sincos", C.c_int32), ("potential", C.c_int32),
                ("scheme", C.c_int32), ("noise", C.c_int32), ("block_threads", C.c_int32), ("gauss", C.c_int32),
                ("n_discard", C.c_int64), ("trace_steps", C.c_int64), ("trace_paths", C.c_int64),
                ("paths_per_thread", C.c_int32), ("adapt_levels", C.c_int32), ("adapt_tol", C.c_double),
                ("event_mode", C.c_int32), ("rsv", C.c_int32)]


class BmError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {status_string(status)}")


_lib = None


def lib():
    """Load libbm.so (fails loudly when it has not been built: there is no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1409_4923_b200.build` "
                               "(no CPU fallback exists)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, u64, u32, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64, C.c_uint32, C.c_double
        cfgp = C.POINTER(BmConfig)
        L.bm_workspace_bytes.argtypes = [cfgp, i32, i64]
        L.bm_workspace_bytes.restype = C.c_size_t
        L.bm_simulate.argtypes = [cfgp, vp, i32, i64, i64, dbl, u64, vp, vp, vp, vp, C.c_size_t, vp]
        L.bm_simulate.restype = C.c_int
        L.bm_simulate_static.argtypes = [cfgp, vp, i32, i64, i64, dbl, u64, vp, vp, vp, vp]
        L.bm_simulate_static.restype = C.c_int
        L.bm_simulate_dt.argtypes = [cfgp, vp, vp, i32, i64, i64, u64, vp, vp, vp, C.c_size_t, vp]
        L.bm_simulate_dt.restype = C.c_int
        L.bm_state_bytes.argtypes = [cfgp, i32, i64]
        L.bm_state_bytes.restype = C.c_size_t
        L.bm_simulate_chunk.argtypes = [cfgp, vp, i32, i64, i64, dbl, u64, i64, i64, vp, C.c_size_t, vp, vp, vp, C.c_size_t, vp]
        L.bm_simulate_chunk.restype = C.c_int
        L.bm_state_histogram.argtypes = [cfgp, i32, i64, vp, C.c_size_t, i32, vp, vp]
        L.bm_state_histogram.restype = C.c_int
        L.bm_state_moments.argtypes = [cfgp, i32, i64, vp, C.c_size_t, vp, vp, vp]
        L.bm_state_moments.restype = C.c_int
        L.bm_simulate_host.argtypes = [cfgp, vp, i32, i64, i64, dbl, u64, vp, vp, vp]
        L.bm_simulate_host.restype = C.c_int
        L.bm_philox_fill.argtypes = [u64, u64, i32, u32, u32, i32, vp, vp]
        L.bm_philox_fill.restype = C.c_int
        L.bm_gauss_fill.argtypes = [i32, i32, u64, u64, i32, u64, i32, vp, vp]
        L.bm_gauss_fill.restype = C.c_int
        L.bm_box_muller_words.argtypes = [i32, vp, i32, vp, vp]
        L.bm_box_muller_words.restype = C.c_int
        L.bm_event_normal_words.argtypes = [vp, i32, vp, vp]
        L.bm_event_normal_words.restype = C.c_int
        ip = C.POINTER(C.c_int32)
        L.bm_kernel_info.argtypes = [cfgp, i32, i64, ip, ip, ip, ip, ip]
        L.bm_kernel_info.restype = C.c_int
        L.bm_pipe_probe.argtypes = [i32, i32, i32, i32, vp, vp]
        L.bm_pipe_probe.restype = C.c_int
        L.bm_status_string.argtypes = [C.c_int]
        L.bm_status_string.restype = C.c_char_p
        L.bm_version.restype = C.c_int
        _lib = L
    return _lib


def status_string(s):
    return lib().bm_status_string(int(s)).decode()


def bm_version():
    return lib().bm_version()


def noise_mask(params):
    """Noise sources a parameter table switches on (host-side helper; the C ABI takes the mask explicitly)."""
    p = np.asarray(params)
    m = 0
    if np.any(p[:, W.COL["D"]] > 0):
        m |= BM_NOISE_GAUSS
    if np.any(p[:, W.COL["lambda"]] > 0):
        m |= BM_NOISE_POISSON
    if np.any(p[:, W.COL["mu_a"]] > 0):
        m |= BM_NOISE_DICH
    return m


def make_config(model=BM_OVERDAMPED, prec=BM_F32, sincos=BM_SINCOS_AUTO, potential=BM_POT_SINE2,
                scheme=BM_SCHEME_JUMP_ADAPTED, noise=BM_NOISE_GAUSS, block_threads=0, n_discard=0, trace_steps=0,
                trace_paths=0, gauss=BM_GAUSS_AUTO, paths_per_thread=0, adapt_tol=float("inf"), adapt_levels=0,
                event_mode=BM_EVENTS_AUTO):
    return BmConfig(model, prec, sincos, potential, scheme, noise, block_threads, gauss, n_discard, trace_steps,
                    trace_paths, paths_per_thread, adapt_levels, adapt_tol, event_mode, 0)


def _stream_ptr(stream):
    import torch
    if stream is None:
        if not torch.cuda.is_available():
            return None          # the library itself reports BM_ERR_CUDA; nothing is computed on the host
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def bm_workspace_bytes(cfg, n_points, n_paths):
    return int(lib().bm_workspace_bytes(C.byref(cfg), n_points, n_paths))


def bm_simulate(cfg, params, n_points, n_paths, n_steps, dt, seed, out_stats, out_paths=None, out_trace=None,
                workspace=None, stream=None):
    """Device-pointer call.  params/out_stats/out_paths/out_trace/workspace are CUDA torch tensors (float64 /
    uint8 workspace).  Asynchronous on `stream` (default: torch's current stream)."""
    import torch
    assert params.is_cuda and params.dtype == torch.float64 and params.is_contiguous() and params.numel() == 16 * n_points
    assert out_stats.is_cuda and out_stats.dtype == torch.float64 and out_stats.is_contiguous() and out_stats.numel() == 8 * n_points
    need = bm_workspace_bytes(cfg, n_points, n_paths)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=params.device)
    op = C.c_void_p(out_paths.data_ptr()) if out_paths is not None else None
    ot = C.c_void_p(out_trace.data_ptr()) if out_trace is not None else None
    if out_paths is not None:
        assert out_paths.is_cuda and out_paths.dtype == torch.float64 and out_paths.numel() == n_points * n_paths * BM_OUT_STRIDE
    if out_trace is not None:
        assert out_trace.is_cuda and out_trace.dtype == torch.float64 and out_trace.numel() == cfg.trace_paths * cfg.trace_steps * 2
    rc = lib().bm_simulate(C.byref(cfg), C.c_void_p(params.data_ptr()), n_points, n_paths, n_steps, float(dt),
                           int(seed), C.c_void_p(out_stats.data_ptr()), op, ot, C.c_void_p(workspace.data_ptr()),
                           workspace.numel(), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_simulate")
    return workspace


def bm_simulate_static(cfg, params, n_points, n_paths, n_steps, dt, seed, out_stats, out_paths=None, out_trace=None,
                       stream=None):
    """bm_simulate for callers that cannot allocate device memory (a plug-in in someone else's GPU heap, a real-time loop
    that must not call cudaMalloc): no workspace argument and no allocation of any kind, here or in the library -- the
    reduction's scratch is a fixed BM_STATIC_SCRATCH_BYTES array inside libbm.so.  Same tensors and results as
    bm_simulate.  Raises BmError(BM_ERR_WORKSPACE) when the launch would need more than that (over 65 536 thread
    blocks).  Calls on one device share the array: do not let two of them overlap on the GPU (one stream, or events)."""
    import torch
    assert params.is_cuda and params.dtype == torch.float64 and params.is_contiguous() and params.numel() == 16 * n_points
    assert out_stats.is_cuda and out_stats.dtype == torch.float64 and out_stats.is_contiguous() and out_stats.numel() == 8 * n_points
    if out_paths is not None:
        assert out_paths.is_cuda and out_paths.dtype == torch.float64 and out_paths.numel() == n_points * n_paths * BM_OUT_STRIDE
    if out_trace is not None:
        assert out_trace.is_cuda and out_trace.dtype == torch.float64 and out_trace.numel() == cfg.trace_paths * cfg.trace_steps * 2
    op = C.c_void_p(out_paths.data_ptr()) if out_paths is not None else None
    ot = C.c_void_p(out_trace.data_ptr()) if out_trace is not None else None
    rc = lib().bm_simulate_static(C.byref(cfg), C.c_void_p(params.data_ptr()), n_points, n_paths, n_steps, float(dt),
                                  int(seed), C.c_void_p(out_stats.data_ptr()), op, ot, _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_simulate_static")


def bm_simulate_dt(cfg, params, dt_points, n_points, n_paths, n_steps, seed, out_stats, out_paths=None, workspace=None,
                   stream=None):
    """bm_simulate with one step length per parameter point (dt_points: CUDA float64 tensor [n_points])."""
    import torch
    assert params.is_cuda and params.dtype == torch.float64 and params.numel() == 16 * n_points
    assert dt_points.is_cuda and dt_points.dtype == torch.float64 and dt_points.is_contiguous() and dt_points.numel() == n_points
    assert out_stats.is_cuda and out_stats.dtype == torch.float64 and out_stats.numel() == 8 * n_points
    if workspace is None:
        workspace = torch.empty(max(bm_workspace_bytes(cfg, n_points, n_paths), 16), dtype=torch.uint8, device=params.device)
    op = C.c_void_p(out_paths.data_ptr()) if out_paths is not None else None
    rc = lib().bm_simulate_dt(C.byref(cfg), C.c_void_p(params.data_ptr()), C.c_void_p(dt_points.data_ptr()), n_points,
                              n_paths, n_steps, int(seed), C.c_void_p(out_stats.data_ptr()), op,
                              C.c_void_p(workspace.data_ptr()), workspace.numel(), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_simulate_dt")
    return workspace


def bm_state_bytes(cfg, n_points, n_paths):
    return int(lib().bm_state_bytes(C.byref(cfg), n_points, n_paths))


def bm_simulate_chunk(cfg, params, n_points, n_paths, n_steps, dt, seed, step_begin, step_count, state, out_stats,
                      out_paths=None, workspace=None, stream=None):
    """Grid steps [step_begin, step_begin + step_count) of a run of n_steps; `state` is a CUDA uint8 tensor of at least
    bm_state_bytes(...) bytes that carries the run from chunk to chunk (the checkpoint)."""
    import torch
    assert params.is_cuda and params.dtype == torch.float64 and params.numel() == 16 * n_points
    assert out_stats.is_cuda and out_stats.dtype == torch.float64 and out_stats.numel() == 8 * n_points
    assert state.is_cuda and state.dtype == torch.uint8 and state.is_contiguous()
    if workspace is None:
        workspace = torch.empty(max(bm_workspace_bytes(cfg, n_points, n_paths), 16), dtype=torch.uint8, device=params.device)
    op = C.c_void_p(out_paths.data_ptr()) if out_paths is not None else None
    rc = lib().bm_simulate_chunk(C.byref(cfg), C.c_void_p(params.data_ptr()), n_points, n_paths, n_steps, float(dt),
                                 int(seed), int(step_begin), int(step_count), C.c_void_p(state.data_ptr()),
                                 state.numel(), C.c_void_p(out_stats.data_ptr()), op,
                                 C.c_void_p(workspace.data_ptr()), workspace.numel(), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_simulate_chunk")
    return workspace


def bm_state_histogram(cfg, n_points, n_paths, state, n_bins, counts, stream=None):
    """counts (CUDA int64 tensor [n_points, n_bins]) += occupation of the reduced coordinate in the checkpoint `state`."""
    import torch
    assert state.is_cuda and state.dtype == torch.uint8
    assert counts.is_cuda and counts.dtype == torch.int64 and counts.is_contiguous() and counts.numel() == n_points * n_bins
    rc = lib().bm_state_histogram(C.byref(cfg), n_points, n_paths, C.c_void_p(state.data_ptr()), state.numel(), n_bins,
                                  C.c_void_p(counts.data_ptr()), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_state_histogram")


def bm_state_moments(cfg, n_points, n_paths, state, out, ref_state=None, stream=None):
    """out (CUDA float64 tensor [n_points, BM_MOM_STRIDE]) = ensemble moments of the checkpoint `state`, optionally
    against the earlier checkpoint `ref_state` of the same run (D_eff, velocity autocovariance)."""
    import torch
    assert state.is_cuda and state.dtype == torch.uint8 and state.is_contiguous()
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() == n_points * BM_MOM_STRIDE
    rp = None
    if ref_state is not None:
        assert ref_state.is_cuda and ref_state.dtype == torch.uint8 and ref_state.numel() >= state.numel()
        rp = C.c_void_p(ref_state.data_ptr())
    rc = lib().bm_state_moments(C.byref(cfg), n_points, n_paths, C.c_void_p(state.data_ptr()), state.numel(), rp,
                                C.c_void_p(out.data_ptr()), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_state_moments")


def bm_simulate_host(cfg, params, n_points, n_paths, n_steps, dt, seed, out_stats, out_paths=None, stream=None):
    """HOST-pointer call: params/out_stats/out_paths are numpy float64 arrays (or pinned CPU torch tensors)."""
    def ptr(a):
        if a is None:
            return None
        if isinstance(a, np.ndarray):
            assert a.dtype == np.float64 and a.flags.c_contiguous
            return C.c_void_p(a.ctypes.data)
        assert (not a.is_cuda) and a.is_contiguous()
        return C.c_void_p(a.data_ptr())
    rc = lib().bm_simulate_host(C.byref(cfg), ptr(params), n_points, n_paths, n_steps, float(dt), int(seed),
                                ptr(out_stats), ptr(out_paths), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_simulate_host")


def bm_philox_fill(seed, path0, n_paths, stream_id, idx0, n_idx, out, stream=None):
    import torch
    assert out.is_cuda and out.dtype in (torch.int32, torch.uint32) and out.numel() == n_paths * n_idx * 4
    rc = lib().bm_philox_fill(int(seed), int(path0), n_paths, stream_id, idx0, n_idx, C.c_void_p(out.data_ptr()),
                              _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_philox_fill")


def bm_gauss_fill(prec, gauss, seed, path0, n_paths, m0, n_m, out, stream=None):
    import torch
    assert out.is_cuda and out.numel() == n_paths * n_m
    assert out.dtype == (torch.float64 if prec == BM_F64 else torch.float32)
    rc = lib().bm_gauss_fill(prec, gauss, int(seed), int(path0), n_paths, int(m0), n_m, C.c_void_p(out.data_ptr()),
                             _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_gauss_fill")


def bm_kernel_info(cfg, n_points=1, n_paths=1 << 30):
    r, b, o, s, w = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
    rc = lib().bm_kernel_info(C.byref(cfg), n_points, n_paths, C.byref(r), C.byref(b), C.byref(o), C.byref(s), C.byref(w))
    if rc != BM_OK:
        raise BmError(rc, "bm_kernel_info")
    return {"regs_per_thread": r.value, "launch_threads": b.value, "blocks_per_sm": o.value, "sm_count": s.value,
            "gauss": int(w.value)}


def bm_box_muller_words(prec, words, n_pairs, out, stream=None):
    """words: CUDA uint32/int32 tensor [n_pairs, 2]; out: float64 (BM_F64) or float32 (BM_F32) CUDA tensor [n_pairs, 2]."""
    rc = lib().bm_box_muller_words(prec, C.c_void_p(words.data_ptr()), n_pairs, C.c_void_p(out.data_ptr()), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_box_muller_words")


def bm_event_normal_words(words, out, stream=None):
    """words: CUDA int32/uint32 tensor [n] (word 2 of event Philox calls); out: CUDA float32 tensor [n] = the normal the
    fp32 kernels give the sub-step that ends on that event (reading R13)."""
    import torch
    assert words.is_cuda and words.dtype in (torch.int32, torch.uint32) and words.is_contiguous()
    assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous() and out.numel() == words.numel()
    rc = lib().bm_event_normal_words(C.c_void_p(words.data_ptr()), words.numel(), C.c_void_p(out.data_ptr()), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_event_normal_words")


def bm_pipe_probe(op, iters, blocks, threads, sink, stream=None):
    rc = lib().bm_pipe_probe(op, iters, blocks, threads, C.c_void_p(sink.data_ptr()), _stream_ptr(stream))
    if rc != BM_OK:
        raise BmError(rc, "bm_pipe_probe")


# ---- conveniences used by tests and bench.py (marshalling only) -------------------------------------------

def config_for(w, prec, sincos=BM_SINCOS_AUTO, block_threads=0, trace_steps=0, trace_paths=0, gauss=BM_GAUSS_AUTO,
               paths_per_thread=0, event_mode=BM_EVENTS_AUTO):
    """bm_config of a workloads.Workload (extra: adapt_tol, adapt_levels for the adaptive scheme)."""
    return make_config(model=w.model, prec=prec, sincos=sincos, potential=w.potential, scheme=w.scheme,
                       noise=noise_mask(w.params), block_threads=block_threads, n_discard=w.n_discard,
                       trace_steps=trace_steps, trace_paths=trace_paths, gauss=gauss, paths_per_thread=paths_per_thread,
                       adapt_tol=w.extra.get("adapt_tol", float("inf")), adapt_levels=w.extra.get("adapt_levels", 0),
                       event_mode=event_mode)


def run_workload(w, prec, want_paths=False, sincos=BM_SINCOS_AUTO, block_threads=0, trace_steps=0, trace_paths=0,
                 device="cuda:0", gauss=BM_GAUSS_AUTO, paths_per_thread=0, event_mode=BM_EVENTS_AUTO):
    """Run a Workload through bm_simulate; returns (stats[n_points,8], paths or None, trace or None) as numpy."""
    import torch
    cfg = config_for(w, prec, sincos, block_threads, trace_steps, trace_paths, gauss, paths_per_thread, event_mode)
    dev = torch.device(device)
    params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
    stats = torch.zeros((w.n_points, 8), dtype=torch.float64, device=dev)
    paths = torch.zeros((w.n_points * w.n_paths, BM_OUT_STRIDE), dtype=torch.float64, device=dev) if want_paths else None
    trace = (torch.zeros((trace_paths, trace_steps, 2), dtype=torch.float64, device=dev)
             if trace_steps and trace_paths else None)
    with torch.cuda.device(dev):
        bm_simulate(cfg, params, w.n_points, w.n_paths, w.n_steps, w.dt, w.seed, stats, paths, trace)
        torch.cuda.synchronize()
    return (stats.cpu().numpy(), paths.cpu().numpy() if paths is not None else None,
            trace.cpu().numpy() if trace is not None else None)
