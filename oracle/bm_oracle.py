"""ctypes front end of the fp64 CPU oracle (oracle/bm_oracle.c) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA package and shares no code with it.  Argument marshalling only: all arithmetic
of the method is in bm_oracle.c.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bm_oracle.c")
_HDR = os.path.join(_HERE, "bm_oracle.h")
_LIB = os.path.join(_HERE, "libbm_oracle.so")

OVERDAMPED, INERTIAL = 0, 1
POT_SINE2, POT_PWL, POT_QUAD = 0, 1, 2
SCHEME_JUMP_ADAPTED, SCHEME_PAPER_LITERAL, SCHEME_ADAPTIVE = 0, 1, 2
OUT_XT, OUT_VT, OUT_VBAR, OUT_JUMPS, OUT_SUBSTEPS, OUT_XTI, OUT_STRIDE = 0, 1, 2, 3, 4, 5, 6

PARAM_FIELDS = ("A1", "A2", "F", "D", "lambda_", "zeta", "Fa", "Fb", "mu_a", "mu_b", "gamma", "amp", "omega",
                "x0_fixed", "v0_lo", "v0_hi")


class OrcParams(C.Structure):
    _fields_ = [(n, C.c_double) for n in PARAM_FIELDS]


class OrcConfig(C.Structure):
    _fields_ = [("model", C.c_int32), ("potential", C.c_int32), ("scheme", C.c_int32), ("reserved", C.c_int32),
                ("n_discard", C.c_int64), ("adapt_tol", C.c_double), ("adapt_levels", C.c_int32), ("reserved2", C.c_int32)]


class OrcStats(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("n", "mean_v", "var_v", "mean_xT", "var_xT", "mean_jumps", "mean_substeps", "rsv")]


def build(force=False):
    """Compile the oracle with gcc (-O2, no fast-math, OpenMP).  Building the checker is not using it."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(_HDR))):
        return _LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _LIB, _SRC, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u32p = C.POINTER(C.c_uint32)
        dp = C.POINTER(C.c_double)
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.orc_philox_call.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, u32p]
        L.orc_u01.argtypes = [C.c_uint32]
        L.orc_u01.restype = C.c_double
        L.orc_gauss_block.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, dp]
        L.orc_gauss.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64]
        L.orc_gauss.restype = C.c_double
        L.orc_drift.argtypes = [C.POINTER(OrcParams), C.c_int, C.c_double, C.c_int]
        L.orc_drift.restype = C.c_double
        L.orc_minus_dV.argtypes = [C.POINTER(OrcParams), C.c_int, C.c_double]
        L.orc_minus_dV.restype = C.c_double
        L.orc_substep_overdamped.argtypes = [C.POINTER(OrcParams), C.c_int, C.c_int, C.c_double, C.c_double,
                                             C.c_double, dp]
        L.orc_substep_overdamped.restype = C.c_double
        L.orc_substep_inertial.argtypes = [C.POINTER(OrcParams), C.c_int, C.c_int, C.c_double, C.c_double,
                                           C.c_double, dp]
        L.orc_simulate.argtypes = [C.POINTER(OrcConfig), C.POINTER(OrcParams), C.c_int32, C.c_int64, C.c_int64,
                                   C.c_double, C.c_uint64, C.POINTER(C.c_int64), C.c_int64, dp, dp, C.c_int64,
                                   C.c_int64, C.c_int32]
        L.orc_simulate.restype = C.c_int
        L.orc_reduce.argtypes = [dp, C.c_int64, C.POINTER(OrcStats)]
        L.orc_threads_used.restype = C.c_int
        _lib = L
    return _lib


def make_params(**kw):
    """One parameter point; unspecified fields are 0 except x0_fixed = -1 (random x0)."""
    p = OrcParams()
    p.x0_fixed = -1.0
    for k, v in kw.items():
        k = "lambda_" if k == "lambda" else k
        if k not in PARAM_FIELDS:
            raise KeyError(k)
        setattr(p, k, float(v))
    return p


def params_array(rows):
    """rows: iterable of dicts (field -> value) or an (n,16) float array -> ctypes array of OrcParams."""
    if isinstance(rows, np.ndarray):
        rows = np.ascontiguousarray(rows, dtype=np.float64)
        assert rows.ndim == 2 and rows.shape[1] == 16
        arr = (OrcParams * rows.shape[0])()
        C.memmove(arr, rows.ctypes.data, rows.nbytes)
        return arr
    rows = list(rows)
    arr = (OrcParams * len(rows))()
    for i, r in enumerate(rows):
        arr[i] = r if isinstance(r, OrcParams) else make_params(**r)
    return arr


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def philox_call(seed, g, stream, idx):
    o = (C.c_uint32 * 4)()
    lib().orc_philox_call(seed, g, stream, idx, o)
    return tuple(int(x) for x in o)


def philox_fill(seed, path0, n_paths, stream, idx0, n_idx):
    """Words of calls (g = path0..path0+n_paths-1) x (idx = idx0..idx0+n_idx-1): uint32 [n_paths][n_idx][4]."""
    out = np.empty((n_paths, n_idx, 4), dtype=np.uint32)
    o = (C.c_uint32 * 4)()
    f = lib().orc_philox_call
    for i in range(n_paths):
        for j in range(n_idx):
            f(seed, path0 + i, stream, (idx0 + j) & 0xFFFFFFFF, o)
            out[i, j, :] = o[:]
    return out


def u01(w):
    return lib().orc_u01(int(w))


def gauss_block(seed, g, b):
    o = (C.c_double * 4)()
    lib().orc_gauss_block(seed, g, b, o)
    return tuple(o)


def gauss(seed, g, m):
    return lib().orc_gauss(seed, g, m)


def drift(p, potential, xi, d=-1):
    return lib().orc_drift(C.byref(p), potential, xi, d)


def substep_overdamped(p, potential, d, x, h, g):
    st = (C.c_double * 5)()
    xn = lib().orc_substep_overdamped(C.byref(p), potential, d, x, h, g, st)
    return xn, tuple(st)


def substep_inertial(p, potential, d, t, h, g, x, v):
    xv = (C.c_double * 2)(x, v)
    lib().orc_substep_inertial(C.byref(p), potential, d, t, h, g, xv)
    return xv[0], xv[1]


def simulate(params, n_paths, n_steps, dt, seed, *, model=OVERDAMPED, potential=POT_SINE2,
             scheme=SCHEME_JUMP_ADAPTED, n_discard=0, ids=None, trace_paths=0, trace_steps=0, threads=0,
             adapt_tol=float("inf"), adapt_levels=0):
    """Run the oracle.  Returns (paths[n][6] float64, trace or None).  ids: global path ids to run (default all)."""
    arr = params if isinstance(params, C.Array) else params_array(params)
    n_points = len(arr)
    cfg = OrcConfig(model, potential, scheme, 0, n_discard, adapt_tol, adapt_levels, 0)
    if ids is not None:
        ids = np.ascontiguousarray(ids, dtype=np.int64)
        n = ids.size
        idp = ids.ctypes.data_as(C.POINTER(C.c_int64))
    else:
        n = n_points * n_paths
        idp = None
    out = np.zeros((n, OUT_STRIDE), dtype=np.float64)
    trace = None
    trp = None
    if trace_paths > 0 and trace_steps > 0:
        trace_paths = min(trace_paths, n)
        trace = np.zeros((trace_paths, trace_steps, 2), dtype=np.float64)
        trp = trace.ctypes.data_as(C.POINTER(C.c_double))
    rc = lib().orc_simulate(C.byref(cfg), arr, n_points, n_paths, n_steps, dt, seed, idp, n,
                            out.ctypes.data_as(C.POINTER(C.c_double)), trp, trace_paths, trace_steps, threads)
    if rc != 0:
        raise ValueError(f"orc_simulate: invalid arguments (rc={rc})")
    return out, trace


def reduce(paths):
    paths = np.ascontiguousarray(paths, dtype=np.float64)
    st = OrcStats()
    lib().orc_reduce(paths.ctypes.data_as(C.POINTER(C.c_double)), paths.shape[0], C.byref(st))
    return {k: getattr(st, k) for k, _ in OrcStats._fields_}


def threads_used():
    return lib().orc_threads_used()


# ---- observables of the stationary state beyond <v> -------------------------
# Plain definitions written out on the oracle's per-path traces (x unfolded, v after every grid step; grid step index
# i = 1, 2, ... is time i*dt).  Test infrastructure like the rest of this module.

def deff_from_trace(trace, i0, i, dt):
    """Effective diffusion coefficient over [t_i0, t_i]: D_eff = Var_p[x_p(t_i) - x_p(t_i0)] / (2 (t_i - t_i0)), unbiased
    variance over the paths p (the spread of the ensemble grows as 2 D_eff t in the stationary state)."""
    dx = trace[:, i - 1, 0] - trace[:, i0 - 1, 0]
    return dx.var(ddof=1) / (2.0 * (i - i0) * dt)


def vacf_from_trace(trace, i0, i):
    """Velocity autocovariance C(t_i - t_i0) = <v(t_i0) v(t_i)> - <v(t_i0)><v(t_i)> over the paths (unbiased, n - 1)."""
    a, b = trace[:, i0 - 1, 1], trace[:, i - 1, 1]
    return ((a - a.mean()) * (b - b.mean())).sum() / (a.size - 1)


def hist_from_trace(trace_x, sample_steps, period, n_bins):
    """Stationary density p(x mod L) of eq. (19), as a histogram: counts of frac(x / L) over n_bins equal
    bins for the unfolded positions trace_x[path, step - 1] after the grid steps `sample_steps` (1-based)."""
    x = trace_x[:, np.asarray(sample_steps) - 1]
    u = x / period
    u = u - np.floor(u)
    b = np.minimum((u * n_bins).astype(np.int64), n_bins - 1)
    return np.bincount(b.ravel(), minlength=n_bins)
