"""GPU test of bm_simulate_static, the entry point for callers that cannot allocate device memory.

Who needs it: code that runs where no allocator may be called -- a plug-in inside an application that owns the GPU heap,
a real-time loop in which cudaMalloc is forbidden (it may synchronise the device and has no time bound), a process whose
device memory is already committed.  bm_simulate makes such a caller bring a workspace; bm_simulate_static keeps the
scratch of the ensemble reduction in a fixed 4 MiB array inside libbm.so instead and allocates nothing.

What is checked: on two calls in a row (a wide launch first, then a narrow one that leaves most of the first call's
partial sums lying in the shared array, then the wide one again) the statistics, per-path records and trace are equal
BIT FOR BIT to those of bm_simulate with a caller-owned workspace -- the tolerance of this repository's determinism
tests, and the strictest one available: both entries launch the same kernels with the same reduction tree.  Also: the
size limit is enforced with BM_ERR_WORKSPACE, and the free device memory does not move across calls.

This file sorts last on purpose (pytest -x stops at the first failure, and this entry point is an add-on: a failure
here must not hide the parity tests).  It passes alone in a fresh process and after the rest of the suite.
"""
import ctypes as C

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


class Case:
    """One workload with every device buffer of both entry points allocated up front (by the test, through torch)."""

    def __init__(self, B, w, prec, trace=0):
        import torch
        self.B, self.w = B, w
        self.cfg = B.config_for(w, prec, trace_steps=trace, trace_paths=trace and min(8, w.n_paths))
        dev = torch.device("cuda:0")
        self.params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
        n = w.n_points * w.n_paths

        def outputs():
            # filled with a pattern, so that an output the call failed to write cannot compare equal by accident
            return (torch.full((w.n_points, 8), -7.0, dtype=torch.float64, device=dev),
                    torch.full((n, B.BM_OUT_STRIDE), -7.0, dtype=torch.float64, device=dev),
                    torch.full((self.cfg.trace_paths, trace, 2), -7.0, dtype=torch.float64, device=dev) if trace else None)
        self.ref, self.got = outputs(), outputs()
        self.workspace = torch.empty(max(B.bm_workspace_bytes(self.cfg, w.n_points, w.n_paths), 16), dtype=torch.uint8,
                                     device=dev)

    def run_reference(self):
        w = self.w
        self.B.bm_simulate(self.cfg, self.params, w.n_points, w.n_paths, w.n_steps, w.dt, w.seed, *self.ref,
                           workspace=self.workspace)

    def run_static(self):
        w = self.w
        for t in self.got:
            if t is not None:
                t.fill_(-7.0)
        self.B.bm_simulate_static(self.cfg, self.params, w.n_points, w.n_paths, w.n_steps, w.dt, w.seed, *self.got)

    def assert_equal(self, what):
        import torch
        torch.cuda.synchronize()
        for name, r, g in zip(("out_stats", "out_paths", "out_trace"), self.ref, self.got):
            if r is None:
                continue
            r, g = r.cpu().numpy(), g.cpu().numpy()
            assert not (r == -7.0).all(), f"{what}: the reference call left {name} unwritten"
            assert np.array_equal(r.view(np.uint64), g.view(np.uint64)), \
                f"{what}: {name} of bm_simulate_static differs from bm_simulate (max |diff| {np.nanmax(np.abs(r - g)):.3e})"


def make_cases(B):
    # wide: 48 points x 3 blocks of the fp32 kernel with kicks (both event forms launch) -- 144 slots of the shared array
    wide = Case(B, W.c4().scaled(n_paths=300, n_steps=400, points=list(range(0, 128 * 128, 345))[:48]), B.BM_F32)
    # narrow: one point, two blocks, fp64 with a trace -- reuses the first two slots, the other 142 hold stale sums
    narrow = Case(B, W.c1().scaled(n_paths=257, n_steps=300), B.BM_F64, trace=16)
    # the inertial model in fp32, ragged
    inertial = Case(B, W.c2().scaled(n_paths=129, n_steps=256), B.BM_F32)
    return wide, narrow, inertial


def test_static_scratch_matches_bm_simulate_on_consecutive_calls(B):
    import torch
    wide, narrow, inertial = make_cases(B)
    for c in (wide, narrow, inertial):
        c.run_reference()
    torch.cuda.synchronize()
    # calls in a row on one stream, no clearing of anything in between
    sequence = [("call 1 (wide)", wide), ("call 2 (narrow, after wide)", narrow), ("call 3 (wide again)", wide),
                ("call 4 (inertial)", inertial), ("call 5 (narrow again)", narrow)]
    for what, c in sequence:
        c.run_static()
        c.assert_equal(what)
    # back to back WITHOUT a synchronisation in between: same stream, so the second call's kernels queue behind the first
    wide.run_static()
    narrow.run_static()
    wide.assert_equal("unsynchronised pair, first")
    narrow.assert_equal("unsynchronised pair, second")


def test_static_scratch_allocates_nothing(B):
    """Free device memory is the same before and after calls (once the kernels are loaded by a first round)."""
    import torch
    wide, narrow, _ = make_cases(B)
    for c in (wide, narrow):          # first round: module / kernel loading and the one-off address look-up happen here
        c.run_static()
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        for c in (wide, narrow):
            c.run_static()
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, (free_before, free_after)


def test_static_scratch_rejects_oversized_launches(B):
    """More thread blocks than the fixed array has slots for: BM_ERR_WORKSPACE, nothing launched, outputs untouched."""
    import torch
    slots = B.BM_STATIC_SCRATCH_BYTES // 64
    assert slots == 65536
    cfg = B.make_config(prec=B.BM_F32, block_threads=128)
    L = B.lib()
    n_points = 512
    params = torch.from_numpy(np.ascontiguousarray(np.repeat(W.c1().params, n_points, axis=0))).cuda()
    stats = torch.full((n_points, 8), -7.0, dtype=torch.float64, device="cuda")

    def call(n_paths):
        return L.bm_simulate_static(C.byref(cfg), params.data_ptr(), n_points, n_paths, 8, 1e-3, 1, stats.data_ptr(), None,
                                    None, None)
    assert B.bm_workspace_bytes(cfg, n_points, 128 * 128) == B.BM_STATIC_SCRATCH_BYTES       # exactly full: accepted
    assert call(128 * 128) == B.BM_OK
    torch.cuda.synchronize()
    assert (stats.cpu().numpy()[:, 0] == 128 * 128).all()
    stats.fill_(-7.0)
    assert B.bm_workspace_bytes(cfg, n_points, 128 * 128 + 1) > B.BM_STATIC_SCRATCH_BYTES    # one block per point more
    assert call(128 * 128 + 1) == B.BM_ERR_WORKSPACE
    with pytest.raises(B.BmError) as e:
        B.bm_simulate_static(cfg, params, n_points, 128 * 128 + 1, 8, 1e-3, 1, stats)
    assert e.value.status == B.BM_ERR_WORKSPACE and "BM_ERR_WORKSPACE" in str(e.value)
    torch.cuda.synchronize()
    assert (stats.cpu().numpy() == -7.0).all()
    assert call(0) == B.BM_ERR_INVALID_ARG                                                   # bm_simulate's own checks still apply
