#!/usr/bin/env python
"""bench.py -- path-steps/s of the hot path (bm_simulate) on B200, with the roofline and the oracle beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--workload C1] [--prec f32]

A "step" is ONE pass of the whole hot path over one batch of synthetic input: one bm_simulate call = path kernel
(a1-a10 of DESIGN.md section 2) + grid pass of the reduction (a11) for the full workload.  Default workload is
BASELINE.json configs[1] = C1 (65536 paths x 1e5 grid steps, overdamped ratchet + Poissonian + Gaussian noise),
the configuration the metric is quoted on; the headline value is fp32, the same workload in fp64 is reported in
`fp64`.  Inputs are synthetic (paper_1409_4923_b200/workloads.py, seeded); nothing is read from disk.

Timing: every step is bracketed by CUDA events on the stream the kernels are launched on; W >= 3 warm-up steps;
an L2 flush (256 MiB device write) runs between steps, outside the event pairs.  N > 1 = independent replicas
("replicas only", rank r uses seed + r); barrier + synchronize on both sides, max over ranks.
--impl reference times the fp64 CPU oracle (oracle/) on this box's host cores on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "path-steps/s"
UNIT = "path-steps/s"
# Algorithmic SFU-class operations per overdamped sub-step in fp32: 3 force cosines + one half
# of a Box-Muller pair (lg2, sqrt, sin, cos for two Gaussians) = 5; the inertial step adds the drive cosine = 6.
# A kick adds 2 lg2 (waiting time, amplitude), a flip 1; sub-steps and events are COUNTED by the kernel.
XU_OPS_PER_SUBSTEP = {0: 5.0, 1: 6.0}
XU_LANES_PER_SM = 16          # MUFU lanes per SM per clock (4 per SM sub-partition); confirmed by bm_pipe_probe
# dram__bytes_read.sum + dram__bytes_write.sum of one path-kernel launch from the committed `ncu --set full` captures
# (profiles/r2_f32_v7.md; C4: its CELLS and LANES launch together): parameters and per-block partials only, the path is
# register-resident.  Bytes per call.
# Each constant is tied to the kernel it was captured from by that kernel's registers per thread (bm_kernel_info): when the
# kernel bm_simulate launches today no longer has that count, the capture is stale and `traffic` is reported as null.
NCU_DRAM_BYTES = {("C1", "f32"): (64512, 84), ("C2", "f32"): (53760, 87), ("C3", "f32"): (86272, 87),
                  ("C4", "f32"): (4351488, 64)}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C1", choices=["C0", "C1", "C2", "C3", "C4", "M1", "M2", "A1"])
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"])
    ap.add_argument("--sincos", default="auto", choices=["auto", "sfu", "fma"])
    ap.add_argument("--block-threads", type=int, default=0)
    ap.add_argument("--gauss", default="auto", choices=["auto", "w32", "w16", "w16p"],
                    help="fp32: Philox words per Box-Muller pair (bm_gauss)")
    ap.add_argument("--paths-per-thread", type=int, default=0, choices=[0, 1, 2],
                    help="fp64: realizations per thread (bm_config.paths_per_thread; 0 = library default)")
    ap.add_argument("--scale-steps", type=float, default=1.0, help="shrink n_steps (profiling runs only; flagged)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fp64", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block of the default run")
    ap.add_argument("--probe-pipes", action="store_true",
                    help="measure the SM's pipe throughputs with bm_pipe_probe and print them as one JSON object")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


def workload_of(args):
    from paper_1409_4923_b200 import workloads as W
    w = W.CONFIGS[args.workload]()
    if args.scale_steps != 1.0:
        w = w.scaled(n_steps=max(8, int(w.n_steps * args.scale_steps)))
    return w


def workload_config(w, args, extra=None):
    c = {"workload": f"{w.name}: BASELINE.json configs[{w.name[1]}]" if (w.name[0] == "C" and w.name[1:].isdigit()) else w.name,
         "n_points": int(w.n_points), "n_paths_per_point": int(w.n_paths), "n_steps": int(w.n_steps),
         "dt": w.dt, "n_discard": int(w.n_discard), "seed": int(w.seed),
         "model": "inertial" if w.model == 1 else "overdamped",
         "l2": "inputs are 128 B/point of parameters (compute-bound path); 256 MiB L2 flush between steps, "
               "outside the event pairs"}
    if args.scale_steps != 1.0:
        c["REDUCED"] = f"n_steps scaled by {args.scale_steps} (profiling run, not a bench value)"
    if extra:
        c.update(extra)
    return c


# ---- clocks sampled DURING the timed region ------------------------------------------------------------------

class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc, self.thr = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thr = threading.Thread(target=self._read, daemon=True)
        self.thr.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        inside = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        for r in inside:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ---- the oracle, timed as it stands (cpu_baseline leg and --impl reference) -----------------------------------

def oracle_time_sample(w, n_sample_paths, threads=0):
    """Oracle on the first n_sample_paths global paths of w at full length; returns seconds."""
    from oracle import bm_oracle as orc
    ids = np.arange(n_sample_paths, dtype=np.int64)
    t0 = time.perf_counter()
    orc.simulate(w.params, w.n_paths, w.n_steps, w.dt, w.seed, model=w.model, potential=w.potential,
                 scheme=w.scheme, n_discard=w.n_discard, ids=ids, threads=threads)
    return time.perf_counter() - t0


def oracle_sample_size(w, target_seconds):
    """Calibrate on 2 paths per core, then size the sample for ~target_seconds of wall time."""
    from oracle import bm_oracle as orc
    orc.lib()
    cores = os.cpu_count() or 1
    total = w.n_points * w.n_paths
    n_cal = min(total, 2 * cores)
    t = oracle_time_sample(w, n_cal)
    per_path = max(t / n_cal, 1e-9)
    n = int(target_seconds / per_path)
    n = max(cores, (n // cores) * cores)
    return min(n, total), orc.threads_used() or cores


def cpu_baseline(w, target_seconds):
    """The oracle as it stands on a bounded sample (about target_seconds of wall time on all host cores)."""
    from oracle import bm_oracle as orc
    n, cores = oracle_sample_size(w, target_seconds)
    t = oracle_time_sample(w, n)
    total = w.n_points * w.n_paths
    if t < 0.7 * target_seconds and n < total:      # the two-paths-per-core calibration overestimates the cost
        n = min(total, max(cores, int(n * target_seconds / max(t, 1e-3)) // cores * cores))
        t = oracle_time_sample(w, n)
    used = int(orc.threads_used() or cores)
    # one core, as the paper's own comparison: a sample of about a third of the time
    n1 = max(1, int(n / max(used, 1) / 3))
    t1 = oracle_time_sample(w, n1, threads=1)
    return {"value": n * w.n_steps / t, "unit": UNIT, "cores": used, "kind": "oracle",
            "sample": f"first {n} of {total} paths of {w.name} at full length "
                      f"({w.n_steps} grid steps), fp64, gcc -O2 + OpenMP, {t:.1f} s",
            "value_1core": n1 * w.n_steps / t1,
            "sample_1core": f"first {n1} paths of {w.name} at full length on one thread, {t1:.1f} s (PAPER.md:437 compares "
                            "with one CPU core)"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = workload_of(args)
    per_step = max(1.0, min(args.cpu_seconds, 150.0 / max(1, args.steps + args.warmup)))
    n, cores = oracle_sample_size(w, per_step)
    for _ in range(args.warmup):
        oracle_time_sample(w, n)
    ts = [oracle_time_sample(w, n) for _ in range(args.steps)]
    from oracle import bm_oracle as orc
    cores = int(orc.threads_used() or cores)
    t = sum(ts) / len(ts)
    value = n * w.n_steps / t
    sample = f"each step = first {n} of {w.n_points * w.n_paths} paths of {w.name} at full length ({w.n_steps} grid steps)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, args, {"sample": sample}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---- our arm ---------------------------------------------------------------------------------------------------

def sincos_of(B, name):
    return {"auto": B.BM_SINCOS_AUTO, "sfu": B.BM_SINCOS_SFU, "fma": B.BM_SINCOS_FMA}[name]


class Runner:
    """Device buffers of one workload + the event-timed bm_simulate call (marshalling only)."""

    def __init__(self, B, torch, w, prec, sincos, block_threads, seed, dev, stream, gauss=0, paths_per_thread=0):
        self.B, self.torch, self.w, self.seed, self.stream, self.dev = B, torch, w, seed, stream, dev
        self.cfg = B.config_for(w, prec, sincos, block_threads, gauss=gauss,
                                paths_per_thread=paths_per_thread if (prec == B.BM_F64 and w.scheme == 0 and w.potential == 0) else 0)
        self.params = torch.from_numpy(np.ascontiguousarray(w.params)).to(dev)
        self.stats = torch.zeros((w.n_points, 8), dtype=torch.float64, device=dev)
        self.ws = torch.empty(max(16, B.bm_workspace_bytes(self.cfg, w.n_points, w.n_paths)), dtype=torch.uint8,
                              device=dev)
        # e2e: pinned host buffers, copied every step inside the timed region by bm_simulate_host
        self.h_params = torch.from_numpy(np.ascontiguousarray(w.params)).pin_memory()
        self.h_stats = torch.zeros((w.n_points, 8), dtype=torch.float64).pin_memory()

    def device_step(self):
        """One step with inputs resident in HBM; returns milliseconds (CUDA events on the launching stream)."""
        t = self.torch
        e0, e1 = t.cuda.Event(enable_timing=True), t.cuda.Event(enable_timing=True)
        with t.cuda.stream(self.stream):
            e0.record(self.stream)
            self.B.bm_simulate(self.cfg, self.params, self.w.n_points, self.w.n_paths, self.w.n_steps, self.w.dt,
                               self.seed, self.stats, workspace=self.ws, stream=self.stream)
            e1.record(self.stream)
        e1.synchronize()
        return e0.elapsed_time(e1)

    def host_step(self):
        """One step through the HOST-pointer entry: H2D of params, kernels, D2H of stats inside the timed region."""
        t = self.torch
        e0, e1 = t.cuda.Event(enable_timing=True), t.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(self.stream)
        self.B.bm_simulate_host(self.cfg, self.h_params, self.w.n_points, self.w.n_paths, self.w.n_steps, self.w.dt,
                                self.seed, self.h_stats, stream=self.stream)
        e1.record(self.stream)
        e1.synchronize()
        return max(e0.elapsed_time(e1), 1e3 * (time.perf_counter() - t0))


# ALGORITHMIC FP64 operations (add, multiply or fused multiply-add = 1) per sub-step, counted from the formulae of the
# method at the accuracy the 1e-8 per-path parity needs ("fp64 operation count"), not from the
# compiled kernel: the count the fp64 roofline fraction `frac` is formed with.
#   force a(x): cos 2 pi x = 5 (reduction, r^2, r^4) + 11 (degree-12 even polynomial, two chains) + 1 (join) = 17, then
#               c (k1 + k2 c) + const = 2                                          -> 19, three per sub-step = 57, + 1 for const
#   one normal = half a Box-Muller pair: (2 x 2 uniforms + 18 ln + 1 + 7 sqrt + 19 sincospi + 1 + 2 products) / 2  = 26
#   over-damped update lines of Alg. 1 (h/2 once, three lines, amp * g)                                            = 10
#   inertial: update lines of x and v = 21, ONE new drive cosine per sub-step (the one at t is the previous sub-step's
#             at t + h): 21 + omega t, t + h, amp * cos = 24
# Not counted: the jump scheduler's comparisons, the fold, conversions, selects -- whatever the compiler or the chosen
# code shape adds.  over-damped 57 + 1 + 10 + 26 = 94, inertial 57 + 1 + 21 + 24 + 26 = 129.
FP64_ALG_OPS_PER_SUBSTEP = {0: 94.0, 1: 129.0}
# FP64-pipe instructions (DFMA, DMUL, DADD, DSETP) per sub-step EXECUTED by the kernels as built, from the committed
# `ncu --set full` captures (profiles/r2_f64_v2.md), each with the registers per thread of the kernel it was counted on:
# reported as `pipe_utilisation` (how busy the FP64 pipe is, whatever it is busy with), null when the kernel has changed.
FP64_BUILT_OPS_PER_SUBSTEP = {0: (110.9, 120), 1: (175.7, 128)}
FP64_LANES_PER_SM = 64        # DFMA lanes per SM per clock (bm_pipe_probe: 63)


def launches_per_call(B, w, prec_name):
    """Kernels one bm_simulate call launches: the path kernel and the grid pass of the reduction; the fp32 over-damped
    jump-adapted kernel with a jump source on is launched in both of its forms (CELLS, LANES) on the same grid."""
    from paper_1409_4923_b200 import workloads as W
    two_forms = (prec_name == "f32" and w.model == W.OVERDAMPED and w.scheme == W.SCHEME_JUMP_ADAPTED
                 and (B.noise_mask(w.params) & 6) != 0)
    return 3 if two_forms else 2


def roofline_of(B, w, prec_name, stats, ms_per_step, clocks, info):
    """Roofline of the path kernel (the grid pass is < 0.1 % of a step), in ALGORITHMIC operations of the binding pipe:
    fp32: MUFU-class operations on the XU pipe; fp64: FP64 operations of the method's formulae (FP64_ALG_OPS_PER_SUBSTEP).
    Peak = lanes x SMs x the SM clock SAMPLED during the timed region (the maximum clock when nvidia-smi gave nothing).
    fp64 also carries `pipe_utilisation`: the same fraction formed with the instructions the kernel as built executes."""
    substeps = float(stats[:, 6].mean())                # counted by the kernel
    jumps = float(stats[:, 5].mean())
    sm_mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965.0
    extra = {}
    if prec_name == "f32":
        per_path = XU_OPS_PER_SUBSTEP[w.model] * substeps + 2.0 * jumps
        if w.scheme == 1:   # the paper's scheme as printed: no Gaussian transcendental; 3 force cosines only for SINE2
            per_path = (3.0 if w.potential == 0 else 0.0) * substeps + 2.0 * jumps
        lanes, pipe = XU_LANES_PER_SM, "xu (MUFU)"
        what = "algorithmic MUFU-class operations (DESIGN.md section 6)"
    else:
        per_path = FP64_ALG_OPS_PER_SUBSTEP[w.model] * substeps
        lanes, pipe = FP64_LANES_PER_SM, "fp64"
        what = "algorithmic FP64 operations of the method's formulae (DESIGN.md section 6, fp64 operation count)"
    ops = per_path * w.n_points * w.n_paths
    peak = lanes * info["sm_count"] * sm_mhz * 1e6 / 1e9
    achieved = ops / (ms_per_step * 1e-3) / 1e9
    if prec_name == "f64":
        built, regs = FP64_BUILT_OPS_PER_SUBSTEP[w.model]
        fresh = w.scheme == 0 and info["regs_per_thread"] == regs
        extra = {"pipe_utilisation": (built * substeps * w.n_points * w.n_paths / (ms_per_step * 1e-3) / 1e9 / peak) if fresh else None,
                 "pipe_utilisation_source": f"{built} executed FP64-pipe instructions per sub-step (profiles/r2_f64_v2.md, kernel with "
                                            f"{regs} registers per thread)" + ("" if fresh else "; the kernel launched now differs: stale")}
    return {"bound": "alu", "pipe": pipe, "achieved": achieved, "peak": peak, "unit": "Gop/s", "frac": achieved / peak,
            "ops_per_path_step": per_path / w.n_steps, "ops_counted": what,
            "peak_source": f"derived: {lanes} lanes/SM/clk x {info['sm_count']} SMs x {sm_mhz:.0f} MHz (SM clock sampled "
                           "during the timed region; lane counts confirmed by bm_pipe_probe, profiles/pipes_r2.json)",
            "kernel_ms": ms_per_step, "regs_per_thread": info["regs_per_thread"],
            "launch_threads": info["launch_threads"], "blocks_per_sm": info["blocks_per_sm"],
            "substeps_per_step": substeps / w.n_steps, **extra}


def traffic_of(w, prec_name, info, scale_steps=1.0):
    """dram bytes of one launch from the committed ncu capture, or None when that capture is of another kernel."""
    rec = NCU_DRAM_BYTES.get((w.name, prec_name))
    if rec is None or scale_steps != 1.0 or info["regs_per_thread"] != rec[1]:
        return None
    return rec[0]


def measure(B, torch, w, prec_name, args, seed, dev, stream, flush, steps, warmup, barrier, sampler_index, sincos=0, gauss=0,
            block_threads=0, paths_per_thread=0):
    """W warm-up steps, then K timed steps of one workload (CUDA events on the launching stream, L2 flush between
    steps outside the event pairs, clocks sampled during the timed region).  Returns (Runner, ms list, clocks, stats)."""
    prec = B.BM_F32 if prec_name == "f32" else B.BM_F64
    run = Runner(B, torch, w, prec, sincos, block_threads, seed, dev, stream, gauss, paths_per_thread)
    for _ in range(max(warmup, 0)):
        run.device_step()
    sampler = ClockSampler(sampler_index)
    sampler.start()
    time.sleep(0.25)
    barrier()
    t0 = time.time()
    ms = []
    for _ in range(steps):
        flush.zero_()                                   # L2 flush, outside the event pair
        torch.cuda.synchronize(dev)
        ms.append(run.device_step())
    barrier()
    t1 = time.time()
    if t1 - t0 < 0.3:                                   # give nvidia-smi (20 ms period) something to sample under load
        t_hold = time.time()
        while time.time() - t_hold < 0.3:
            run.device_step()
        torch.cuda.synchronize(dev)
        t1 = time.time()
    clocks = sampler.stop(t0, t1)
    return run, ms, clocks, run.stats.cpu().numpy().copy()


# every kernel family the library ships, timed in the default run: the five BASELINE.json configs in fp32, C1 / C2 in
# fp64, the paper's own programs (scheme as printed) and the adaptive scheme (row f4) on C1's physics
PER_CONFIG = (("C0", "f32"), ("C2", "f32"), ("C3", "f32"), ("C4", "f32"), ("C1", "f64"), ("C2", "f64"), ("M1", "f32"),
              ("M2", "f32"), ("A1", "f64"))


def run_ours(args):
    import torch
    from paper_1409_4923_b200 import binding as B, workloads as W
    B.lib()                                             # raises when libbm.so is missing: there is no fallback
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product has no CPU path)")
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    stream = torch.cuda.Stream(device=dev)
    w = workload_of(args)
    sc = sincos_of(B, args.sincos)
    gs = {"auto": B.BM_GAUSS_AUTO, "w32": B.BM_GAUSS_W32, "w16": B.BM_GAUSS_W16, "w16p": B.BM_GAUSS_W16P}[args.gauss]
    from paper_1409_4923_b200 import replicas
    seed = replicas.replica_seed(w.seed, rank)          # replicas only: independent ensembles, no collective
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    run, ms, clocks, stats = measure(B, torch, w, args.prec, args, seed, dev, stream, flush, args.steps, args.warmup, barrier,
                                     local_rank, sc, gs, args.block_threads, args.paths_per_thread)
    info = B.bm_kernel_info(run.cfg, w.n_points, w.n_paths)
    total_ms = replicas.max_over_ranks(float(sum(ms)), dist, dev)   # timing plumbing only (max over ranks)
    ms_per_step = total_ms / args.steps
    value = replicas.whole_job_value(w.path_steps, world, ms_per_step)

    # e2e: same metric through the HOST-pointer C-ABI call (copies inside the timed region)
    run.host_step()
    barrier()
    e2e_ms = [run.host_step() for _ in range(max(2, min(args.steps, 5)))]
    e2e_total = replicas.max_over_ranks(float(np.mean(e2e_ms)), dist, dev)
    e2e = {"value": replicas.whole_job_value(w.path_steps, world, e2e_total), "unit": UNIT,
           "h2d_bytes_per_step": int(run.h_params.numel() * 8), "d2h_bytes_per_step": int(run.h_stats.numel() * 8),
           "ms_per_step": e2e_total, "call": "bm_simulate_host (stream-ordered alloc + H2D + kernels + D2H + sync per call)"}
    if world == 1 and not np.array_equal(run.h_stats.numpy(), stats):
        raise SystemExit("bench.py: host-pointer call and device-pointer call disagree (determinism contract broken)")

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    roof = roofline_of(B, w, args.prec, stats, ms_per_step, clocks, info)
    # the XU peak measured live with the library's probe kernel (8 independent MUFU chains per thread), beside the
    # derived one: lane-operations per second of MUFU.COS on this device at its current clocks
    sink = torch.zeros(info["sm_count"] * 4 * 256, dtype=torch.float32, device=dev)
    probe_ms = []
    for r in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        B.bm_pipe_probe(B.BM_PROBE_MUFU_COS if args.prec == "f32" else B.BM_PROBE_DFMA, 1000, info["sm_count"] * 4, 256, sink)
        e1.record()
        e1.synchronize()
        probe_ms.append(e0.elapsed_time(e1))
    roof["peak_probe"] = info["sm_count"] * 4 * 256 * 1000 * 64 / (min(probe_ms) * 1e-3) / 1e9
    roof["frac_of_probe"] = roof["achieved"] / roof["peak_probe"]
    roof["traffic"] = traffic_of(w, args.prec, info, args.scale_steps)
    roof["traffic_source"] = ("a constant from the committed ncu --set full capture of this kernel (profiles/, dram bytes of "
                              "one launch: parameters and per-block partials; independent of n_steps), not read in this run; null when "
                              "the kernel launched now has another register count than the captured one")
    roof["kernel"] = "bm_paths_literal" if w.scheme == 1 else ("bm_paths_f32" if args.prec == "f32" else "bm_paths_f64")
    roof["gauss"] = {1: "w32", 2: "w16", 3: "w16p"}.get(info["gauss"], "n/a")
    jumps = float(stats[:, 5].mean())
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": args.prec, "data": "synthetic",
            "config": workload_config(w, args, {"parallelism": "replicas only" if world > 1 else "single GPU",
                                                "sincos": args.sincos, "substeps_per_step": roof["substeps_per_step"]}),
            "ms_median": float(np.median(ms)), "ms_best": float(min(ms)),
            "substeps_per_s": world * roof["substeps_per_step"] * w.path_steps / (ms_per_step * 1e-3),
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_call(B, w, args.prec) * args.steps, "roofline": roof,
            "result": {"mean_v": float(stats[0, 1]), "var_v": float(stats[0, 2]), "mean_jumps": jumps}}

    # every BASELINE.json config, both precisions and every other kernel family beside the headline (3 warm-up + 3 timed
    # full-size steps each), compactly INSIDE the roofline object
    if world == 1 and not args.no_per_config and args.scale_steps == 1.0 and args.workload == "C1" and args.prec == "f32":
        def compact(name, pn, wc, mps, best, rf, ck):
            meaningful = not (pn == "f32" and wc.scheme == 1 and wc.potential != 0)   # PWL as printed: no MUFU in the step
            return {"ms": round(mps, 4), "ms_best": round(best, 4), "value": wc.path_steps / (mps * 1e-3),
                    "frac": round(rf["frac"], 4) if meaningful else None,
                    "pipe_utilisation": (round(rf["pipe_utilisation"], 4) if rf.get("pipe_utilisation") else None) if pn == "f64" else None,
                    "ops_per_path_step": round(rf["ops_per_path_step"], 4), "substeps_per_step": round(rf["substeps_per_step"], 5),
                    "regs": rf["regs_per_thread"], "threads": rf["launch_threads"],
                    "sm_mhz": ck.get("sm_mhz"), "reasons": ck.get("reasons", [])}
        per = {"C1_f32": compact("C1", "f32", w, ms_per_step, float(min(ms)), roof, clocks)}
        launches = 0
        for name, pn in PER_CONFIG:
            wc = W.CONFIGS[name]()
            r2, ms2, ck2, st2 = measure(B, torch, wc, pn, args, wc.seed, dev, stream, flush, 3, 3, barrier, local_rank)
            i2 = B.bm_kernel_info(r2.cfg, wc.n_points, wc.n_paths)
            mps = float(np.mean(ms2))
            rf = roofline_of(B, wc, pn, st2, mps, ck2, i2)
            per[f"{name}_{pn}"] = compact(name, pn, wc, mps, float(min(ms2)), rf, ck2)
            launches += launches_per_call(B, wc, pn) * 3
            del r2
        roof["per_config"] = per
        line["gpu_launches"] += launches
        line["fp64"] = {"value": per["C1_f64"]["value"], "unit": UNIT, "ms_per_step": per["C1_f64"]["ms"],
                        "frac": per["C1_f64"]["frac"], "pipe_utilisation": per["C1_f64"]["pipe_utilisation"]}
    elif world == 1 and not args.no_fp64 and args.prec == "f32":
        r64 = Runner(B, torch, w, B.BM_F64, sc, args.block_threads, seed, dev, stream)
        r64.device_step()
        m64 = [r64.device_step() for _ in range(3)]
        line["fp64"] = {"value": w.path_steps / (float(np.mean(m64)) * 1e-3), "unit": UNIT, "ms_per_step": float(np.mean(m64)),
                        "mean_v": float(r64.stats.cpu().numpy()[0, 1])}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w, args.cpu_seconds)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def probe_pipes():
    """Throughput of the SM's arithmetic pipes measured with the library's probe kernels (bm_pipe_probe): warp
    instructions of one kind, 8 independent chains per thread, 4 blocks of 256 threads per SM.  Printed as
    lane-operations per SM and clock at the SM clock sampled during the probes (profiles/pipes_r2.json)."""
    import torch
    from paper_1409_4923_b200 import binding as B
    dev = torch.device("cuda", 0)
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    names = {B.BM_PROBE_FFMA: "FFMA", B.BM_PROBE_MUFU_COS: "MUFU.COS", B.BM_PROBE_MUFU_LG2: "MUFU.LG2",
             B.BM_PROBE_MUFU_SQRT: "MUFU.SQRT", B.BM_PROBE_IMAD_WIDE: "IMAD.WIDE.U32", B.BM_PROBE_LOP3: "LOP3",
             B.BM_PROBE_DFMA: "DFMA", B.BM_PROBE_I2F: "I2F", B.BM_PROBE_FADD: "FADD", B.BM_PROBE_MIX: "MUFU+IMAD.WIDE mix"}
    sink = torch.zeros(sms * 4 * 256, dtype=torch.float32, device=dev)
    iters = 2000
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.25)
    t0 = time.time()
    best = {}
    for op, nm in names.items():
        for rep in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            B.bm_pipe_probe(op, iters, sms * 4, 256, sink)
            e1.record()
            e1.synchronize()
            if rep:
                best[nm] = min(best.get(nm, 1e30), e0.elapsed_time(e1))
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    mhz = clocks.get("sm_mhz") or 1965.0
    ops = sms * 4 * 256 * iters * 64
    table = {nm: {"ms": ms, "Gop_per_s": ops / (ms * 1e-3) / 1e9,
                  "lane_ops_per_sm_per_clk": ops / (ms * 1e-3) / (sms * mhz * 1e6),
                  "cycles_per_warp_instr_per_subpartition": 32.0 / (ops / (ms * 1e-3) / (sms * mhz * 1e6) / 4.0)}
             for nm, ms in best.items()}
    print(json.dumps({"what": "bm_pipe_probe throughputs", "gpu": torch.cuda.get_device_name(dev), "sm_count": sms,
                      "launch": f"{sms * 4} blocks x 256 threads x {iters} x 64 operations per thread", "clocks": clocks,
                      "pipes": table}, indent=1))
    return 0


def main():
    args = parse()
    if args.probe_pipes:
        return probe_pipes()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
