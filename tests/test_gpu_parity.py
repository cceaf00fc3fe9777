"""GPU parity tests: the CUDA path (through the C ABI / ctypes binding) against the fp64 CPU oracle on the same
seeded inputs.  Tolerances are BASELINE.json's:
  Philox words bit-exact; fp64 per-path x(T) |d| <= 1e-8 (1+|x|) on the overdamped configs; fp64 per-path state
  within 1e-10 relative over the first 1000 steps on the inertial configs; fp64 ensemble <v> within 1e-9 relative;
  fp32 ensemble <v> and variance within 3 combined standard errors of the fp64 oracle.
"""
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
    binding.lib()                     # raises if libbm.so is missing: no fallback
    return binding


from parity_util import assert_3se, assert_counts_close, assert_few_ill_conditioned, ill_conditioned, oracle_run  # noqa: E402


# ---- a3: Philox words -------------------------------------------------------------------------------------

@pytest.mark.parametrize("path0,stream,idx0", [(0, 0, 0), (0, 1, 0), (65530, 2, 7), (2 ** 32 - 3, 3, 2 ** 32 - 5),
                                                (67108860, 1, 24990), (2 ** 40 + 11, 1, 123456)])
def test_philox_words_bit_exact(B, orc, path0, stream, idx0):
    import torch
    n_paths, n_idx = 37, 9      # ragged: 333 calls, not a multiple of the block
    out = torch.zeros((n_paths, n_idx, 4), dtype=torch.int32, device="cuda")
    B.bm_philox_fill(W.SEED, path0, n_paths, stream, idx0, n_idx, out)
    got = out.cpu().numpy().view(np.uint32)
    exp = orc.philox_fill(W.SEED, path0, n_paths, stream, idx0, n_idx)
    assert np.array_equal(got, exp)


def test_philox_other_seed_high_bits(B, orc):
    import torch
    seed = (0xDEADBEEF << 32) | 0x12345678
    out = torch.zeros((64, 4, 4), dtype=torch.int32, device="cuda")
    B.bm_philox_fill(seed, 5, 64, 1, 0, 4, out)
    assert np.array_equal(out.cpu().numpy().view(np.uint32), orc.philox_fill(seed, 5, 64, 1, 0, 4))


# ---- a4: variate transforms -------------------------------------------------------------------------------

def test_gauss_f64_matches_oracle(B, orc):
    import torch
    n_paths, n_m = 33, 403      # ragged tail (403 = 100 blocks + 3)
    out = torch.zeros((n_paths, n_m), dtype=torch.float64, device="cuda")
    B.bm_gauss_fill(B.BM_F64, 0, W.SEED, 100, n_paths, 8, n_m, out)
    got = out.cpu().numpy()
    exp = np.array([[orc.gauss(W.SEED, 100 + p, 8 + j) for j in range(n_m)] for p in range(n_paths)])
    assert np.abs(got - exp).max() < 5e-15 * (1 + np.abs(exp).max())


def test_gauss_f32_w32_tracks_oracle_and_has_unit_moments(B, orc):
    import torch
    n_paths, n_m = 64, 4096
    out = torch.zeros((n_paths, n_m), dtype=torch.float32, device="cuda")
    B.bm_gauss_fill(B.BM_F32, B.BM_GAUSS_W32, W.SEED, 0, n_paths, 0, n_m, out)
    got = out.cpu().numpy().astype(np.float64)
    exp = np.array([[orc.gauss(W.SEED, p, j) for j in range(256)] for p in range(n_paths)])
    d = np.abs(got[:, :256] - exp)
    # same words, 23-bit uniforms and MUFU accuracy: typical error 1e-6, tails up to ~1e-3
    assert np.median(d) < 5e-6 and np.quantile(d, 0.999) < 2e-3
    n = got.size
    assert abs(got.mean()) < 4 / math.sqrt(n)
    assert abs(got.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs((got ** 4).mean() - 3) < 4 * math.sqrt(96 / n)


@pytest.mark.parametrize("gauss", ["W16", "W16P"])
def test_gauss_f32_w16_is_standard_normal(B, orc, gauss):
    """W16 / W16P (R13): eight normals per Philox call, radius from the top 23 bits and angle from the low 16 bits of one
    word.  Checked against what the mathematics fixes: moments up to order 6, independence of the two members of a
    pair and of neighbouring normals, Kolmogorov distance to Phi; and against the oracle's Philox words directly
    (the pair of word w is sqrt(-2 ln u) (cos, sin)(2 pi k/65536) with u, k read off w)."""
    import torch
    from scipy import stats as st
    n_paths, n_m = 256, 8192
    out = torch.zeros((n_paths, n_m), dtype=torch.float32, device="cuda")
    B.bm_gauss_fill(B.BM_F32, B.BM_GAUSS_W16P if gauss == "W16P" else B.BM_GAUSS_AUTO, W.SEED, 7, n_paths, 16, n_m, out)
    got = out.cpu().numpy().astype(np.float64)
    n = got.size
    assert abs(got.mean()) < 4 / math.sqrt(n)
    assert abs(got.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs((got ** 3).mean()) < 4 * math.sqrt(15 / n)
    assert abs((got ** 4).mean() - 3) < 4 * math.sqrt(96 / n)
    assert abs((got ** 6).mean() - 15) < 4 * math.sqrt((10395 - 225) / n)
    a, b = got[:, 0::2].ravel(), got[:, 1::2].ravel()          # the two members of each pair
    assert abs((a * b).mean()) < 4 / math.sqrt(a.size)
    assert abs((a * a * b * b).mean() - 1) < 4 * math.sqrt(8 / a.size)
    assert abs((got[:, 1:-1:2] * got[:, 2::2]).mean()) < 4 / math.sqrt(a.size)   # across pairs
    assert st.kstest(got.ravel()[::7], "norm").statistic < 1.63 / math.sqrt(n / 7)  # 1 % critical value
    # word by word: normals 8 b + 2 i, 8 b + 2 i + 1 of path g come from word i of Gaussian-stream call b
    for p in (0, 100):
        for b in (2, 500):
            w = orc.philox_call(W.SEED, 7 + p, 1, b)
            for i in range(4):
                u = ((int(w[i]) >> 9) + 1) * 2.0 ** -23
                ang = 2 * math.pi * (int(w[i]) & 0xFFFF) / 65536.0
                r = math.sqrt(-2 * math.log(u))
                j = 8 * (b - 2) + 2 * i
                assert abs(got[p, j] - r * math.cos(ang)) < 2e-5 * (1 + r)
                assert abs(got[p, j + 1] - r * math.sin(ang)) < 2e-5 * (1 + r)


@pytest.mark.parametrize("stream", [2, 3])
def test_event_normal_of_r13_word_by_word(B, orc, stream):
    """Reading R13: the sub-step that ends on event k of a jump stream takes its normal from word 2 of call k of THAT stream
    (radius from the top 23 bits, angle from the low 16).  No Gaussian-stream fill reaches that code; here the words of
    calls k = 0.. of the Poisson (2) and dichotomous (3) streams go through it: every normal against the definition, and
    the sample against the standard normal law (moments, KS) and against the kick amplitude drawn from word 1 of the same
    call (no correlation)."""
    import torch
    from scipy import stats as st
    n_paths, n_k = 512, 256
    raw = torch.zeros((n_paths, n_k, 4), dtype=torch.int32, device="cuda")
    B.bm_philox_fill(W.SEED, 3, n_paths, stream, 0, n_k, raw)
    words = raw[:, :, 2].contiguous().view(-1)
    out = torch.zeros(words.numel(), dtype=torch.float32, device="cuda")
    B.bm_event_normal_words(words, out)
    torch.cuda.synchronize()
    w = words.cpu().numpy().view(np.uint32).astype(np.int64)
    got = out.cpu().numpy().astype(np.float64)
    assert int(w.reshape(n_paths, n_k)[5, 7]) == orc.philox_call(W.SEED, 3 + 5, stream, 7)[2]            # the oracle's word
    u = ((w >> 9) + 1) * 2.0 ** -23
    r = np.sqrt(-2.0 * np.log(u))
    exp = r * np.cos(2 * math.pi * (w & 0xFFFF) / 65536.0)
    assert np.abs(got - exp).max() < 2e-5 * (1 + r.max()), np.abs(got - exp).max()
    assert np.all(np.abs(got - exp) < 2e-5 * (1 + r))
    n = got.size
    assert abs(got.mean()) < 4 / math.sqrt(n) and abs(got.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs((got ** 3).mean()) < 4 * math.sqrt(15 / n) and abs((got ** 4).mean() - 3) < 4 * math.sqrt(96 / n)
    assert st.kstest(got[::5], "norm").statistic < 1.63 / math.sqrt(n / 5)
    w1 = raw[:, :, 1].contiguous().view(-1).cpu().numpy().view(np.uint32).astype(np.float64)
    amp = -np.log((w1 + 0.5) / 4294967296.0)            # the kick amplitude / the other words of the same call
    assert abs(np.corrcoef(got, amp)[0, 1]) < 4 / math.sqrt(n)
    assert abs(np.corrcoef(got[:-1], got[1:])[0, 1]) < 4 / math.sqrt(n)


# ---- fp64 per-path parity, overdamped ---------------------------------------------------------------------

def check_fp64_overdamped(B, orc, w, ids=None, what="", ref=None):
    """fp64 per-path criterion |dx| <= 1e-8 (1 + |x|) with equal event and sub-step counts.  Paths beyond the bound are
    put through the A17 check (a second and third oracle run with x0 moved by +-1 ulp): only those whose
    ORACLE result itself moves by more than 1e-9 (1 + |x|) are ill-conditioned and excluded; their number is bounded
    (assert_few_ill_conditioned).  ref: the oracle's records for these paths, if the caller has them already.
    Returns (stats, paths, ref, bad = ids beyond the bound that are NOT ill-conditioned, dx)."""
    stats, paths, _ = B.run_workload(w, B.BM_F64, want_paths=True)
    if ref is None:
        ref, _ = oracle_run(orc, w, ids=ids)
    got = paths if ids is None else paths[ids]
    assert np.array_equal(got[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS]), what + ": event counts differ"
    assert np.array_equal(got[:, B.BM_OUT_SUBSTEPS], ref[:, orc.OUT_SUBSTEPS]), what + ": sub-step counts differ"
    dx = np.abs(got[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT])
    tol = 1e-8 * (1 + np.abs(ref[:, orc.OUT_XT]))
    over = np.nonzero(dx > tol)[0]
    bad = over
    if over.size:
        gids = over if ids is None else np.asarray(ids)[over]
        ill = ill_conditioned(orc, w, gids)
        assert_few_ill_conditioned(int(ill.sum()), got.shape[0], what)
        bad = over[~ill]
    return stats, paths, ref, bad, dx


def test_c0_fp64_full(B, orc):
    w = W.c0()
    stats, paths, ref, bad, dx = check_fp64_overdamped(B, orc, w, what="C0")
    assert bad.size == 0, f"C0: {bad.size} paths beyond 1e-8(1+|x|), max {dx.max():.3e}"
    o = orc.reduce(ref)
    assert abs(stats[0, 1] - o["mean_v"]) <= 1e-9 * abs(o["mean_v"]) + 1e-13     # <v> within 1e-9 relative
    assert abs(stats[0, 4] - o["var_xT"]) <= 1e-9 * o["var_xT"]
    assert abs(stats[0, 2] - o["var_v"]) <= 1e-9 * o["var_v"]
    assert stats[0, 0] == w.n_paths


def test_c1_fp64_scaled_full_compare(B, orc):
    w = W.c1().scaled(n_paths=1000, n_steps=5000)      # ragged: 1000 is not a multiple of the block size
    stats, paths, ref, bad, dx = check_fp64_overdamped(B, orc, w, what="C1 scaled")
    assert bad.size == 0, f"C1 scaled: {bad.size} paths beyond tolerance, max {dx.max():.3e}"
    o = orc.reduce(ref)
    assert abs(stats[0, 1] - o["mean_v"]) <= 1e-9 * abs(o["mean_v"])
    assert abs(stats[0, 5] - o["mean_jumps"]) < 1e-12 and abs(stats[0, 6] - o["mean_substeps"]) < 1e-9


def test_c1_fp64_full_size_all_paths(B, orc, c1_full_oracle):
    """Full C1 (65536 paths x 1e5 steps) on the GPU and in the oracle, every path compared; ensemble statistics of the
    on-device reduction against the oracle's two-pass reduction within 1e-9 relative."""
    w = W.c1()
    stats, paths, ref, bad, dx = check_fp64_overdamped(B, orc, w, what="C1 full", ref=c1_full_oracle)
    assert bad.size == 0, f"C1 full: {bad.size} well-conditioned paths beyond tolerance (max {dx[bad].max():.3e})"
    o = orc.reduce(ref)
    assert stats[0, 0] == w.n_paths
    assert abs(stats[0, 1] - o["mean_v"]) <= 1e-9 * abs(o["mean_v"])
    assert abs(stats[0, 2] - o["var_v"]) <= 1e-9 * o["var_v"]
    assert abs(stats[0, 3] - o["mean_xT"]) <= 1e-9 * abs(o["mean_xT"])
    assert abs(stats[0, 4] - o["var_xT"]) <= 1e-9 * o["var_xT"]
    assert abs(stats[0, 5] - o["mean_jumps"]) <= 1e-12 * o["mean_jumps"]
    lamT = 2.0 * w.n_steps * w.dt
    assert abs(stats[0, 5] - lamT) < 5 * math.sqrt(lamT / w.n_paths)           # Poisson count law, eq. (4)


# ---- fp64 per-path parity, inertial (first 1000 steps) ----------------------------------------------------

def test_c2_fp64_trace_first_1000_steps(B, orc):
    w = W.c2().scaled(n_paths=512, n_steps=1200)
    stats, paths, trace = B.run_workload(w, B.BM_F64, want_paths=True, trace_steps=1000, trace_paths=512)
    ref, rtrace = oracle_run(orc, w, trace_paths=512, trace_steps=1000)
    scale = np.maximum(1.0, np.abs(rtrace))
    rel = np.abs(trace - rtrace) / scale
    assert rel.max() <= 1e-10, f"inertial trace: max relative deviation {rel.max():.3e}"
    # ensemble means of x(t_1000), v(t_1000) within 1e-9 relative
    for k in (0, 1):
        a, b = trace[:, -1, k].mean(), rtrace[:, -1, k].mean()
        assert abs(a - b) <= 1e-9 * max(1.0, abs(b))
    assert np.array_equal(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS])


def test_c2_fp64_full_length_statistics(B, orc):
    """Full-length inertial runs are chaotic: independent codes agree statistically only."""
    w = W.c2().scaled(n_paths=2048, n_steps=40000)
    stats, paths, _ = B.run_workload(w, B.BM_F64, want_paths=True)
    ref, _ = oracle_run(orc, w)
    assert_3se(paths, ref, B.BM_OUT_VBAR, "C2 fp64 <v>")
    assert_3se(paths, ref, B.BM_OUT_VT, "C2 fp64 v(T)")
    # the flip clocks do not depend on the (chaotic) motion: the same words give the same flips in both codes
    assert np.array_equal(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS])


def test_c2_fp64_full_size(B, orc):
    """Full C2 (65536 paths x 2e5 steps) in fp64 on the GPU: the first 1000 grid steps of the first 4096 paths against
    the oracle per path (criterion for the inertial configs), the full-length ensemble against an oracle sample of 2048
    paths within 3 combined standard errors (the motion is chaotic), flips per path exactly."""
    w = W.c2()
    n_tr = 4096
    stats, paths, trace = B.run_workload(w, B.BM_F64, want_paths=True, trace_steps=1000, trace_paths=n_tr)
    assert stats[0, 0] == w.n_paths
    _, rtrace = oracle_run(orc, w.scaled(n_steps=1000, n_discard=0), ids=np.arange(n_tr), trace_paths=n_tr, trace_steps=1000)
    rel = np.abs(trace - rtrace) / np.maximum(1.0, np.abs(rtrace))
    assert rel.max() <= 1e-10, f"C2 full: trace deviates by {rel.max():.3e}"
    ids = np.sort(np.random.default_rng(21).choice(w.n_paths, 2048, replace=False))
    ref, _ = oracle_run(orc, w, ids=ids)
    assert np.array_equal(paths[ids, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS])
    assert_3se(paths, ref, B.BM_OUT_VBAR, "C2 full fp64 <v>")
    assert_3se(paths, ref, B.BM_OUT_VT, "C2 full fp64 v(T)")
    assert_3se(paths, ref, B.BM_OUT_XT, "C2 full fp64 x(T)")
    muT = 1.0 * w.n_steps * w.dt
    assert abs(stats[0, 5] - muT) < 5 * math.sqrt(muT / w.n_paths)


# ---- fp32 statistical parity ------------------------------------------------------------------------------

FP32_CASES = [
    ("C0", lambda: W.c0(), None),
    ("C1", lambda: W.c1().scaled(n_paths=4096, n_steps=20000), None),
    ("C2", lambda: W.c2().scaled(n_paths=2048, n_steps=40000), None),
    ("C3", lambda: W.c3().scaled(n_paths=512, n_steps=24000, points=[0, 100, 255]), None),
    ("C4", lambda: W.c4().scaled(n_paths=2048, n_steps=20000, points=[0, 64 * 128 + 64, 127 * 128 + 127, 127 * 128]), None),
]


_ORACLE_CACHE = {}


def cached_oracle_run(orc, name, w):
    if name not in _ORACLE_CACHE:
        _ORACLE_CACHE[name] = oracle_run(orc, w)[0]
    return _ORACLE_CACHE[name]


@pytest.mark.parametrize("sincos", ["SFU", "FMA", "SFU-W32", "SFU-W16P"])
@pytest.mark.parametrize("name,make,_", FP32_CASES, ids=[c[0] for c in FP32_CASES])
def test_fp32_within_3_combined_se(B, orc, name, make, _, sincos):
    w = make()
    sc = B.BM_SINCOS_FMA if sincos == "FMA" else B.BM_SINCOS_SFU
    gs = B.BM_GAUSS_W32 if sincos.endswith("W32") else B.BM_GAUSS_W16P if sincos.endswith("W16P") else B.BM_GAUSS_AUTO
    stats, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True, sincos=sc, gauss=gs)
    ref = cached_oracle_run(orc, name, w)
    for pt in range(w.n_points):
        sl = slice(pt * w.n_paths, (pt + 1) * w.n_paths)
        assert_3se(paths[sl], ref[sl], B.BM_OUT_VBAR, f"{name}/{sincos} point {pt} <v>")
        assert_3se(paths[sl], ref[sl], B.BM_OUT_XT, f"{name}/{sincos} point {pt} x(T)")
        o = orc.reduce(ref[sl])
        # stats come from the on-device reduction of the same per-path values
        assert abs(stats[pt, 1] - paths[sl, B.BM_OUT_VBAR].mean()) <= 1e-12 * max(1, abs(stats[pt, 1]))
        assert_counts_close(paths[sl, B.BM_OUT_JUMPS], ref[sl, orc.OUT_JUMPS], f"{name}/{sincos} point {pt}")
        assert abs(stats[pt, 5] - paths[sl, B.BM_OUT_JUMPS].mean()) <= 1e-12 * max(1.0, o["mean_jumps"])


def test_fp32_paths_are_common_random_number_close(B, orc):
    """Same words for the same purpose: fp32 paths follow the fp64 oracle's path by path on a short horizon."""
    w = W.c0().scaled(n_paths=512, n_steps=400)
    _, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True, gauss=B.BM_GAUSS_W32)
    ref, _ = oracle_run(orc, w)
    d = np.abs(paths[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT])
    assert np.median(d) < 1e-4 and np.quantile(d, 0.99) < 1e-2


# ---- other potentials -------------------------------------------------------------------------------------

def test_pwl_model_I_fp64_and_fp32(B, orc):
    a, DP = 1.5, 1.0
    zeta, lam = DP / a, a * a / DP
    w = W.Workload("PWL-I", W.OVERDAMPED, W.params_table(1, A1=1.0, D=0.0, lambda_=lam, zeta=zeta), 768, 6000,
                   (1 / lam) / 100, 600, potential=W.POT_PWL)
    stats, paths, ref, bad, dx = check_fp64_overdamped(B, orc, w, what="PWL")
    # the force is discontinuous: a rounding difference at a kink flips a stage force, and the oracle's own result then
    # moves under a 1-ulp change of x0; only such paths are excluded (check_fp64_overdamped prints their number)
    assert bad.size == 0, f"PWL: {bad.size} well-conditioned paths beyond tolerance"
    _, p32, _ = B.run_workload(w, B.BM_F32, want_paths=True)
    assert_3se(p32, ref, B.BM_OUT_VBAR, "PWL fp32 <v>")


def test_quad_ou_fp64_matches_closed_form_and_oracle(B, orc):
    theta, D, x0, n, h = 1.0, 0.5, 1.5, 20, 0.05
    w = W.Workload("OU", W.OVERDAMPED, W.params_table(1, A1=theta, D=D, x0_fixed=x0), 4096, n, h, 0,
                   potential=W.POT_QUAD)
    stats, paths, ref, bad, dx = check_fp64_overdamped(B, orc, w, what="OU")
    assert bad.size == 0 and dx.max() < 1e-12
    z = theta * h
    R = 1 - z + z * z / 2 - z ** 3 / 4
    S = 1 - z / 2 + z * z / 4
    var_n = 2 * D * h * S * S * (1 - R ** (2 * n)) / (1 - R * R)
    assert abs(stats[0, 3] - x0 * R ** n) < 4 * math.sqrt(var_n / 4096)
    assert abs(stats[0, 4] - var_n) < 4 * var_n * math.sqrt(2 / 4095)
    _, p32, _ = B.run_workload(w, B.BM_F32, want_paths=True, gauss=B.BM_GAUSS_W32)
    assert np.abs(p32[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT]).max() < 1e-4
    _, p16, _ = B.run_workload(w, B.BM_F32, want_paths=True)          # W16: other normals, same law
    assert abs(p16[:, B.BM_OUT_XT].mean() - x0 * R ** n) < 4 * math.sqrt(var_n / 4096)
    assert abs(p16[:, B.BM_OUT_XT].var(ddof=1) - var_n) < 4 * var_n * math.sqrt(2 / 4095)


# ---- row f1: the paper's own scheme as printed (Alg. 1-4), CUDA against the oracle ------------------------------

def literal_workloads():
    a, DP = 1.5, 1.0
    zeta, lam = DP / a, a * a / DP
    Fa, Fb, tau = 3.0, 1.6, 0.3
    mu_a, mu_b = Fa / (tau * (Fa + Fb)), Fb / (tau * (Fa + Fb))
    L = W.SCHEME_PAPER_LITERAL
    return {
        # model I of the paper: piece-wise linear potential + white Poissonian noise (+ thermal)
        "I": W.Workload("lit-I", W.OVERDAMPED, W.params_table(1, A1=1.0, D=0.05, lambda_=lam, zeta=zeta), 777, 8000,
                        (1 / lam) / 400, 800, potential=W.POT_PWL, scheme=L),
        # model II: piece-wise linear potential + dichotomous noise
        "II": W.Workload("lit-II", W.OVERDAMPED, W.params_table(1, A1=1.0, D=0.0, Fa=Fa, Fb=Fb, mu_a=mu_a, mu_b=mu_b),
                         640, 8000, min(1 / mu_a, 1 / mu_b) / 200, 800, potential=W.POT_PWL, scheme=L),
        # all three sources on the smooth two-harmonic potential, a two-point sweep with a switched-off point
        "all": W.Workload("lit-all", W.OVERDAMPED,
                          W.params_table(2, A1=1.0, A2=0.25, F=0.05, D=[0.02, 0.0], lambda_=[2.0, 0.0], zeta=0.3,
                                         Fa=0.4, Fb=0.8, mu_a=1.5, mu_b=3.0), 300, 5000, 1e-3, 500, scheme=L),
    }


@pytest.mark.parametrize("name", ["I", "II", "all"])
def test_literal_scheme_fp64_matches_oracle_per_path(B, orc, name):
    w = literal_workloads()[name]
    stats, paths, _ = B.run_workload(w, B.BM_F64, want_paths=True)
    ref, _ = oracle_run(orc, w)
    assert np.array_equal(paths[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS]), "kick / flip counts differ"
    assert np.array_equal(paths[:, B.BM_OUT_SUBSTEPS], ref[:, orc.OUT_SUBSTEPS])
    dx = np.abs(paths[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT])
    bad = np.nonzero(dx > 1e-8 * (1 + np.abs(ref[:, orc.OUT_XT])))[0]
    if bad.size:    # piece-wise linear force: a rounding difference at a kink flips a stage force (A17 check decides)
        ill = ill_conditioned(orc, w, bad, ulps=(1, -1, 2, -2))
        assert ill.all(), f"{int((~ill).sum())} well-conditioned paths beyond tolerance, max {dx[bad[~ill]].max():.3e}"
        assert_few_ill_conditioned(int(ill.sum()), dx.size, f"literal {name}")
    good = np.setdiff1d(np.arange(dx.size), bad)
    assert np.abs(paths[good, B.BM_OUT_VBAR] - ref[good, orc.OUT_VBAR]).max() < 1e-8
    if bad.size == 0:
        for pt in range(w.n_points):
            o = orc.reduce(ref[pt * w.n_paths:(pt + 1) * w.n_paths])
            assert abs(stats[pt, 1] - o["mean_v"]) <= 1e-9 * abs(o["mean_v"]) + 1e-12
            assert abs(stats[pt, 5] - o["mean_jumps"]) <= 1e-12 * max(1.0, o["mean_jumps"])


def test_literal_scheme_fp64_trace(B, orc):
    w = literal_workloads()["all"].scaled(n_paths=64, n_steps=600)
    ref, tr_ref = oracle_run(orc, w, trace_paths=64, trace_steps=600)
    _, _, tr = B.run_workload(w, B.BM_F64, want_paths=True, trace_steps=600, trace_paths=64)
    assert np.abs(tr[:, :, 0] - tr_ref[:, :, 0]).max() < 1e-9 and np.all(tr[:, :, 1] == 0.0)


@pytest.mark.parametrize("name", ["I", "II", "all"])
def test_literal_scheme_fp32_within_3_combined_se(B, orc, name):
    w = literal_workloads()[name].scaled(n_paths=2048)
    _, paths, _ = B.run_workload(w, B.BM_F32, want_paths=True)
    ref, _ = oracle_run(orc, w)
    for pt in range(w.n_points):
        sl = slice(pt * w.n_paths, (pt + 1) * w.n_paths)
        assert_3se(paths[sl], ref[sl], B.BM_OUT_VBAR, f"literal {name} point {pt} <v>")
        assert_3se(paths[sl], ref[sl], B.BM_OUT_XT, f"literal {name} point {pt} x(T)")
        # same words, countdowns quantised to the grid: a count changes only where fp32 rounding of a waiting time
        # moves a countdown across an integer, which shifts the remaining kicks of that path by one step
        dcount = np.abs(paths[sl, B.BM_OUT_JUMPS] - ref[sl, orc.OUT_JUMPS])
        assert dcount.max() <= 2 and dcount.mean() <= 0.02, (dcount.max(), dcount.mean())


def test_literal_scheme_rejects_inertial(B):
    import torch
    w = W.c2().scaled(n_paths=32, n_steps=16)
    cfg = B.config_for(w, B.BM_F64)
    cfg.scheme = B.BM_SCHEME_PAPER_LITERAL
    p = torch.from_numpy(np.ascontiguousarray(w.params)).cuda()
    st = torch.zeros((1, 8), dtype=torch.float64, device="cuda")
    with pytest.raises(B.BmError) as e:
        B.bm_simulate(cfg, p, 1, w.n_paths, w.n_steps, w.dt, w.seed, st)
    assert e.value.status == B.BM_ERR_UNSUPPORTED


# ---- the paper's own validation (Fig. 3) on the GPU, against the closed forms of eq. (21)-(23) ----

@pytest.mark.parametrize("scheme", ["literal", "jump-adapted"])
def test_gpu_reproduces_paper_fig3a_model_I(B, scheme):
    """Fig. 3a: <v> vs D_P at a = 1.5, D_G = 0, 1024 paths, t_f = 1e3/lambda, spp = 400, 10 % discarded (:418-423);
    <v> = L J_I with J_I of eq. (21a).  Both the scheme as printed and the exact-time hot path must land on it."""
    from test_oracle_physics import J_model_I
    a = 1.5
    for DP in (0.5, 1.0, 2.0):
        zeta, lam = DP / a, a * a / DP
        n = 400_000
        w = W.Workload("fig3a", W.OVERDAMPED, W.params_table(1, A1=1.0, D=0.0, lambda_=lam, zeta=zeta), 1024, n,
                       (1 / lam) / 400, n // 10, potential=W.POT_PWL,
                       scheme=W.SCHEME_PAPER_LITERAL if scheme == "literal" else W.SCHEME_JUMP_ADAPTED)
        stats, _, _ = B.run_workload(w, B.BM_F32)
        v_th = 2 * J_model_I(a, DP)
        se = math.sqrt(stats[0, 2] / 1024)
        # literal scheme: O(dt) bias of the grid-quantised kick rate (A2), a few 1e-3 at spp = 400
        bias = 0.01 if scheme == "literal" else 0.002
        assert abs(stats[0, 1] - v_th) < 4 * se + bias, (scheme, DP, stats[0, 1], v_th, se)


def test_gpu_reproduces_paper_fig3b_model_II(B):
    """Fig. 3b: <v> vs tau at F_a = 3, F_b = 1.6, spp = 200 (:425); <v> = L J_II, eq. (21b) with reading R12."""
    from test_oracle_physics import J_model_II
    Fa, Fb = 3.0, 1.6
    for tau in (0.1, 0.3, 1.0):
        mu_a, mu_b = Fa / (tau * (Fa + Fb)), Fb / (tau * (Fa + Fb))
        n = 200_000
        w = W.Workload("fig3b", W.OVERDAMPED, W.params_table(1, A1=1.0, D=0.0, Fa=Fa, Fb=Fb, mu_a=mu_a, mu_b=mu_b),
                       1024, n, min(1 / mu_a, 1 / mu_b) / 200, n // 10, potential=W.POT_PWL,
                       scheme=W.SCHEME_PAPER_LITERAL)
        stats, _, _ = B.run_workload(w, B.BM_F32)
        v_th = 2 * J_model_II(Fa, Fb, tau)
        se = math.sqrt(stats[0, 2] / 1024)
        assert abs(stats[0, 1] - v_th) < 4 * se + 0.01, (tau, stats[0, 1], v_th, se)


# ---- per-point step length (row f2): a sweep over noise parameters at fixed steps per characteristic time --------

def test_per_point_dt_sweep_matches_oracle_and_fig3a(B, orc):
    """Fig. 3a in ONE launch: three values of D_P at a = 1.5, each with its own dt = (1/lambda)/400.
    fp64 per path against the oracle (run point by point with that point's dt and the same global path ids), the
    ensemble against eq. (21a); fp32 within 3 combined standard errors."""
    import torch
    from test_oracle_physics import J_model_I
    a, DPs = 1.5, np.array([0.5, 1.0, 2.0])
    lam, zeta = a * a / DPs, DPs / a
    params = W.params_table(3, A1=1.0, D=0.0, lambda_=lam, zeta=zeta)
    dts = (1.0 / lam) / 400
    n_paths, n_steps, nd = 512, 40_000, 4_000
    dev = torch.device("cuda:0")
    res = {}
    for prec in (B.BM_F64, B.BM_F32):
        cfg = B.make_config(prec=prec, potential=B.BM_POT_PWL, scheme=B.BM_SCHEME_PAPER_LITERAL, noise=B.BM_NOISE_POISSON,
                            n_discard=nd)
        st = torch.zeros((3, 8), dtype=torch.float64, device=dev)
        pa = torch.zeros((3 * n_paths, B.BM_OUT_STRIDE), dtype=torch.float64, device=dev)
        B.bm_simulate_dt(cfg, torch.from_numpy(params).to(dev), torch.from_numpy(dts).to(dev), 3, n_paths, n_steps, W.SEED, st, pa)
        torch.cuda.synchronize()
        res[prec] = (st.cpu().numpy(), pa.cpu().numpy())
    for pt in range(3):
        ids = pt * n_paths + np.arange(n_paths)
        ref, _ = orc.simulate(params, n_paths, n_steps, float(dts[pt]), W.SEED, potential=orc.POT_PWL,
                              scheme=orc.SCHEME_PAPER_LITERAL, n_discard=nd, ids=ids)
        s64, p64 = res[B.BM_F64]
        got = p64[ids]
        assert np.array_equal(got[:, B.BM_OUT_JUMPS], ref[:, orc.OUT_JUMPS])
        dx = np.abs(got[:, B.BM_OUT_XT] - ref[:, orc.OUT_XT])
        over = np.nonzero(dx > 1e-8 * (1 + np.abs(ref[:, orc.OUT_XT])))[0]
        if over.size:   # a stage force flipped at a kink: the A17 check on the same paths at this point's own dt
            wp = W.Workload("pt", W.OVERDAMPED, params, n_paths, n_steps, float(dts[pt]), nd, potential=W.POT_PWL,
                            scheme=W.SCHEME_PAPER_LITERAL)
            ill = ill_conditioned(orc, wp, ids[over], ulps=(1, -1, 2, -2))
            assert ill.all(), f"point {pt}: {int((~ill).sum())} well-conditioned paths beyond tolerance, max {dx.max():.3e}"
            assert_few_ill_conditioned(int(ill.sum()), n_paths, f"per-point dt, point {pt}")
        v_th = 2 * J_model_I(a, float(DPs[pt]))
        se = math.sqrt(s64[pt, 2] / n_paths)
        assert abs(s64[pt, 1] - v_th) < 4 * se + 0.01, (pt, s64[pt, 1], v_th)
        _, p32 = res[B.BM_F32]
        assert_3se(p32[ids], ref, B.BM_OUT_VBAR, f"per-point dt, fp32, point {pt}")


def test_per_point_dt_equal_entries_reproduce_scalar_dt(B):
    """dt_points all equal to dt must give bit-identical results to bm_simulate(dt) for both hot-path kernels."""
    import torch
    for w, prec in ((W.c4().scaled(n_paths=64, n_steps=400, points=[3, 9000, 16383]), B.BM_F32),
                    (W.c3().scaled(n_paths=64, n_steps=240, points=[0, 200]), B.BM_F64)):
        s0, p0, _ = B.run_workload(w, prec, want_paths=True)
        cfg = B.config_for(w, prec)
        dev = torch.device("cuda:0")
        st = torch.zeros((w.n_points, 8), dtype=torch.float64, device=dev)
        pa = torch.zeros((w.n_points * w.n_paths, B.BM_OUT_STRIDE), dtype=torch.float64, device=dev)
        B.bm_simulate_dt(cfg, torch.from_numpy(np.ascontiguousarray(w.params)).to(dev),
                         torch.full((w.n_points,), w.dt, dtype=torch.float64, device=dev), w.n_points, w.n_paths, w.n_steps,
                         w.seed, st, pa)
        torch.cuda.synchronize()
        assert np.array_equal(st.cpu().numpy(), s0) and np.array_equal(pa.cpu().numpy(), p0)


def test_box_muller_edge_words_against_the_definition(B):
    """The kernels' own fp64 ln / sqrt / sincospi (sim_f64.cuh) on the words the Philox stream reaches only by chance: u next
    to 0 and to 1 (w = 0, 2^32 - 1), angles on and next to the quadrant boundaries, mantissas around sqrt(2) (the split of
    ln u = k ln 2 + ln m), every exponent k.  Expected values: eq. (27), with u(w) = (w + 1/2) 2^-32 (R3),
    evaluated with mpmath at 40 digits -- the definition itself, not the oracle's libm value (which carries the rounding
    of 2 pi u: up to 4e-16 r in a normal)."""
    import mpmath as mp
    import torch
    mp.mp.dps = 40
    edge = [0, 1, 2, 3, 2 ** 32 - 1, 2 ** 32 - 2, 2 ** 31, 2 ** 31 - 1, 2 ** 31 + 1, 2 ** 30, 2 ** 30 - 1, 2 ** 30 + 1,
            3 * 2 ** 30, 3 * 2 ** 30 - 1, 3 * 2 ** 30 + 1, 2 ** 29, 5 * 2 ** 29, 7 * 2 ** 29 + 1,
            int(2 ** 32 / mp.sqrt(2)), int(2 ** 32 / mp.sqrt(2)) + 1, int(2 ** 31 / mp.sqrt(2)), int(2 ** 31 * mp.sqrt(2)) - 1]
    edge += [2 ** k for k in range(1, 32)] + [2 ** k - 1 for k in range(2, 32)] + [2 ** k + 1 for k in range(2, 32)]
    rng = np.random.default_rng(20141409)
    rnd = [int(v) for v in rng.integers(0, 2 ** 32, 200)]
    pairs = [(a, b) for a in edge for b in (0, 2 ** 30, 2 ** 31 - 1, 2 ** 31, 3 * 2 ** 30 + 1, 2 ** 32 - 1, 123456789)]
    pairs += [(a, b) for b in edge for a in (0, 2 ** 32 - 1, 987654321)] + list(zip(rnd[:100], rnd[100:]))
    words = torch.tensor(np.array(pairs, dtype=np.uint32).view(np.int32), dtype=torch.int32, device="cuda")
    out = torch.zeros((len(pairs), 2), dtype=torch.float64, device="cuda")
    B.bm_box_muller_words(B.BM_F64, words, len(pairs), out)
    got = out.cpu().numpy()
    worst = 0.0
    for (wa, wb), g in zip(pairs, got):
        ua, ub = (mp.mpf(wa) + mp.mpf(1) / 2) / 2 ** 32, (mp.mpf(wb) + mp.mpf(1) / 2) / 2 ** 32
        r = mp.sqrt(-2 * mp.log(ua))
        e0, e1 = r * mp.cos(2 * mp.pi * ub), r * mp.sin(2 * mp.pi * ub)
        for e, v in ((e0, g[0]), (e1, g[1])):
            # absolute error in units of the ulp of the RADIUS: a normal next to a zero of the angle is a small
            # difference of O(r) terms and is good to ulp(r), not to its own ulp
            err = abs(mp.mpf(float(v)) - e) / mp.mpf(float(np.spacing(float(r))))
            worst = max(worst, float(err))
    assert worst <= 2.0, f"fp64 Box-Muller: {worst:.2f} ulp of the radius from the definition"
    # fp32 W32 transform: MUFU accuracy class (lg2, sqrt, sin, cos approximations), u on a 2^-23 grid (R3)
    out32 = torch.zeros((len(pairs), 2), dtype=torch.float32, device="cuda")
    B.bm_box_muller_words(B.BM_F32, words, len(pairs), out32)
    g32 = out32.cpu().numpy().astype(np.float64)
    assert np.isfinite(g32).all() and np.abs(g32).max() < 6.0
    # the fp32 reading of R3: u = ((w >> 9) + 1) 2^-23 for the radius, (w >> 9) 2^-23 turns for the angle
    wa, wb = np.array([p[0] for p in pairs], dtype=np.int64), np.array([p[1] for p in pairs], dtype=np.int64)
    r32 = np.sqrt(-2.0 * np.log(((wa >> 9) + 1) * 2.0 ** -23))
    ang = 2.0 * np.pi * (wb >> 9) * 2.0 ** -23
    exp32 = np.stack([r32 * np.cos(ang), r32 * np.sin(ang)], axis=1)
    d32 = np.abs(g32 - exp32).max()
    assert d32 < 2e-5, f"fp32 Box-Muller (MUFU lg2, sqrt, sin, cos): {d32:.2e} from the definition"
