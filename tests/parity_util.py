"""Helpers shared by the GPU parity tests (test infrastructure; calls only oracle/ and numpy)."""
import math

import numpy as np


def oracle_run(orc, w, ids=None, trace_paths=0, trace_steps=0):
    return orc.simulate(w.params, w.n_paths, w.n_steps, w.dt, w.seed, model=w.model, potential=w.potential,
                        scheme=w.scheme, n_discard=w.n_discard, ids=ids, trace_paths=trace_paths,
                        trace_steps=trace_steps)


def se_mean(v):
    return v.std(ddof=1) / math.sqrt(v.size)


def se_var(v):
    c = v - v.mean()
    m2, m4 = (c ** 2).mean(), (c ** 4).mean()
    return math.sqrt(max(m4 - m2 * m2, 0.0) / v.size)


def assert_3se(gpu_paths, orc_paths, col, what):
    """fp32 criterion: mean and variance of column `col` within 3 combined SE."""
    a, b = gpu_paths[:, col], orc_paths[:, col]
    dm = abs(a.mean() - b.mean())
    sm = math.hypot(se_mean(a), se_mean(b))
    assert dm <= 3 * sm + 1e-12, f"{what}: mean differs by {dm:.3e} > 3 SE = {3 * sm:.3e}"
    dv = abs(a.var(ddof=1) - b.var(ddof=1))
    sv = math.hypot(se_var(a), se_var(b))
    assert dv <= 3 * sv + 1e-12, f"{what}: variance differs by {dv:.3e} > 3 SE = {3 * sv:.3e}"
    return dm / max(sm, 1e-300), dv / max(sv, 1e-300)


def assert_few_ill_conditioned(n_ill, n_paths, what):
    """SURVEY.md A17 expects the ill-conditioned paths to be "a few of 65 536": the exclusion must not become a way for a
    kernel that diverges on many paths to pass.  At most 8 of a full-size ensemble (>= 65 536 paths), at most 2 of the
    smaller cases (observed counts: DESIGN.md section 7)."""
    limit = 8 if n_paths >= 65536 else 2
    print(f"A17 {what}: {n_ill} of {n_paths} paths ill-conditioned and excluded (limit {limit})")
    assert n_ill <= limit, f"{what}: {n_ill} of {n_paths} paths excluded as ill-conditioned, more than the {limit} A17 allows"


def ill_conditioned(orc, w, ids, ulps=(1, -1)):
    """which of the global path ids `ids` are ill-conditioned, i.e. have an ORACLE result x(T) that moves
    by more than 1e-9 (1 + |x|) when x0 is moved by one unit in the last place (a kick that lands next to a potential
    maximum amplifies a rounding difference by the inverse of its distance).  The perturbed runs keep every random word
    of the path: the table is re-laid out with one path per parameter point (g = point), the point's row carrying
    x0_fixed = x0 of that path moved by `ulps`.  Returns a boolean array aligned with ids."""
    ids = np.asarray(ids, dtype=np.int64)
    if ids.size == 0:
        return np.zeros(0, dtype=bool)
    x0_col = 13                                    # bm_params.x0_fixed
    rows = int(ids.max()) + 1                      # one path per row up to the largest id asked for
    base, _ = oracle_run(orc, w, ids=ids)
    period = {0: 1.0, 1: 2.0, 2: 1.0}[w.potential]
    flagged = np.zeros(ids.size, dtype=bool)
    if rows > (1 << 20):
        # ids deep inside a large sweep (C4: up to 6.7e7): a row per path id would not fit.  One oracle call per path
        # and perturbation instead, in the workload's own layout: the row of the path's point carries the moved x0 and
        # only that path is run, so it keeps its id and with it every random word.
        for n, g in enumerate(ids):
            pt = int(g) // w.n_paths
            x_start = w.params[pt, x0_col]
            if x_start < 0.0:
                x_start = period * (orc.philox_call(w.seed, int(g), 0, 0)[0] * 2.0 ** -32)
            for k in ulps:
                x0 = x_start
                for _ in range(abs(k)):
                    x0 = np.nextafter(x0, np.inf if k > 0 else -np.inf)
                table = np.array(w.params, copy=True)
                table[pt, x0_col] = max(x0, 0.0)
                pert, _ = orc.simulate(table, w.n_paths, w.n_steps, w.dt, w.seed, model=w.model, potential=w.potential,
                                       scheme=w.scheme, n_discard=w.n_discard, ids=np.array([g], dtype=np.int64))
                d = abs(pert[0, orc.OUT_XT] - base[n, orc.OUT_XT])
                flagged[n] |= bool(d > 1e-9 * (1 + abs(base[n, orc.OUT_XT])))
        return flagged
    for k in ulps:
        table = np.ascontiguousarray(w.params[np.arange(rows) // w.n_paths])
        for g in ids:
            x0 = table[g, x0_col]
            if x0 < 0.0:                           # random x0: word 0 of init-stream call 0 (reading R4)
                x0 = period * (orc.philox_call(w.seed, int(g), 0, 0)[0] * 2.0 ** -32)
            for _ in range(abs(k)):
                x0 = np.nextafter(x0, np.inf if k > 0 else -np.inf)
            table[g, x0_col] = max(x0, 0.0)
        pert, _ = orc.simulate(table, 1, w.n_steps, w.dt, w.seed, model=w.model, potential=w.potential,
                               scheme=w.scheme, n_discard=w.n_discard, ids=ids)
        d = np.abs(pert[:, orc.OUT_XT] - base[:, orc.OUT_XT])
        flagged |= d > 1e-9 * (1 + np.abs(base[:, orc.OUT_XT]))
    return flagged


def assert_counts_close(gpu_counts, orc_counts, what):
    """fp32 event counts: the jump clocks run on the oracle's own Philox words with times rounded to fp32, so a path's
    count can differ from the oracle's only by an event within rounding of t_f: at most 1 per path, and rarely."""
    d = np.abs(gpu_counts - orc_counts)
    assert d.max() <= 1, f"{what}: a path's event count differs by {d.max()}"
    assert d.mean() <= 5e-3, f"{what}: {d.sum():.0f} of {d.size} paths differ in their event count"
