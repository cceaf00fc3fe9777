"""Pins for the oracle's random-number layer (R1-R3).  CPU only.

P1  Philox4x32-10 against PyTorch's at::philox_engine (independent library routine), bit-exact.
P13 Box-Muller: exact values recomputed in 50-digit arithmetic from the raw words, and moments.
"""
import numpy as np
import mpmath as mp
import pytest

from paper_1409_4923_b200.workloads import SEED


def test_p1_philox_matches_aten_engine(orc, aten_philox):
    rng = np.random.default_rng(1)
    cases = [((0, 0, 0, 0), (0, 0)), ((0xFFFFFFFF,) * 4, (0xFFFFFFFF,) * 2), ((1, 0, 0, 0), (0, 0)),
             ((0, 0, 0, 1), (0, 0)), ((0, 0, 0, 0), (1, 0)), ((0, 0, 0, 0), (0, 1))]
    for _ in range(3000):
        c = tuple(int(x) for x in rng.integers(0, 2**32, 4))
        k = tuple(int(x) for x in rng.integers(0, 2**32, 2))
        cases.append((c, k))
    for c, k in cases:
        seed = k[0] | (k[1] << 32)
        offset = c[0] | (c[1] << 32)
        subseq = c[2] | (c[3] << 32)
        assert orc.philox4x32_10(c, k) == aten_philox(seed, subseq, offset), (c, k)


def test_p1_keyed_call_layout(orc, aten_philox):
    """R2: key=(seed lo,hi); counter=(idx, stream, g lo, g hi) == ATen (seed, subsequence=g, offset=idx|stream<<32)."""
    for g in (0, 1, 65535, 2**32 + 7, 67108863):
        for stream in (0, 1, 2, 3):
            for idx in (0, 1, 12345, 2**32 - 1):
                assert orc.philox_call(SEED, g, stream, idx) == aten_philox(SEED, g, idx | (stream << 32))


def test_p1_philox_is_a_bijection_on_a_sample(orc):
    seen = set()
    for idx in range(4096):
        out = orc.philox_call(SEED, 5, 1, idx)
        assert out not in seen
        seen.add(out)


def test_p1_philox_words_are_uniform(orc):
    w = orc.philox_fill(SEED, 0, 64, 1, 0, 256).ravel()      # 65536 words
    counts = np.bincount(w >> 24, minlength=256)
    chi2 = ((counts - w.size / 256) ** 2 / (w.size / 256)).sum()
    assert 150 < chi2 < 380                                   # 255 dof: mean 255, sd 22.6
    bits = np.unpackbits(w.view(np.uint8)).mean()
    assert abs(bits - 0.5) < 4 * 0.5 / np.sqrt(w.size * 32)


def test_r3_uniform_is_open_interval_and_exact(orc):
    assert orc.u01(0) == 2.0 ** -33
    assert orc.u01(2**32 - 1) == 1.0 - 2.0 ** -33
    assert orc.u01(2**31) == 0.5 + 2.0 ** -33


def test_p13_box_muller_exact_values(orc):
    """Recompute four Gaussians from the raw Philox words in 50-digit arithmetic (R3 formula, cos first)."""
    mp.mp.dps = 50
    for g, b in ((0, 0), (3, 17), (65535, 24999)):
        w = orc.philox_call(SEED, g, 1, b)
        u = [(mp.mpf(x) + mp.mpf(1) / 2) / mp.mpf(2) ** 32 for x in w]
        r0 = mp.sqrt(-2 * mp.log(u[0]))
        r1 = mp.sqrt(-2 * mp.log(u[2]))
        ref = [r0 * mp.cos(2 * mp.pi * u[1]), r0 * mp.sin(2 * mp.pi * u[1]),
               r1 * mp.cos(2 * mp.pi * u[3]), r1 * mp.sin(2 * mp.pi * u[3])]
        got = orc.gauss_block(SEED, g, b)
        for a, e in zip(got, ref):
            assert abs(a - float(e)) <= 4e-15 * max(1.0, abs(float(e)))
        for m in range(4):
            assert orc.gauss(SEED, g, 4 * b + m) == got[m]


def test_p13_box_muller_moments(orc):
    n_paths, n_blocks = 256, 1000
    g = np.array([orc.gauss_block(SEED, p, b) for p in range(n_paths) for b in range(n_blocks)]).ravel()
    n = g.size                                               # 1.024e6
    assert abs(g.mean()) < 4 / np.sqrt(n)
    assert abs(g.var() - 1) < 4 * np.sqrt(2 / n)
    assert abs((g ** 3).mean()) < 4 * np.sqrt(15 / n)
    assert abs((g ** 4).mean() - 3) < 4 * np.sqrt(96 / n)
    # components of one block are uncorrelated with each other
    gb = g.reshape(-1, 4)
    c = np.corrcoef(gb.T)
    assert np.abs(c - np.eye(4)).max() < 4 / np.sqrt(gb.shape[0])
