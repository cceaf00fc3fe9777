import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)



def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box with -m gpu)")


@pytest.fixture(scope="session")
def orc():
    """The fp64 CPU oracle (built on demand with gcc)."""
    from oracle import bm_oracle
    bm_oracle.lib()
    return bm_oracle


@pytest.fixture(scope="session")
def c1_full_oracle(orc):
    """The oracle's per-path records of the WHOLE of C1 (65 536 paths x 1e5 steps; under a minute on 16 host cores),
    computed once per session: the fp64 per-path test and the fp32 full-size test both compare against all of it."""
    from paper_1409_4923_b200 import workloads as W
    w = W.c1()
    ref, _ = orc.simulate(w.params, w.n_paths, w.n_steps, w.dt, w.seed, model=w.model, potential=w.potential,
                          scheme=w.scheme, n_discard=w.n_discard)
    return ref


@pytest.fixture(scope="session")
def aten_philox(tmp_path_factory):
    """PyTorch's own at::philox_engine compiled into a tiny shared object: an independent library routine."""
    import ctypes as C
    import torch
    inc = os.path.join(os.path.dirname(torch.__file__), "include")
    src = os.path.join(ROOT, "tests", "helpers", "aten_philox.cpp")
    out = str(tmp_path_factory.mktemp("aten") / "aten_philox.so")
    subprocess.run(["g++", "-O1", "-std=c++17", "-fPIC", "-shared", "-I" + inc, "-o", out, src], check=True)
    lib = C.CDLL(out)
    lib.aten_philox4x32_10.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(C.c_uint32)]

    def call(seed, subsequence, offset):
        o = (C.c_uint32 * 4)()
        lib.aten_philox4x32_10(seed, subsequence, offset, o)
        return tuple(int(x) for x in o)
    return call
