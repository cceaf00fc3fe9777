"""The coefficient tables of the fp64 kernels' own elementary functions (sim_f64.cuh, __constant__ arrays and the split
constants of ln 2 and pi/2) are the output of csrc/make_poly_f64.py: the generator is run here and compared with what is
pasted in the header, so a table edited by hand or a generator that drifted fails.  CPU only (mpmath)."""
import contextlib
import io
import os
import re
import runpy

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1409_4923_b200", "csrc")


@pytest.fixture(scope="module")
def generated():
    pytest.importorskip("mpmath")
    buf = io.StringIO()
    with contextlib.redirect_stdout(buf):
        runpy.run_path(os.path.join(CSRC, "make_poly_f64.py"), run_name="__main__")
    out = buf.getvalue()
    tables = {m.group(1): [float(x) for x in m.group(2).split(",")] for m in re.finditer(r"(\w+)\[\d+\] = \{([^}]*)\}", out)}
    scalars = {m.group(1): float(m.group(2)) for m in re.finditer(r"(\w+) = ([-+0-9.e]+)", out)}
    return tables, scalars


def header_tables():
    src = open(os.path.join(CSRC, "sim_f64.cuh")).read()
    return src, {m.group(1): [float(x) for x in m.group(3).split(",")]
                 for m in re.finditer(r"__constant__ double (\w+)\[(\d+)\] = \{([^}]*)\}", src)}


def test_constant_tables_are_the_generators_output(generated):
    tables, _ = generated
    _, hdr = header_tables()
    assert set(hdr) == {"SINPI_C", "COSPI_C", "LOGP_C", "SIN_C", "COS_C", "COS2PI_E", "COS2PI_O"}
    for name, coeffs in hdr.items():
        gen = tables[name]
        assert len(gen) == len(coeffs), name
        for i, (a, b) in enumerate(zip(coeffs, gen)):
            # the interpolation system is solved at 60 digits; what is left is the last-place rounding of a pasted literal
            assert abs(a - b) <= 4e-16 * max(abs(b), 1e-300) or abs(a - b) < 1e-22, (name, i, a, b)


def test_split_constants_are_the_generators_output(generated):
    _, scalars = generated
    src, _ = header_tables()
    for name in ("LN2_HI", "LN2_LO", "PIO2_1", "PIO2_2", "PIO2_3", "TWO_OVER_PI"):
        lit = repr(scalars[name])
        assert lit in src, f"{name} = {lit} of make_poly_f64.py does not appear in sim_f64.cuh"
