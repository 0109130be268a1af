"""The minimax tables of csrc/trace_math.cuh are the output of csrc/gen_poly.py: regenerate them
and compare, and check each table's accuracy claim against numpy's atan / atanh in float64."""
import importlib.util
import os
import re

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_1505_07674_b200", "csrc")


def _gen_poly():
    spec = importlib.util.spec_from_file_location("gen_poly", os.path.join(CSRC, "gen_poly.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


def _tables_in_header():
    text = open(os.path.join(CSRC, "trace_math.cuh")).read()
    out = {}
    for name, n, body in re.findall(r"__device__ constexpr float (kAtanh?\w+)\[(\d+)\] = \{([^}]*)\};", text):
        vals = [float(v.strip().rstrip("f")) for v in body.split(",")]
        assert len(vals) == int(n)
        out[name] = np.array(vals)
    return out


def test_header_tables_are_what_gen_poly_writes_and_as_accurate_as_claimed():
    header = _tables_in_header()
    gen = _gen_poly().generate()
    assert set(header) == {g[0] for g in gen}
    for name, T, deg, centred, coef, fit_err, err32 in gen:
        assert len(header[name]) == deg + 1
        assert np.allclose(header[name], coef, rtol=2e-7, atol=1e-9), name       # 10 printed digits, lstsq noise
        assert fit_err < 7e-8 and err32 < 2e-7, (name, fit_err, err32)
        # the header's numbers, evaluated in float64, against numpy (not against gen_poly's own f)
        t = np.linspace(1e-9, T, 20001)
        z = np.sqrt(t)
        x = 2 * t / T - 1 if centred else t
        p = np.polyval(header[name], x)
        ref = np.arctanh(z) / z * 2 / np.log(2) if "Atanh" in name else np.arctan(z) / z
        assert np.max(np.abs(p / ref - 1)) < 7e-8, name
