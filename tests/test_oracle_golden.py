"""Golden fixtures: closed-form values (tests/golden/closed_forms.txt, each
with its source) and the oracle regression fixture written by
tests/golden/make_golden.py from oracle/ only."""
import importlib.util
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def _closed_forms():
    out = {}
    for line in open(os.path.join(HERE, "golden", "closed_forms.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, val = line.split()[:2]
        out[name] = float(val)
    return out


def test_closed_forms(ora):
    cf = _closed_forms()
    assert abs(ora.shape(2, 0.0) - cf["S2_at_0"]) < 1e-16
    assert abs(ora.shape(2, 1.0) - cf["S2_at_1"]) < 1e-16
    assert abs(ora.shape(3, 0.0) - cf["S3_at_0"]) < 1e-16
    assert abs(ora.shape(3, -1.0) - cf["S3_at_1"]) < 1e-16
    assert abs(ora.shape(3, 0.5) - cf["S3_at_half"]) < 1e-16
    g = ora.make_grid(32, 32, 32, 0.5e-6, 0.5e-6, 0.5e-6)
    assert abs(ora.courant_dt(g) / cf["courant_dt_cubic_0p5um"] - 1) < 1e-15
    wp = np.sqrt(1e25 * 1.602176634e-19 ** 2 / (ora.lib().ora_const_eps0() * 9.1093837015e-31))
    assert abs(wp / cf["omega_p_n0_1e25"] - 1) < 1e-15
    assert ora.lib().ora_const_c() == 299792458.0


def test_oracle_regression_fixture(ora):
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mg = importlib.util.module_from_spec(spec); spec.loader.exec_module(mg)
    sims = {}
    n = 0
    for line in open(os.path.join(HERE, "golden", "oracle_cycle_4x4x4.txt")):
        if line.startswith("#"):
            continue
        order, name, idx, val = line.split()
        order, idx, val = int(order), int(idx), float(val)
        if order not in sims:
            sim = mg.case(order)
            sims[order] = {**sim.get_fields(), **sim.get_particles(0)}
        got = sims[order][name][idx]
        assert got == val or abs(got - val) <= 1e-14 * abs(val), (order, name, idx, got, val)
        n += 1
    assert n == 3 * (9 * 4 + 6 * 6)
