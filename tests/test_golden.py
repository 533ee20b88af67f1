"""Regression fixture of the oracle + input generator (see tests/golden/make_golden.py)."""
import importlib.util
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_golden_fixture_reproduces():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    rows = mod.compute()
    with open(os.path.join(HERE, "golden", "oracle_2x2x2x2_L5_4.txt")) as fh:
        stored = [ln.strip().split(" | ") for ln in fh if not ln.startswith("#")]
    assert len(stored) == len(rows)
    for (name, re, im), (sname, sre, sim) in zip(rows, stored):
        assert name == sname
        scale = max(1.0, abs(float(sre)), abs(float(sim)))
        assert abs(re - float(sre)) < 1e-12 * scale and abs(im - float(sim)) < 1e-12 * scale
