"""The oracle and the input generator still produce the frozen config-1 numbers (tests/golden/)."""
import importlib.util
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_matches_frozen_config1_values():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    stored = {}
    for line in open(os.path.join(HERE, "golden", "oracle_config1.txt")):
        if line.startswith("#"):
            continue
        name, v = line.split()
        stored[name] = float(v)
    now = dict(mod.compute())
    assert set(now) == set(stored)
    for name, v in now.items():
        ref = stored[name]
        if name.startswith("cg_iters") or name.startswith("cg_freeze"):
            assert v == ref, name
        elif name.startswith("cg_x"):
            assert abs(v - ref) <= 1e-9 * abs(ref), name           # solutions: insensitive to compiler rounding
        else:
            assert abs(v - ref) <= 1e-12 * max(1.0, abs(ref)), name
