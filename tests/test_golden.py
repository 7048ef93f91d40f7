"""The oracle reproduces its frozen output on the tiny scene (tests/golden/tiny_scene.txt, written by
tests/golden/make_golden.py from oracle/ only).  A regression net for the oracle, not a pin: the pins are in
test_oracle_pins.py."""
import importlib.util
import os

import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_matches_its_golden_file(oracle):
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    want = {}
    for line in open(os.path.join(HERE, "golden", "tiny_scene.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        want[k] = float(v)
    got = dict(mod.compute())
    assert set(got) == set(want)
    for k, v in want.items():
        assert got[k] == pytest.approx(v, rel=1e-11, abs=1e-13), k
