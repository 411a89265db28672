"""The oracle reproduces its committed golden samples (regression pin; see tests/golden/make_golden.py)."""
import importlib.util
import os

HERE = os.path.dirname(os.path.abspath(__file__))


def test_cfg1_golden_samples():
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    got = {(t, a, b, c): v for t, a, b, c, v in mod.samples()}
    n = 0
    with open(os.path.join(HERE, "golden", "cfg1_block_samples.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            t, a, b, c, v = line.split()
            assert abs(got[(t, int(a), int(b), int(c))] - float(v)) < 1e-9
            n += 1
    assert n == 48
