"""The oracle against its own frozen results on configs[0] (tests/golden/oracle_tiny.txt, written by make_golden.py from
oracle/ alone): guards the pinned oracle against accidental changes. fp64 sums, compared to 1e-10 relative."""
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_reproduces_its_frozen_values():
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    now = mod.values()
    stored = {}
    for line in open(os.path.join(HERE, "golden", "oracle_tiny.txt")):
        if not line.startswith("#"):
            k, v = line.split()
            stored[k] = float(v)
    assert set(now) == set(stored)
    for k, v in stored.items():
        assert np.isclose(now[k], v, rtol=1e-10, atol=1e-12), (k, now[k], v)
