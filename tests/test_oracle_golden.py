"""The oracle reproduces its committed regression fixture (tests/golden/oracle_regression.txt, written by
tests/golden/make_golden.py from oracle/ only).  A change of the oracle's arithmetic has to regenerate the fixture
and say why in its commit message.  CPU only."""
import importlib.util
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


def test_oracle_matches_its_committed_fixture(ref):
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    now = mod.rows()
    stored = [l.rstrip("\n") for l in open(os.path.join(HERE, "golden", "oracle_regression.txt")) if not l.startswith("#")]
    assert len(now) == len(stored) == 28
    for a, b in zip(now, stored):
        assert a.split()[:4] == b.split()[:4]
        va, vb = np.array(a.split()[4:], float), np.array(b.split()[4:], float)
        # summation order inside OpenMP-free loops is fixed; allow only libm-level noise
        assert np.allclose(va, vb, rtol=1e-12, atol=0), (a, b)
