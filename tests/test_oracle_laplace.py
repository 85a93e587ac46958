"""Laplace's law for the oracle (north_star: dp = 2 sigma / R within 3 %), config 1.

The 10 000-step run is too long for the CPU suite, so its trajectory is a stored fixture written
by tests/golden/make_laplace.py, which calls only oracle/.  This test (i) checks the stored
settled values against 2 sigma/R and (ii) re-runs the first 100 steps live to make sure the
fixture still belongs to the oracle as it stands.
"""
import os

import numpy as np

from oracle import Oracle
from paper_2012_06144_b200 import inputs

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "laplace_config1.txt")


def _rows():
    rows = [l.split() for l in open(GOLDEN) if not l.startswith("#")]
    return {int(r[0]): (float(r[1]), float(r[2]), float(r[3])) for r in rows}


def test_laplace_law_settled_within_3_percent():
    rows = _rows()
    for s in (8000, 9000, 10000):
        ratio, drift, umax = rows[s]
        assert abs(ratio - 1.0) < 0.03, (s, ratio)
        assert abs(drift) < 1e-12                     # sum(phi) conserved over the whole run
        assert umax < 5e-5                            # spurious currents stay small
    # before the acoustic transient has decayed the law does NOT hold (guards against a trivial fixture)
    assert abs(rows[100][0] - 1.0) > 0.5


def test_fixture_belongs_to_current_oracle():
    p, phi, u = inputs.config1()
    o = Oracle.from_params(p)
    o.init(phi, u)
    o.step(100)
    _, uu, pr = o.fields()
    c = p.nx // 2
    ratio = (pr[c, c, c] - pr[0, 0, 0]) / (2 * p.sigma / 8.0)
    assert abs(ratio - _rows()[100][0]) < 1e-9 * abs(ratio)
    assert abs(np.abs(uu).max() - _rows()[100][2]) < 1e-9
