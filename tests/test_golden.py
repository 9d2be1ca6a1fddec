"""The oracle reproduces its own committed values (tests/golden/, written by make_golden.py from the
oracle alone).  Guards against silent drift of the oracle or of the seeded input generators."""
import os

import numpy as np
import pytest

from oracle import oracle
from paper_1211_3556_b200 import workloads as wl

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def load_golden(name):
    data = np.loadtxt(os.path.join(GOLDEN, name), comments="#")
    return data[:, 0].astype(np.int64), data[:, 1]


@pytest.mark.parametrize("cfg,name", [(0, "cfg0_samples.txt"), (1, "cfg1_samples.txt")])
def test_oracle_reproduces_golden(cfg, name):
    w = wl.config(cfg)[0]
    pix, expect = load_golden(name)
    got = oracle.convolve(w.map_f32(), w.table(), w.theta_cut, level=1, pixels=pix)
    np.testing.assert_allclose(got, expect, rtol=1e-13, atol=1e-15)
