"""CPU tests of the C-ABI library: it loads, exports every symbol include/arkcos.h declares, and
its host-side ring-pair scheduler (step S1) agrees with brute force and with the oracle's pair count.
No compute call is made (no GPU here): plans are created with ARKCOS_PLAN_HOST_ONLY."""
import ctypes
import math
import os
import re

import numpy as np
import pytest

from oracle import oracle
from paper_1211_3556_b200 import arkcos
from paper_1211_3556_b200 import workloads as wl
from tests import helpers as H

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
DEG = math.pi / 180.0


def host_plan(n_theta, n_phi, cut, n_table=8):
    return arkcos.Plan(n_theta, n_phi, np.ones(n_table), cut, flags=arkcos.PLAN_HOST_ONLY)


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "arkcos.h")).read() + open(os.path.join(ROOT, "include", "arkcos_measure.h")).read() + open(os.path.join(ROOT, "include", "arkcos_spectral.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(arkcos_[a-z_]+)\s*\(", header))
    assert len(declared) >= 12
    bound = {name for name, _, _ in arkcos.SYMBOLS}
    assert declared == bound, (declared ^ bound)
    handle = ctypes.CDLL(arkcos.library_path()) if os.path.exists(arkcos.library_path()) else arkcos.lib()
    for name in declared:
        assert hasattr(handle, name), name
    assert arkcos.lib().arkcos_status_string(0) == b"ARKCOS_OK"


def test_argument_validation():
    t = np.ones(8)
    cases = [
        (0, 8, t, 0.5, arkcos.EINVAL), (4, 0, t, 0.5, arkcos.EINVAL), (4, 8, t, 0.0, arkcos.EINVAL),
        (4, 8, t, -1.0, arkcos.EINVAL), (4, 8, t, 3.2, arkcos.EINVAL), (4, 8, t, float("nan"), arkcos.EINVAL),
        (4, 8, np.ones(1), 0.5, arkcos.EINVAL), (4, 8, np.array([1.0, np.inf]), 0.5, arkcos.EINVAL),
        (4, 10, t, 0.5, arkcos.EUNSUPPORTED),
    ]
    for nt, nph, tab, cut, status in cases:
        with pytest.raises(arkcos.ArkcosError) as e:
            arkcos.Plan(nt, nph, tab, cut, flags=arkcos.PLAN_HOST_ONLY)
        assert e.value.status == status, (nt, nph, cut)
    with pytest.raises(arkcos.ArkcosError) as e:
        arkcos.Plan(4, 8, t, 0.5, flags=1024)
    assert e.value.status == arkcos.EINVAL


def test_host_only_plan_refuses_compute():
    p = host_plan(8, 16, 0.5)
    x = np.zeros((8, 16), dtype=np.float32)
    with pytest.raises(arkcos.ArkcosError) as e:
        p.convolve_host(x, x.copy())
    assert e.value.status == arkcos.EUNSUPPORTED
    with pytest.raises(arkcos.ArkcosError) as e:
        p.pair_weights(0, 0)
    assert e.value.status == arkcos.EUNSUPPORTED


def brute_windows(n_theta, n_phi, cut):
    """window[i][j] from atan2 angles of every dphi (independent of the library's haversine)."""
    theta, phi = H.centres(n_theta, n_phi)
    out = np.full((n_theta, n_theta), -1, dtype=np.int64)
    d = np.arange(n_phi)
    for i in range(n_theta):
        u = np.array([math.sin(theta[i]), 0.0, math.cos(theta[i])])
        for j in range(n_theta):
            v = np.stack([np.sin(theta[j]) * np.cos(phi[d]), np.sin(theta[j]) * np.sin(phi[d]),
                          np.full(n_phi, math.cos(theta[j]))], axis=-1)
            g = H.angle_atan2(u[None, :], v)
            inside = g <= cut
            if inside.all():
                out[i, j] = n_phi
            elif inside.any():
                dd = np.minimum(d, n_phi - d)[inside]
                out[i, j] = dd.max()
                assert inside.sum() == 2 * dd.max() + 1      # contiguous symmetric window
    return out


@pytest.mark.parametrize("n_theta,n_phi,cut_deg", [(12, 24, 33.0), (9, 16, 50.0), (16, 32, 7.0), (7, 12, 100.0),
                                                   (10, 20, 180.0), (64, 128, 9.0), (1, 4, 10.0), (3, 8, 61.0)])
def test_windows_match_brute_force(n_theta, n_phi, cut_deg):
    cut = cut_deg * DEG
    p = host_plan(n_theta, n_phi, cut)
    expect = brute_windows(n_theta, n_phi, cut)
    got = np.array([[p.window(i, j) for j in range(n_theta)] for i in range(n_theta)])
    assert (got == expect).all()
    assert (got == got[::-1, ::-1]).all()                    # N/S mirror, used by the FFMA2 pairing
    taps = np.where(expect == n_phi, n_phi, np.where(expect >= 0, 2 * expect + 1, 0))
    pe, w, r = p.work()
    assert w == taps.sum() and pe == taps.sum() * n_phi
    dth = math.pi / n_theta
    assert r == min(n_theta - 1, int(math.floor(cut / dth + 1e-12)))


def test_pair_evals_equal_the_oracles_pair_count_config0():
    w = wl.config(0)[0]
    p = arkcos.Plan(w.n_theta, w.n_phi, w.table(), w.theta_cut, flags=arkcos.PLAN_HOST_ONLY)
    _, pairs = oracle.convolve(w.map(), w.table(), w.theta_cut, level=0, return_pairs=True)
    assert p.work()[0] == pairs
    assert p.work()[2] == 3                                   # R = 3


@pytest.mark.parametrize("cfg,k,pairs,r", [(1, 0, 8.95e8, 5), (2, 0, 1.733e10, 5), (3, 0, 1.33e9, 3), (3, 3, 1.72e10, 12),
                                           (4, 0, 2.00e9, 1), (4, 3, 1.09e11, 15)])
def test_work_counts_of_the_baseline_configs(cfg, k, pairs, r):
    """SURVEY.md §8(d) table (computed independently during the survey)."""
    w = wl.config(cfg)[k]
    p = host_plan(w.n_theta, w.n_phi, w.theta_cut)
    pe, nw, rr = p.work()
    assert rr == r
    assert abs(pe / pairs - 1.0) < 6e-3
    info = p.info()
    assert info.fma_slots >= pe and info.n_items > 0 and info.sm_count == 0
    assert info.kernels_per_convolve in (2, 3)          # generator + wide and/or narrow convolution kernel


def test_sampled_ring_pair_counts_match_oracle_on_config1():
    """Per-output-pixel tap counts of S1 == the oracle's in-support pair count for that pixel."""
    w = wl.config(1)[0]
    p = host_plan(w.n_theta, w.n_phi, w.theta_cut)
    x = np.zeros((w.n_theta, w.n_phi))
    table = w.table()
    for i in (0, 1, 5, 6, 7, 100, 511, 512, 1017, 1023):
        _, pairs = oracle.convolve(x, table, w.theta_cut, level=1, pixels=np.array([i * w.n_phi + 3]), return_pairs=True)
        taps = 0
        for j in range(max(0, i - 8), min(w.n_theta, i + 9)):
            d = p.window(i, j)
            taps += w.n_phi if d == w.n_phi else (2 * d + 1 if d >= 0 else 0)
        assert taps == pairs, i
