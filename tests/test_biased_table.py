"""The paper's two-zone ("biased") interpolation table, PAPER.md:L88 / SURVEY.md §8(f) N3:
"we place half the available interpolation nodes within the first 1/16th of the available support".

CPU part: pins the oracle's two-zone lookup against numpy.interp over the explicit node positions, checks
what the bias is for (a kernel that oscillates at small angles is interpolated far better with the same number
of nodes), the argument validation of arkcos_plan_create_biased, and the generator + convolution through the
host emulation.  GPU part (`gpu` marker): generated weights and a whole map against the oracle."""
import math
import os
import subprocess

import numpy as np
import pytest

from oracle import oracle
from paper_1211_3556_b200 import workloads as wl
from tests import helpers as H
from tests.test_emu_parity import emu_bin, emulate  # noqa: F401  (fixture + runner)

N_THETA, N_PHI = 48, 96
CUT = math.radians(17.3)
N_TABLE, M_SPLIT, T_SPLIT = 257, 128, CUT / 16.0     # the paper's bias: half the nodes in the first 1/16


def wiggly(theta):
    """oscillates fastest at small angles, like the split kernel of PAPER.md:L88"""
    return np.cos(40.0 * np.sqrt(theta / CUT)) * np.exp(-3.0 * theta / CUT) * 30.0


def biased_table():
    return wiggly(wl.biased_nodes(CUT, N_TABLE, M_SPLIT, T_SPLIT))


def test_nodes():
    nodes = wl.biased_nodes(CUT, N_TABLE, M_SPLIT, T_SPLIT)
    assert nodes.size == N_TABLE and nodes[0] == 0.0 and abs(nodes[-1] - CUT) < 1e-15
    assert abs(nodes[M_SPLIT] - T_SPLIT) < 1e-15 and (np.diff(nodes) > 0).all()
    assert (nodes <= T_SPLIT * (1 + 1e-12)).sum() == M_SPLIT + 1     # half the nodes in the first 1/16


def test_oracle_two_zone_lookup_matches_numpy_interp_on_delta_input():
    """delta input at (j0, k0): out[p] = A_j0 * K(gamma) inside the support, gamma by atan2, K by numpy.interp over
    the explicit (non-uniform) node positions - an independent statement of the two-zone table."""
    table = biased_table()
    nodes = wl.biased_nodes(CUT, N_TABLE, M_SPLIT, T_SPLIT)
    j0, k0 = 17, 5
    x = np.zeros((N_THETA, N_PHI)); x[j0, k0] = 1.0
    for level in (0, 1):
        got = oracle.convolve(x, table, CUT, level=level, m_split=M_SPLIT, theta_split=T_SPLIT)
        v = H.unit_vectors(N_THETA, N_PHI)
        g = H.angle_atan2(v, v[j0 * N_PHI + k0][None, :]).reshape(N_THETA, N_PHI)
        expect = np.where(g <= CUT, np.interp(g, nodes, table), 0.0) * H.area_by_sine(N_THETA, N_PHI)[j0]
        np.testing.assert_allclose(got, expect, rtol=1e-11, atol=1e-13 * np.abs(expect).max())
    # and it is NOT what the uniform reading of the same table gives
    uni = oracle.convolve(x, table, CUT, level=1)
    assert np.abs(uni - expect).max() > 1e-2 * np.abs(expect).max()


def test_bias_interpolates_a_small_angle_oscillation_better():
    """The reason for the bias: with the same number of nodes, the two-zone table follows a kernel
    that oscillates at small angles several times better than the uniform table."""
    fine = np.linspace(0.0, CUT, 200001)
    err_u = np.abs(np.interp(fine, wl.table_nodes(CUT, N_TABLE), wiggly(wl.table_nodes(CUT, N_TABLE))) - wiggly(fine)).max()
    nodes = wl.biased_nodes(CUT, N_TABLE, M_SPLIT, T_SPLIT)
    err_b = np.abs(np.interp(fine, nodes, wiggly(nodes)) - wiggly(fine)).max()
    assert err_b < 0.25 * err_u


def test_plan_create_biased_validates_its_arguments():
    from paper_1211_3556_b200 import arkcos
    t = np.ones(17)
    ok = arkcos.Plan(16, 32, t, 0.5, flags=arkcos.PLAN_HOST_ONLY, m_split=8, theta_split=0.5 / 16)
    ok.destroy()
    for m, ts in ((16, 0.1), (-1, 0.1), (8, 0.0), (8, 0.5), (8, 0.7), (8, float("nan"))):
        with pytest.raises(arkcos.ArkcosError):
            import ctypes
            h = ctypes.c_void_p()
            arkcos._check(arkcos.lib().arkcos_plan_create_biased(ctypes.byref(h), 16, 32, t.ctypes.data, 17, 0.5, m, ts,
                                                                 arkcos.PLAN_HOST_ONLY), "arkcos_plan_create_biased")


def test_emulated_generator_and_convolution_with_biased_table(emu_bin, tmp_path):  # noqa: F811
    table = biased_table()
    x32 = np.random.default_rng(11).standard_normal((N_THETA, N_PHI)).astype(np.float32)
    os.environ["EMU_M_SPLIT"], os.environ["EMU_THETA_SPLIT"] = str(M_SPLIT), repr(T_SPLIT)
    try:
        got, log = emulate(emu_bin, tmp_path, x32, table, CUT)
    finally:
        del os.environ["EMU_M_SPLIT"], os.environ["EMU_THETA_SPLIT"]
    expect = oracle.convolve(x32, table, CUT, level=1, m_split=M_SPLIT, theta_split=T_SPLIT)
    rms = math.sqrt((expect ** 2).mean())
    assert math.sqrt(((got - expect) ** 2).mean()) / rms <= 1e-6 and float(np.abs(got - expect).max()) / rms <= 1e-5, log


@pytest.mark.gpu
def test_gpu_biased_table_weights_and_map():
    import torch
    from paper_1211_3556_b200 import arkcos
    assert torch.cuda.is_available()
    table = biased_table()
    nodes = wl.biased_nodes(CUT, N_TABLE, M_SPLIT, T_SPLIT)
    theta, phi = H.centres(N_THETA, N_PHI)
    area = H.area_by_sine(N_THETA, N_PHI)
    x32 = np.random.default_rng(11).standard_normal((N_THETA, N_PHI)).astype(np.float32)
    with arkcos.Plan(N_THETA, N_PHI, table, CUT, m_split=M_SPLIT, theta_split=T_SPLIT) as plan:
        for (i, j) in [(0, 0), (3, 1), (23, 24), (24, 20), (47, 45)]:
            got = plan.pair_weights(i, j)
            dwin = plan.window(i, j)
            dmax = N_PHI // 2 if dwin == N_PHI else dwin
            u = np.array([math.sin(theta[i]), 0.0, math.cos(theta[i])])
            d = np.arange(dmax + 1)
            v = np.stack([math.sin(theta[j]) * np.cos(phi[d]), math.sin(theta[j]) * np.sin(phi[d]),
                          np.full(d.size, math.cos(theta[j]))], axis=-1)
            expect = area[j] * np.interp(H.angle_atan2(u[None, :], v), nodes, table)
            np.testing.assert_allclose(got, expect, rtol=1.2e-7, atol=2e-7 * np.abs(expect).max())
        d_in = torch.from_numpy(x32).cuda()
        d_out = torch.full_like(d_in, float("nan"))
        plan.convolve(d_in, d_out, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        got = d_out.cpu().numpy().astype(np.float64)
    expect = oracle.convolve(x32, table, CUT, level=1, m_split=M_SPLIT, theta_split=T_SPLIT)
    rms = math.sqrt((expect ** 2).mean())
    assert math.sqrt(((got - expect) ** 2).mean()) / rms <= 1e-6 and float(np.abs(got - expect).max()) / rms <= 1e-5


# ------------------------------------------------------------------ the paper's own regime (second half) ---
def paper_regime_table(w):
    """The oscillatory residual kernel of configs[4] on the paper's two-zone nodes: half the nodes in the first 1/16
    of the support."""
    m_split, t_split = (w.n_table - 1) // 2, w.theta_cut / 16.0
    nodes = wl.biased_nodes(w.theta_cut, w.n_table, m_split, t_split)
    return wl.residual_profile(nodes, w.sigma, w.l_band), m_split, t_split


def test_emulated_large_ring_band_with_the_papers_table(emu_bin, tmp_path):  # noqa: F811
    """A small-scale analogue of the paper's regime (theta_cut = 240' on nside 2048, R = 91): R = 23 ring
    half band (every ring WIDE, 47 input rows per output ring), an oscillatory kernel on the two-zone table."""
    n_theta, n_phi = 120, 256
    cut = 23.4 * math.pi / n_theta
    m_split, t_split = 128, cut / 16.0
    nodes = wl.biased_nodes(cut, 257, m_split, t_split)
    table = np.cos(9.0 * nodes / cut) * np.exp(-0.5 * (nodes / (0.35 * cut)) ** 2)
    x32 = np.random.default_rng(91).standard_normal((n_theta, n_phi)).astype(np.float32)
    os.environ["EMU_M_SPLIT"], os.environ["EMU_THETA_SPLIT"], os.environ["EMU_ITEM_STRIDE"] = str(m_split), repr(t_split), "3"
    try:
        got, log = emulate(emu_bin, tmp_path, x32, table, cut)
    finally:
        del os.environ["EMU_M_SPLIT"], os.environ["EMU_THETA_SPLIT"], os.environ["EMU_ITEM_STRIDE"]
    assert "R 23" in log, log
    written = ~np.isnan(got)
    pix = np.flatnonzero(written.reshape(-1))
    assert written.mean() > 0.25
    expect = oracle.convolve(x32, table, cut, level=1, pixels=pix, m_split=m_split, theta_split=t_split)
    rms = math.sqrt((expect ** 2).mean())
    err = got.reshape(-1)[pix] - expect
    assert math.sqrt((err ** 2).mean()) / rms <= 1e-6 and float(np.abs(err).max()) / rms <= 1e-5, log


@pytest.mark.gpu
def test_gpu_paper_regime_240_arcmin_sampled():
    """theta_cut = 240' on 4096 x 8192 (R = 91; 2.9e12 kernel-pixel evaluations), the residual kernel on the paper's
    two-zone table; sampled output pixels (poles, equator, seeded random) against the oracle."""
    import torch
    from paper_1211_3556_b200 import arkcos
    assert torch.cuda.is_available()
    w = wl.paper_regime_workload()
    table, m_split, t_split = paper_regime_table(w)
    x32 = w.map_f32()
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut, m_split=m_split, theta_split=t_split) as plan:
        assert plan.work()[2] == 91
        d_in = torch.from_numpy(x32).cuda()
        d_out = torch.full_like(d_in, float("nan"))
        plan.convolve(d_in, d_out, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        got = d_out.cpu().numpy()
    assert np.isfinite(got).all()
    rng = np.random.default_rng(240)
    ks = [0, 1, 31, 32, 1023, 1024, 1025, 4095, 4096, 8191]
    rings = [0, 1, 90, 91, 92, 183, 184, 1000, 2047, 2048, 4095 - 91, 4095]
    pix = np.array(sorted({i * w.n_phi + k for i in rings for k in ks} | {int(p) for p in rng.integers(0, w.n_pix, 300)}), dtype=np.int64)
    expect = oracle.convolve(x32, table, w.theta_cut, level=1, pixels=pix, m_split=m_split, theta_split=t_split)
    scale = math.sqrt((got.astype(np.float64) ** 2).mean())
    err = got.reshape(-1)[pix] - expect
    assert math.sqrt((err ** 2).mean()) / scale <= 1e-6 and float(np.abs(err).max()) / scale <= 1e-5
