"""Pins of the FP64 CPU oracle against what the mathematics fixes (no GPU; `-m "not gpu"`).

The paper prints no convolution output, so the oracle is pinned by closed forms,
exact invariants and an independent numpy all-pairs sum (SURVEY.md §8(c) "What pins each part"):
a dropped area factor, a transposed ring index (A_i for A_j), a wrong node convention, a sign error
in phi, an exclusive support test or a too-narrow level-1 window each fail at least one test here.
"""
import math

import numpy as np
import pytest
from scipy.special import eval_legendre

from oracle import oracle
from paper_1211_3556_b200 import workloads as wl
from tests import helpers as H

DEG = math.pi / 180.0


# ---------------------------------------------------------------- area -------------------------
@pytest.mark.parametrize("n_theta,n_phi", [(1, 4), (7, 12), (64, 128), (4096, 8192)])
def test_ring_areas_tile_the_sphere(n_theta, n_phi):
    a = oracle.ring_area(n_theta, n_phi)
    assert abs(a.sum() * n_phi - 4.0 * math.pi) < 1e-12 * 4.0 * math.pi
    np.testing.assert_allclose(a, H.area_by_sine(n_theta, n_phi), rtol=1e-9, atol=0)
    np.testing.assert_allclose(a, a[::-1], rtol=1e-9)          # N/S symmetric


# ---------------------------------------------------------------- delta input -------------------
@pytest.mark.parametrize("j0,k0", [(0, 0), (3, 17), (31, 64), (63, 127), (40, 5)])
def test_delta_input_gives_area_times_kernel(j0, k0):
    """in = delta at (j0,k0)  =>  out[i,k] = A_{j0} K(gamma) inside the cut, exactly 0 outside.
    gamma from atan2 (independent of the oracle's chord); K from numpy.interp."""
    w = wl.config(0)[0]
    nt, nph = w.n_theta, w.n_phi
    table = w.table()
    x = np.zeros((nt, nph)); x[j0, k0] = 1.0
    out = oracle.convolve(x, table, w.theta_cut, level=1)
    v = H.unit_vectors(nt, nph)
    g = H.angle_atan2(v, v[j0 * nph + k0][None, :]).reshape(nt, nph)
    nodes = np.linspace(0.0, w.theta_cut, w.n_table)
    area = H.area_by_sine(nt, nph)
    expect = np.where(g <= w.theta_cut, np.interp(g, nodes, table) * area[j0], 0.0)
    # margin: no pixel of this grid sits within 1e-9 rad of the cut (else the two angle formulas could disagree)
    assert np.abs(g - w.theta_cut).min() > 1e-9
    assert (out[g > w.theta_cut] == 0.0).all()
    np.testing.assert_allclose(out, expect, rtol=1e-11, atol=1e-16)
    # ... and against the ANALYTIC Gaussian within the linear-interpolation error bound h^2 K''/8
    hh = w.theta_cut / (w.n_table - 1)
    k0_ = 1.0 / (2 * math.pi * w.sigma ** 2)
    bound = hh * hh * (k0_ / w.sigma ** 2) / 8.0 * area[j0] * 1.01 + 1e-16
    analytic = np.where(g <= w.theta_cut, wl.gaussian_profile(g, w.sigma) * area[j0], 0.0)
    assert np.abs(out - analytic).max() <= bound


def test_delta_input_uses_input_ring_area_not_output_ring_area():
    """A transposed area index would pass symmetric tests; this one is asymmetric by construction."""
    nt, nph = 16, 32
    cut = 40 * DEG
    table = np.ones(64)                       # K == 1 inside the cut
    x = np.zeros((nt, nph)); x[2, 0] = 1.0    # input near the pole, small area
    out = oracle.convolve(x, table, cut, level=0)
    area = H.area_by_sine(nt, nph)
    assert out[5, 0] == pytest.approx(area[2], rel=1e-12)
    assert abs(out[5, 0] - area[5]) > 0.3 * area[5]


# ---------------------------------------------------------------- brute force on tiny maps ------
@pytest.mark.parametrize("n_theta,n_phi,cut_deg,n_table", [
    (6, 8, 50.0, 17), (9, 16, 33.0, 33), (12, 24, 180.0, 9), (5, 12, 100.0, 5), (1, 4, 95.0, 3)])
@pytest.mark.parametrize("level", [0, 1])
def test_matches_independent_numpy_all_pairs_sum(n_theta, n_phi, cut_deg, n_table, level):
    rng = np.random.default_rng(n_theta * 100 + n_phi)
    cut = cut_deg * DEG
    table = rng.standard_normal(n_table)       # arbitrary, sign-changing kernel
    x = rng.standard_normal((n_theta, n_phi))
    m, n_inside = H.all_pairs_matrix(n_theta, n_phi, table, cut)
    expect = (m @ x.reshape(-1)).reshape(n_theta, n_phi)
    out, pairs = oracle.convolve(x, table, cut, level=level, return_pairs=True)
    np.testing.assert_allclose(out, expect, rtol=1e-12, atol=1e-13 * np.abs(expect).max())
    assert pairs == n_inside


# ---------------------------------------------------------------- level 1 == level 0 ------------
def test_level1_equals_level0_on_config0():
    w = wl.config(0)[0]
    x, table = w.map(), w.table()
    o0, p0 = oracle.convolve(x, table, w.theta_cut, level=0, return_pairs=True)
    o1, p1 = oracle.convolve(x, table, w.theta_cut, level=1, return_pairs=True)
    assert p0 == p1
    assert p0 == 770_432 or abs(p0 - 7.70e5) < 0.01e5      # 7.70e5 pair evals
    np.testing.assert_allclose(o1, o0, rtol=0, atol=1e-14 * np.abs(o0).max())


@pytest.mark.parametrize("cut_deg", [1.0, 7.3, 29.0, 91.0, 180.0])
def test_level1_equals_level0_small_grid_any_cut(cut_deg):
    rng = np.random.default_rng(5)
    nt, nph = 20, 40
    x = rng.standard_normal((nt, nph)); table = rng.standard_normal(50)
    o0, p0 = oracle.convolve(x, table, cut_deg * DEG, level=0, return_pairs=True)
    o1, p1 = oracle.convolve(x, table, cut_deg * DEG, level=1, return_pairs=True)
    assert p0 == p1
    np.testing.assert_allclose(o1, o0, rtol=0, atol=1e-13 * max(1e-300, np.abs(o0).max()))


def test_level1_equals_level0_at_planck_scale_polar_pixels():
    """The acos window of level 1 (arkcos_oracle.c: pixel_level1) at configs[2]'s polar sin(theta) ~ 4e-4 and at the
    configs[4]-40' cut, where (cos cut - cos t_i cos t_j)/(sin t_i sin t_j) is a ratio of two tiny numbers: level 1
    must visit every in-support pair level 0 (ALL 33.5 M input pixels per output pixel) finds.  ~12 pixels x 2 cuts."""
    rng = np.random.default_rng(11)
    x = rng.standard_normal((4096, 8192))
    for w in (wl.config(2)[0], wl.config(4)[3]):
        table = w.table()
        r = int(w.theta_cut / (math.pi / w.n_theta))
        rings = [0, 1, 2, r, r + 1, 2 * r + 3]
        pix = np.array([i * w.n_phi + int(k) for i in rings for k in (0, int(rng.integers(1, w.n_phi)))][:6] +
                       [(w.n_theta - 1) * w.n_phi + 7, (w.n_theta - 1 - r) * w.n_phi + 8191], dtype=np.int64)
        o0, p0 = oracle.convolve(x, table, w.theta_cut, level=0, pixels=pix, return_pairs=True)
        o1, p1 = oracle.convolve(x, table, w.theta_cut, level=1, pixels=pix, return_pairs=True)
        assert p0 == p1 and p0 > 1e4 * len(pix)
        np.testing.assert_allclose(o1, o0, rtol=0, atol=1e-13 * np.abs(o0).max())


def test_pixel_subset_matches_full_map():
    w = wl.config(0)[0]
    x, table = w.map(), w.table()
    full = oracle.convolve(x, table, w.theta_cut, level=1)
    pix = np.array([0, 5, 127, 128, 4000, 8191, 77, 77], dtype=np.int64)
    sub = oracle.convolve(x, table, w.theta_cut, level=1, pixels=pix)
    assert (sub == full.reshape(-1)[pix]).all()


# ---------------------------------------------------------------- exact invariants --------------
def test_phi_shift_and_mirror_equivariance():
    w = wl.config(0)[0]
    x, table = w.map(), w.table()
    base = oracle.convolve(x, table, w.theta_cut)
    for s in (1, 7, 64):
        rolled = oracle.convolve(np.roll(x, s, axis=1), table, w.theta_cut)
        assert np.abs(rolled - np.roll(base, s, axis=1)).max() < 1e-13 * np.abs(base).max()
    flipped = oracle.convolve(x[::-1].copy(), table, w.theta_cut)
    assert np.abs(flipped - base[::-1]).max() < 1e-13 * np.abs(base).max()
    # phi reflection k -> -k also commutes (kernel is radial)
    refl = oracle.convolve(np.roll(x[:, ::-1], 1, axis=1).copy(), table, w.theta_cut)
    assert np.abs(refl - np.roll(base[:, ::-1], 1, axis=1)).max() < 1e-13 * np.abs(base).max()


def test_area_weighted_self_adjointness():
    """A_i M_ij is symmetric:  sum_p A_p u_p (M v)_p == sum_p A_p v_p (M u)_p."""
    w = wl.config(0)[0]
    rng = np.random.default_rng(11)
    table = w.table()
    u = rng.standard_normal((w.n_theta, w.n_phi)); v = rng.standard_normal((w.n_theta, w.n_phi))
    a = oracle.ring_area(w.n_theta, w.n_phi)[:, None]
    mu = oracle.convolve(u, table, w.theta_cut); mv = oracle.convolve(v, table, w.theta_cut)
    l1 = (a * u * mv).sum(); l2 = (a * v * mu).sum()
    assert abs(l1 - l2) <= 1e-12 * abs(l1)


def test_linearity():
    w = wl.config(0)[0]
    rng = np.random.default_rng(12)
    table = w.table()
    u = rng.standard_normal((w.n_theta, w.n_phi)); v = rng.standard_normal((w.n_theta, w.n_phi))
    lhs = oracle.convolve(2.0 * u - 3.0 * v, table, w.theta_cut)
    rhs = 2.0 * oracle.convolve(u, table, w.theta_cut) - 3.0 * oracle.convolve(v, table, w.theta_cut)
    assert np.abs(lhs - rhs).max() < 1e-13 * np.abs(rhs).max()


# ---------------------------------------------------------------- closed forms ------------------
def _fine_table(w):
    """2^18 nodes: the midpoint rule integrates the KINKED piecewise-linear interpolant only to
    ~(theta_cut/n)^2/sigma^2; at 16384 nodes that residual is 7e-9, at 2^18 it is 2e-11 (measured)."""
    return wl.gaussian_table(w.sigma, w.theta_cut, 1 << 18)


def _interior(w):
    dth = math.pi / w.n_theta
    nex = int(math.ceil(w.theta_cut / dth)) + 2
    return slice(nex, w.n_theta - nex)


def test_constant_map_closed_form():
    """c -> c * sinc(dtheta/2) * 2 pi int_0^cut K sin(theta) dtheta on rings away from the poles;
    exactly ring-wise constant everywhere (SURVEY §8(c) 'normalisation, interior')."""
    w = wl.small_selfcheck_workload()
    table = _fine_table(w)
    c = 2.5
    out = oracle.convolve(np.full((w.n_theta, w.n_phi), c), table, w.theta_cut)
    assert np.abs(out - out[:, :1]).max() < 1e-13 * np.abs(out).max()       # depends on the ring only
    integral = H.gauss_legendre_cells(table, w.theta_cut, lambda t: np.ones_like(t))
    expect = c * H.sinc_half(w.n_theta) * integral
    sl = _interior(w)
    assert np.abs(out[sl] / expect - 1.0).max() < 1e-10


@pytest.mark.parametrize("l,m,part", [(0, 0, "cos"), (2, 1, "cos"), (7, 0, "cos"), (10, 3, "sin"),
                                      (20, 20, "cos"), (20, 1, "sin"), (20, 0, "cos")])
def test_ylm_input_is_scaled_by_legendre_coefficient(l, m, part):
    """Spherical convolution theorem: Y_lm (*) K = b_l Y_lm,
    b_l = 2 pi int K(t) P_l(cos t) sin t dt  (the Legendre transform P_l,theta),
    times the sinc(dtheta/2) of the exact-area weight, on interior rings."""
    w = wl.small_selfcheck_workload()
    table = _fine_table(w)
    theta, phi = wl.ecp_centres(w.n_theta, w.n_phi)
    y = wl.real_ylm(l, m, part, theta, phi)
    out = oracle.convolve(y, table, w.theta_cut)
    b_l = H.gauss_legendre_cells(table, w.theta_cut, lambda t: eval_legendre(l, np.cos(t)))
    expect = H.sinc_half(w.n_theta) * b_l * y
    sl = _interior(w)
    rms = math.sqrt((expect ** 2).mean())
    assert np.abs(out[sl] - expect[sl]).max() < 1e-9 * rms
    # b_l is not 1: the check is sensitive to the kernel normalisation and to l
    assert 0.05 < b_l < 1.0 or l == 0


def test_config0_constant_map_is_within_its_documented_3e3():
    """configs[0] as specified has a hard 1% jump at the cut and sigma ~ 1.07 px, so the continuum
    closed form only holds to ~3e-3 there; pin that number so a regression shows."""
    w = wl.config(0)[0]
    table = w.table()
    out = oracle.convolve(np.ones((w.n_theta, w.n_phi)), table, w.theta_cut)
    integral = H.gauss_legendre_cells(table, w.theta_cut, lambda t: np.ones_like(t))
    sl = _interior(w)
    dev = np.abs(out[sl] / (H.sinc_half(w.n_theta) * integral) - 1.0).max()
    assert 1e-4 < dev < 6e-3


def test_polar_error_converges_at_second_order():
    """Poles are not pinned by continuum closed forms (midpoint rule in theta); they converge at
    2nd order under refinement (SURVEY §8(c) 'polar rings')."""
    errs = []
    sigma = 3.0 * DEG
    for nt in (64, 128, 256):
        cut = 5.0 * sigma
        table = wl.gaussian_table(sigma, cut, 4096)
        theta, phi = wl.ecp_centres(nt, 2 * nt)
        y = wl.real_ylm(1, 0, "cos", theta, phi)
        pix = oracle.ring_pixels(2 * nt, [0])
        out = oracle.convolve(y, table, cut, pixels=pix)
        b1 = H.gauss_legendre_cells(table, cut, lambda t: eval_legendre(1, np.cos(t)))
        errs.append(abs(out[0] / (H.sinc_half(nt) * b1 * y[0, 0]) - 1.0))
    assert errs[0] > errs[1] > errs[2]
    assert 2.5 < errs[0] / errs[1] < 6.0 and 2.5 < errs[1] / errs[2] < 8.0


# ---------------------------------------------------------------- interpolation / conventions ---
def test_table_doubling_changes_result_at_second_order():
    w = wl.config(0)[0]
    x = w.map()
    ref = oracle.convolve(x, wl.gaussian_table(w.sigma, w.theta_cut, 65536), w.theta_cut)
    e = []
    for n in (257, 513, 1025):
        o = oracle.convolve(x, wl.gaussian_table(w.sigma, w.theta_cut, n), w.theta_cut)
        e.append(np.abs(o - ref).max())
    assert 2.5 < e[0] / e[1] < 5.5 and 2.5 < e[1] / e[2] < 5.5   # ~4x per doubling (discrete gammas: not exactly 4)


def test_support_edge_is_sharp_around_exact_ring_spacing():
    """theta_cut just inside / just outside 2 ring spacings on the same meridian: the support is a sharp disc.
    This does NOT tell `<` from `<=`: gamma == theta_cut exactly is decided by FP64 rounding of the unit vectors,
    not by the method (R3), and no config has a tap within 1e-7 of the cut."""
    nt, nph = 18, 36
    dth = math.pi / nt
    table = np.ones(8)
    x = np.zeros((nt, nph)); x[9, 0] = 1.0
    inside = oracle.convolve(x, table, 2 * dth * (1 + 1e-9), level=0)
    outside = oracle.convolve(x, table, 2 * dth * (1 - 1e-9), level=0)
    assert inside[7, 0] > 0 and inside[11, 0] > 0
    assert outside[7, 0] == 0 and outside[11, 0] == 0 and outside[8, 0] > 0


def test_invalid_arguments_are_rejected():
    x = np.zeros((4, 8)); t = np.ones(4)
    with pytest.raises(ValueError):
        oracle.convolve(x, t, 0.0)
    with pytest.raises(ValueError):
        oracle.convolve(x, t, 4.0)
    with pytest.raises(ValueError):
        oracle.convolve(x, np.ones(1), 1.0)
    with pytest.raises(ValueError):
        oracle.convolve(x, t, 1.0, pixels=np.array([32]))
