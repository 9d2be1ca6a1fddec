"""include/arkcos_split.h - the specified arithmetic of the paper's kernel split (Eq. 2.1-2.4;
SURVEY.md §8(f) N4), checked against closed forms, scipy quadrature and brute-force numpy.  Host only."""
import math

import numpy as np
import pytest
from scipy import integrate, special

from paper_1211_3556_b200 import arkcos, split
from paper_1211_3556_b200 import workloads as wl
from tests import helpers as H


def test_library_exports_every_symbol_of_arkcos_split_h():
    import os
    import re
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "arkcos_split.h")).read()
    declared = set(re.findall(r"\b(arkcos_[a-z_]+)\s*\(", hdr))
    assert declared == {name for name, _, _ in split.SYMBOLS}
    lib = arkcos.lib()
    for name in declared:
        assert hasattr(lib, name)


def test_legendre_closed_forms():
    # K = 1 on the whole sphere: b_0 = 4 pi, every other b_l = 0 (orthogonality)
    b = split.table_legendre(np.ones(4001), math.pi, 40)
    assert abs(b[0] - 4.0 * math.pi) < 1e-12 and np.abs(b[1:]).max() < 1e-12
    # K = cos(theta) = P_1: b_1 = 4 pi / 3, others 0 (up to the linear-interpolation error h^2/8 of the table)
    th = np.linspace(0.0, math.pi, 20001)
    b = split.table_legendre(np.cos(th), math.pi, 10)
    assert abs(b[1] - 4.0 * math.pi / 3.0) < 1e-7 and np.abs(np.delete(b, 1)).max() < 1e-7
    # a resolved narrow Gaussian: b_l -> exp(-l(l+1) sigma^2 / 2) (flat-sky limit, corrections O(sigma^2))
    sig = math.radians(1.0)
    b = split.table_legendre(wl.gaussian_table(sig, 8 * sig, 8193), 8 * sig, 200)
    ell = np.arange(201)
    assert np.abs(b - np.exp(-0.5 * ell * (ell + 1) * sig * sig)).max() < 2e-4


@pytest.mark.parametrize("m_split", [0, 6])
def test_legendre_matches_scipy_quadrature_of_the_interpolant(m_split):
    """independent statement: integrate numpy.interp(theta; nodes, table) * P_l(cos) * sin cell by cell with QUADPACK"""
    cut, n = 0.9, 13
    t_split = cut / 5.0
    nodes = wl.biased_nodes(cut, n, m_split, t_split) if m_split else wl.table_nodes(cut, n)
    table = np.cos(9.0 * nodes) * np.exp(-nodes)
    got = split.table_legendre(table, cut, 60, m_split=m_split, theta_split=t_split if m_split else 0.0)
    for ell in (0, 1, 2, 7, 31, 60):
        f = lambda t: np.interp(t, nodes, table) * special.eval_legendre(ell, math.cos(t)) * math.sin(t)   # noqa: E731
        ref = 2.0 * math.pi * sum(integrate.quad(f, nodes[m], nodes[m + 1], epsabs=1e-14, epsrel=1e-13)[0] for m in range(n - 1))
        assert abs(got[ell] - ref) < 1e-12, (ell, got[ell], ref)


def test_legendre_agrees_with_the_b_l_that_pins_the_oracle():
    """tests/helpers.gauss_legendre_cells is what the oracle's Y_lm pin uses (convolution theorem)"""
    sig = math.radians(3.0); cut = 3 * sig
    table = wl.gaussian_table(sig, cut, 4096)
    b = split.table_legendre(table, cut, 20)
    for ell in (0, 3, 11, 20):
        ref = H.gauss_legendre_cells(table, cut, lambda t: special.eval_legendre(ell, np.cos(t)))
        assert abs(b[ell] - ref) < 1e-13


def numpy_sigma(k, b, l_cut, compensate, alpha):
    ell = np.arange(k.size)
    khat = np.where(ell <= l_cut, k - b if compensate else k, 0.0)
    kt = khat + b
    return alpha * math.sqrt(((2 * ell + 1) * (kt - k) ** 2).sum() / ((2 * ell + 1) * k ** 2).sum()), khat, kt


def test_split_error_eq_2_1_and_2_2():
    rng = np.random.default_rng(5)
    k = np.exp(-np.arange(65) / 20.0); b = k * (1.0 + 0.05 * rng.standard_normal(65)) * (np.arange(65) > 3)
    for comp in (False, True):
        for l_cut in (-1, 0, 10, 64):
            s, khat, kt = split.split_error(k, b, l_cut, compensate=comp, alpha=5.0, full=True)
            s_ref, khat_ref, kt_ref = numpy_sigma(k, b, l_cut, comp, 5.0)
            assert abs(s - s_ref) <= 1e-13 * max(1.0, s_ref)
            np.testing.assert_allclose(khat, khat_ref, rtol=0, atol=1e-15); np.testing.assert_allclose(kt, kt_ref, rtol=0, atol=1e-15)
    # compensated split reproduces K_l exactly up to l_cut ("essentially zero error")
    s, khat, kt = split.split_error(k, b, 64, compensate=True, full=True)
    assert s == 0.0 and np.array_equal(kt, khat + b)
    with pytest.raises(arkcos.ArkcosError):
        split.split_error(k, b, 65)
    with pytest.raises(arkcos.ArkcosError):
        split.split_error(k, b * np.nan, 3)


def test_split_search_equals_brute_force_and_reports_no_solution():
    rng = np.random.default_rng(9)
    l_max = 96
    ell = np.arange(l_max + 1)
    k = np.exp(-ell * (ell + 1) * 2e-4)
    thetas = np.array([5.0, 10.0, 20.0, 40.0, 80.0])
    # wider cuts reproduce K_l better at high l
    b = np.stack([k * (1.0 - np.exp(-ell / (2.0 + c)) * 0.0 + 0.3 / (1 + c) ** 2 * rng.standard_normal(l_max + 1)) for c in range(5)])
    cost = dict(gpu_a2=1e-3, gpu_a1=0.0, gpu_c=0.1, cpu_full_s=160.0, cpu_l_ref=128.0)
    for comp in (True, False):
        for bound in (0.5, 0.1, 0.02):
            got = split.split_search(k, thetas, b, bound, compensate=comp, alpha=1.0, cost=cost)
            best = (-1, -1, math.inf, math.inf)
            for c in range(5):
                for l_cut in range(-1, l_max + 1):
                    s = numpy_sigma(k, b[c], l_cut, comp, 1.0)[0]
                    if s <= bound:      # smallest admissible l_cut of this candidate
                        t = max(1e-3 * thetas[c] ** 2 + 0.1, 160.0 * max(l_cut, 0) ** 2 * l_max / 128.0 ** 3)
                        if t < best[2]:
                            best = (c, l_cut, t, s)
                        break
            assert got[0] == best[0] and got[1] == best[1]
            if best[0] >= 0:
                assert abs(got[2] - best[2]) < 1e-12 and abs(got[3] - best[3]) < 1e-12
    assert split.split_search(k, thetas, b, 1e-30, compensate=False, alpha=1.0, cost=cost)[0] == -1


def test_gaussian_beam_split_scenario():
    """A worked scenario with what the paper specifies: K_l = B_l of a 30' beam (C_l = 1), real-space
    part = the beam truncated at theta_cut, l-space part compensated; wider cuts lower the estimated error (Eq. 2.2)
    and the search returns the pair that balances Eq. 2.3 against Eq. 2.4."""
    l_max = 768
    sig = math.radians(30.0 / 60.0) / math.sqrt(8.0 * math.log(2.0))
    # K_l = the exact Legendre transform of the (practically untruncated, 12 sigma) Gaussian beam; the flat-sky
    # exp(-l(l+1) sigma^2/2) differs from it by O(sigma^2) = 1e-5, which would mask the truncation error
    k = split.table_legendre(wl.gaussian_table(sig, 12 * sig, 32769), 12 * sig, l_max)
    cuts = np.array([20.0, 30.0, 45.0, 60.0, 90.0])
    b = np.stack([split.table_legendre(wl.gaussian_table(sig, math.radians(c / 60.0), 16385), math.radians(c / 60.0), l_max) for c in cuts])
    sig_plain = [split.split_error(k, b[i], -1, compensate=True) for i in range(cuts.size)]
    assert all(a > c for a, c in zip(sig_plain, sig_plain[1:])) and sig_plain[-1] < 1e-5 < sig_plain[0]
    for i in range(cuts.size):                         # the error is non-increasing in l_cut when compensated
        s = [split.split_error(k, b[i], lc, compensate=True) for lc in (-1, 50, 200, 768)]
        assert all(x >= y for x, y in zip(s, s[1:])) and s[-1] == 0.0
    cand, l_cut, t, s = split.split_search(k, cuts, b, 1e-5, compensate=True, alpha=5.0, cost=split.PAPER_COST)
    assert cand >= 0 and s <= 1e-5
    t_gpu = 0.0232 * cuts[cand] + 2.428
    t_cpu = 160.0 * max(l_cut, 0) ** 2 * l_max / 4096.0 ** 3
    assert abs(t - max(t_gpu, t_cpu)) < 1e-12


def test_split_search_consumes_a_b200_cost_curve_built_from_the_plans_work_counts():
    """The cost curve the split optimiser consumes (Eq. 2.3), for this library's direct sum on B200.
    NO measured B200 curve exists yet (GPU access closed): the curve here is a MODEL - the exact
    kernel-pixel evaluation counts of the real plans of configs[4] (theta_cut = 5, 10, 20, 40 arcmin on 4096 x 8192)
    divided by the FMA rate round 1 measured (58.4 % of 148 x 128 x 1.965e9 FMA/s, commit 2dde936).  It checks the
    pipeline plan work -> quadratic fit -> arkcos_split_search, and that a direct sum is quadratic, not linear, in
    theta_cut.  `bench.py --sweep` prints the same two fits from measured times."""
    rate = 0.584 * 148 * 128 * 1.965e9
    cuts, t = [], []
    for w in wl.config(4):
        with arkcos.Plan(w.n_theta, w.n_phi, np.ones(16), w.theta_cut, flags=arkcos.PLAN_HOST_ONLY) as plan:
            cuts.append(w.theta_cut / wl.ARCMIN)
            t.append(plan.work()[0] / rate)
    cuts, t = np.array(cuts), np.array(t)
    quad = np.linalg.lstsq(np.stack([cuts ** 2, np.ones_like(cuts)], 1), t, rcond=None)[0]
    lin = np.linalg.lstsq(np.stack([cuts, np.ones_like(cuts)], 1), t, rcond=None)[0]
    res_q = np.sqrt(np.mean((quad[0] * cuts ** 2 + quad[1] - t) ** 2))
    res_l = np.sqrt(np.mean((lin[0] * cuts + lin[1] - t) ** 2))
    assert quad[0] > 0 and res_q < 0.05 * t.max() and res_q < 0.2 * res_l        # the quadratic form fits, the linear does not
    assert 2e-3 < quad[0] * 40.0 ** 2 + quad[1] < 2e-2                            # ~5 ms per map at 40 arcmin
    # the Gaussian-beam scenario of the test above with this cost model in place of Eq. 2.3
    l_max = 768
    sig = math.radians(30.0 / 60.0) / math.sqrt(8.0 * math.log(2.0))
    k = split.table_legendre(wl.gaussian_table(sig, 12 * sig, 32769), 12 * sig, l_max)
    cand_cuts = np.array([20.0, 30.0, 45.0, 60.0, 90.0])
    b = np.stack([split.table_legendre(wl.gaussian_table(sig, math.radians(c / 60.0), 16385), math.radians(c / 60.0), l_max) for c in cand_cuts])
    b200 = dict(gpu_a2=float(quad[0]), gpu_a1=0.0, gpu_c=float(max(quad[1], 0.0)), cpu_full_s=160.0, cpu_l_ref=4096.0)
    c_b, l_b, t_b, s_b = split.split_search(k, cand_cuts, b, 1e-5, compensate=True, alpha=5.0, cost=b200)
    c_p, l_p, t_p, s_p = split.split_search(k, cand_cuts, b, 1e-5, compensate=True, alpha=5.0, cost=split.PAPER_COST)
    assert c_b >= 0 and s_b <= 1e-5
    t_gpu = b200["gpu_a2"] * cand_cuts[c_b] ** 2 + b200["gpu_c"]
    assert abs(t_b - max(t_gpu, 160.0 * max(l_b, 0) ** 2 * l_max / 4096.0 ** 3)) < 1e-12
    # a GPU half that costs milliseconds moves the optimum to the wider cut / the smaller l_cut, and the pair is faster
    assert c_b >= c_p and l_b <= l_p and t_b < t_p
