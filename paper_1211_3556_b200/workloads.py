"""Seeded synthetic workloads: the five BASELINE.json `configs`, their maps and radial kernel tables.

This module serves BOTH the CUDA path and the CPU oracle (tests, bench) and therefore holds none of
the method's arithmetic: no ring geometry, no pixel areas, no support test, no interpolation, no
convolution.  It only produces *inputs*: a pixel map `[n_theta][n_phi]` and a radial kernel table
`K(theta_m)`, `theta_m = m * theta_cut / (n_table - 1)` (the library's input convention,
include/arkcos.h).

Recipes:
  * maps: i.i.d. N(0,1) from `numpy.random.default_rng(seed)`; the paper's test input is a
    "uniform-noise" (white) map at Planck resolution - these stand in for it.
  * kernels: Gaussian beam `exp(-t^2/2s^2)/(2 pi s^2)`, `s = FWHM/sqrt(8 ln 2)` (PAPER.md:L82
    "a Gaussian beam with a given FWHM"), or the residual of a Gaussian after removing its
    l <= 600 band-limited part (configs[4]; a synthetic stand-in for the paper's real-space split
    kernel).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Callable, List, Optional, Sequence, Tuple

import numpy as np

ARCMIN = math.pi / 180.0 / 60.0
DEG = math.pi / 180.0
FWHM_TO_SIGMA = 1.0 / math.sqrt(8.0 * math.log(2.0))


# --------------------------------------------------------------------------------------------
# radial kernels (inputs to the library: the table IS the kernel)
# --------------------------------------------------------------------------------------------
def gaussian_profile(theta: np.ndarray, sigma: float) -> np.ndarray:
    """Flat-sky normalised Gaussian beam profile K(theta)."""
    theta = np.asarray(theta, dtype=np.float64)
    return np.exp(-0.5 * (theta / sigma) ** 2) / (2.0 * math.pi * sigma * sigma)


def table_nodes(theta_cut: float, n_table: int) -> np.ndarray:
    """Uniform nodes theta_m = m*theta_cut/(n_table-1), both ends included."""
    return np.arange(n_table, dtype=np.float64) * (theta_cut / (n_table - 1))


def biased_nodes(theta_cut: float, n_table: int, m_split: int, theta_split: float) -> np.ndarray:
    """Nodes of the paper's two-zone table: node m_split sits at theta_split, the nodes are
    uniform on [0, theta_split] and on [theta_split, theta_cut].  The paper's choice: m_split = (n-1)/2,
    theta_split = theta_cut/16.  Where the caller samples K; the lookup itself is the library's and the
    oracle's own business."""
    inner = np.arange(m_split + 1, dtype=np.float64) * (theta_split / m_split)
    outer = theta_split + np.arange(1, n_table - m_split, dtype=np.float64) * ((theta_cut - theta_split) / (n_table - 1 - m_split))
    return np.concatenate([inner, outer])


def gaussian_table(sigma: float, theta_cut: float, n_table: int) -> np.ndarray:
    return gaussian_profile(table_nodes(theta_cut, n_table), sigma)


def legendre_sum(x: np.ndarray, coeff: np.ndarray) -> np.ndarray:
    """sum_l coeff[l] * P_l(x) by the three-term recurrence, FP64 (used only to BUILD an input)."""
    x = np.asarray(x, dtype=np.float64)
    p_prev = np.ones_like(x)
    acc = coeff[0] * p_prev
    if len(coeff) == 1:
        return acc
    p_cur = x.copy()
    acc = acc + coeff[1] * p_cur
    for l in range(1, len(coeff) - 1):
        p_next = ((2 * l + 1) * x * p_cur - l * p_prev) / (l + 1)
        p_prev, p_cur = p_cur, p_next
        acc = acc + coeff[l + 1] * p_cur
    return acc


def residual_profile(theta: np.ndarray, sigma: float, l_band: int) -> np.ndarray:
    """Gaussian beam minus its l <= l_band band-limited part:
    K_res = G(theta) - sum_{l<=l_band} (2l+1)/(4 pi) B_l P_l(cos theta), B_l = exp(-l(l+1) s^2/2)."""
    ell = np.arange(l_band + 1, dtype=np.float64)
    coeff = (2.0 * ell + 1.0) / (4.0 * math.pi) * np.exp(-0.5 * ell * (ell + 1.0) * sigma * sigma)
    theta = np.asarray(theta, dtype=np.float64)
    return gaussian_profile(theta, sigma) - legendre_sum(np.cos(theta), coeff)


def residual_table(sigma: float, l_band: int, theta_cut: float, n_table: int) -> np.ndarray:
    return residual_profile(table_nodes(theta_cut, n_table), sigma, l_band)


# --------------------------------------------------------------------------------------------
# maps
# --------------------------------------------------------------------------------------------
def ecp_centres(n_theta: int, n_phi: int) -> Tuple[np.ndarray, np.ndarray]:
    """Ring / pixel centre coordinates as configs[0] states them (grid description, not method)."""
    theta = (np.arange(n_theta, dtype=np.float64) + 0.5) * (math.pi / n_theta)
    phi = np.arange(n_phi, dtype=np.float64) * (2.0 * math.pi / n_phi)
    return theta, phi


def real_ylm(l: int, m: int, part: str, theta: np.ndarray, phi: np.ndarray) -> np.ndarray:
    """Real orthonormal spherical harmonic on the grid theta[:,None], phi[None,:].
    m = 0: Y_l0; m > 0: sqrt(2) Re Y_lm ('cos') or sqrt(2) Im Y_lm ('sin')."""
    from scipy.special import sph_harm_y

    y = sph_harm_y(l, m, theta[:, None], phi[None, :])
    if m == 0:
        return np.real(y) + 0.0 * phi[None, :]
    return math.sqrt(2.0) * (np.real(y) if part == "cos" else np.imag(y))


def white_map(n_theta: int, n_phi: int, seed: int, dtype=np.float32) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.standard_normal((n_theta, n_phi), dtype=dtype)


def draw_modes(seed: int, n_modes: int, l_max: int) -> List[Tuple[int, int, str]]:
    """n_modes seeded (l, m, cos|sin) triples, 1 <= l <= l_max, 0 <= m <= l."""
    rng = np.random.default_rng(seed)
    modes = []
    for _ in range(n_modes):
        l = int(rng.integers(1, l_max + 1))
        m = int(rng.integers(0, l + 1))
        part = "cos" if int(rng.integers(0, 2)) == 0 else "sin"
        modes.append((l, m, part))
    return modes


# --------------------------------------------------------------------------------------------
# the five configs of BASELINE.json
# --------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Workload:
    """One (grid, map recipe, kernel, theta_cut) case.  `theta_cut`-sweeps expand to several."""
    name: str
    n_theta: int
    n_phi: int
    theta_cut: float                    # radians
    n_table: int
    kernel: str                         # "gaussian" | "residual"
    sigma: float                        # radians
    map_seeds: Tuple[int, ...]          # one map per seed
    map_dtype: str = "float32"          # dtype the map is DRAWN in (configs[0]: float64)
    ylm_seed: Optional[int] = None      # configs[1]: add 8 real Y_lm modes
    ylm_amp: float = 10.0
    l_band: int = 600                   # residual kernel only
    note: str = ""

    @property
    def n_pix(self) -> int:
        return self.n_theta * self.n_phi

    def table(self) -> np.ndarray:
        """FP64 radial table, the library's kernel input."""
        if self.kernel == "gaussian":
            return gaussian_table(self.sigma, self.theta_cut, self.n_table)
        if self.kernel == "residual":
            return residual_table(self.sigma, self.l_band, self.theta_cut, self.n_table)
        raise ValueError(self.kernel)

    def map(self, which: int = 0) -> np.ndarray:
        """The `which`-th input map in the dtype it is drawn in."""
        dt = np.float64 if self.map_dtype == "float64" else np.float32
        x = white_map(self.n_theta, self.n_phi, self.map_seeds[which], dtype=dt)
        if self.ylm_seed is not None:
            theta, phi = ecp_centres(self.n_theta, self.n_phi)
            for (l, m, part) in draw_modes(self.ylm_seed, 8, 20):
                x = x + (self.ylm_amp * real_ylm(l, m, part, theta, phi)).astype(dt)
        return np.ascontiguousarray(x)

    def map_f32(self, which: int = 0) -> np.ndarray:
        """What the GPU receives: the FP32 rounding of the drawn map."""
        return np.ascontiguousarray(self.map(which).astype(np.float32))


def _g(fwhm_arcmin: float) -> float:
    return fwhm_arcmin * ARCMIN * FWHM_TO_SIGMA


def config(index: int) -> List[Workload]:
    """BASELINE.json configs[index] expanded over its theta_cut sweep (if any)."""
    if index == 0:
        return [Workload("cfg0_64x128_gauss3deg", 64, 128, 9.0 * DEG, 4096, "gaussian", 3.0 * DEG,
                         (0,), map_dtype="float64", note="FP64 map seed 0; sigma=3deg; cut=3 sigma")]
    if index == 1:
        return [Workload("cfg1_1024x2048_fwhm30", 1024, 2048, 60.0 * ARCMIN, 8192, "gaussian", _g(30.0),
                         (1,), ylm_seed=101, note="N(0,1) seed 1 + 8 real Y_lm (seed 101, amp 10)")]
    if index == 2:
        return [Workload("cfg2_planck_4096x8192_fwhm5", 4096, 8192, 15.0 * ARCMIN, 16384, "gaussian",
                         _g(5.0), (2,), note="Planck resolution; FWHM 5'; cut = 3 FWHM")]
    if index == 3:
        return [Workload(f"cfg3_2048x4096_fwhm33_cut{mult:g}x", 2048, 4096, mult * 33.0 * ARCMIN, 8192,
                         "gaussian", _g(33.0), (3,), note="wide beam; cost-vs-theta_cut sweep")
                for mult in (0.5, 1.0, 1.5, 2.0)]
    if index == 4:
        return [Workload(f"cfg4_4096x8192_resid10_cut{cut:g}", 4096, 8192, cut * ARCMIN, 16384,
                         "residual", _g(10.0), tuple(range(10, 18)), l_band=600,
                         note="batch of 8 maps; Gaussian FWHM 10' minus its l<=600 part")
                for cut in (5.0, 10.0, 20.0, 40.0)]
    raise IndexError(index)


def all_workloads() -> List[Workload]:
    out: List[Workload] = []
    for i in range(5):
        out.extend(config(i))
    return out


def by_name(name: str) -> Workload:
    for w in all_workloads():
        if w.name == name:
            return w
    raise KeyError(name)


def paper_regime_workload(theta_cut_arcmin: float = 240.0) -> Workload:
    """SURVEY §8(f) N3, second half: the paper's own radius.  PAPER.md:L104 (§3) works its example at
    theta_cut = 240 arcmin on nside 2048 (here: the 4096 x 8192 ECP grid that stands in for it, R = 91), with
    an oscillatory real-space split kernel; the residual kernel of configs[4] (Gaussian FWHM 10' minus its
    l <= 600 part) is the synthetic stand-in for the paper's fitted kernel (unspecified).
    Tabulated by the caller on the paper's two-zone nodes: see `biased_nodes`."""
    return Workload(f"paper_4096x8192_resid10_cut{theta_cut_arcmin:g}", 4096, 8192, theta_cut_arcmin * ARCMIN, 16384,
                    "residual", _g(10.0), (20,), l_band=600,
                    note="the paper's regime (PAPER.md:L104): theta_cut 240', oscillatory kernel; not a BASELINE config")


def small_selfcheck_workload() -> Workload:
    """SURVEY §8(c) 'recommended extra self-check configuration': 128x256, Gaussian FWHM 240',
    cut = 3 FWHM - the px-per-sigma ratios of configs[2], O(N^2) feasible."""
    return Workload("selfcheck_128x256_fwhm240", 128, 256, 720.0 * ARCMIN, 16384, "gaussian", _g(240.0),
                    (7,), map_dtype="float64")
