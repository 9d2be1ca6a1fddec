"""Independent reference formulas used ONLY by tests to pin the oracle (numpy/scipy, FP64).

Nothing here is imported by the oracle or by the CUDA path.  The angle between pixel centres is
computed with atan2(|n x n'|, n.n') - a different formulation from the oracle's chord/asin and from
the CUDA plan's haversine - and interpolation is numpy.interp.
"""
import math

import numpy as np


def centres(n_theta, n_phi):
    theta = (np.arange(n_theta) + 0.5) * (math.pi / n_theta)
    phi = np.arange(n_phi) * (2.0 * math.pi / n_phi)
    return theta, phi


def unit_vectors(n_theta, n_phi):
    theta, phi = centres(n_theta, n_phi)
    st, ct = np.sin(theta)[:, None], np.cos(theta)[:, None]
    v = np.stack([st * np.cos(phi)[None, :], st * np.sin(phi)[None, :], ct + 0.0 * phi[None, :]], axis=-1)
    return v.reshape(-1, 3)


def angle_atan2(u, v):
    """Angle between unit vectors u[...,3], v[...,3], accurate for all separations."""
    cr = np.cross(u, v)
    return np.arctan2(np.sqrt((cr * cr).sum(-1)), (u * v).sum(-1))


def area_by_sine(n_theta, n_phi):
    """2 dphi sin(theta_j) sin(dtheta/2): the product-to-sum identity of cos(j dt) - cos((j+1) dt)."""
    theta, _ = centres(n_theta, n_phi)
    return 2.0 * (2.0 * math.pi / n_phi) * np.sin(theta) * math.sin(0.5 * math.pi / n_theta)


def all_pairs_matrix(n_theta, n_phi, table, theta_cut):
    """Dense operator M[p,q] = [gamma<=cut] * interp(table)(gamma) * A_q for tiny maps, plus the pair count."""
    v = unit_vectors(n_theta, n_phi)
    g = angle_atan2(v[:, None, :], v[None, :, :])
    nodes = np.linspace(0.0, theta_cut, len(table))
    k = np.interp(g, nodes, table)
    inside = g <= theta_cut
    area = np.repeat(area_by_sine(n_theta, n_phi), n_phi)
    return np.where(inside, k, 0.0) * area[None, :], int(inside.sum())


def gauss_legendre_cells(table, theta_cut, f, order=8):
    """2 pi * integral_0^cut K_lin(t) f(t) sin(t) dt, K_lin = the piecewise-linear table interpolant,
    integrated cell by cell with Gauss-Legendre (exact to rounding for smooth f)."""
    n = len(table)
    h = theta_cut / (n - 1)
    x, w = np.polynomial.legendre.leggauss(order)
    left = np.arange(n - 1)[:, None] * h
    t = left + 0.5 * h * (x[None, :] + 1.0)
    frac = 0.5 * (x[None, :] + 1.0)
    k = table[:-1, None] * (1.0 - frac) + table[1:, None] * frac
    return 2.0 * math.pi * float((k * f(t) * np.sin(t) * (0.5 * h * w[None, :])).sum())


def sinc_half(n_theta):
    a = 0.5 * math.pi / n_theta
    return math.sin(a) / a


def rel_rms(a, b):
    return float(np.sqrt(((a - b) ** 2).mean() / (b ** 2).mean()))
