"""ctypes binding of include/arkcos_split.h (argument marshalling only): the specified arithmetic of the
paper's kernel split - Legendre transform of the truncated table (Eq. 2.1), error estimate (Eq. 2.2),
cost models (Eq. 2.3 / 2.4) and the equal-time search.  Host only, no device needed."""
from __future__ import annotations

import ctypes
from typing import Optional, Tuple

import numpy as np

from . import arkcos as _a


class CostModel(ctypes.Structure):
    """t_gpu = a2*theta^2 + a1*theta + c [s], theta in arcmin;  t_cpu = cpu_full_s * l_cut^2 * l_max / cpu_l_ref^3."""
    _fields_ = [("gpu_a2", ctypes.c_double), ("gpu_a1", ctypes.c_double), ("gpu_c", ctypes.c_double),
                ("cpu_full_s", ctypes.c_double), ("cpu_l_ref", ctypes.c_double)]


PAPER_COST = dict(gpu_a2=0.0, gpu_a1=0.0232, gpu_c=2.428, cpu_full_s=160.0, cpu_l_ref=4096.0)   # Eq. 2.3, Eq. 2.4

# every symbol include/arkcos_split.h declares
SYMBOLS = [
    ("arkcos_table_legendre", ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_double,
                                             ctypes.c_int, ctypes.c_void_p]),
    ("arkcos_split_error", ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                          ctypes.c_double, ctypes.POINTER(ctypes.c_double), ctypes.c_void_p, ctypes.c_void_p]),
    ("arkcos_split_search", ctypes.c_int, [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p,
                                           ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.POINTER(CostModel),
                                           ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int),
                                           ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]),
]
_bound = False


def _lib():
    global _bound
    lib = _a.lib()
    if not _bound:
        for name, res, args in SYMBOLS:
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _bound = True
    return lib


def table_legendre(k_table, theta_cut: float, l_max: int, m_split: int = 0, theta_split: float = 0.0) -> np.ndarray:
    t = np.ascontiguousarray(k_table, dtype=np.float64)
    b = np.empty(int(l_max) + 1 if l_max >= 0 else 1, dtype=np.float64)
    _a._check(_lib().arkcos_table_legendre(t.ctypes.data, int(t.size), float(theta_cut), int(m_split), float(theta_split),
                                           int(l_max), b.ctypes.data), "arkcos_table_legendre")
    return b


def split_error(k_l, b_l, l_cut: int, compensate: bool = True, alpha: float = 5.0, full: bool = False):
    k = np.ascontiguousarray(k_l, dtype=np.float64); b = np.ascontiguousarray(b_l, dtype=np.float64)
    if k.shape != b.shape or k.ndim != 1:
        raise ValueError("k_l and b_l must be 1-D arrays of equal length l_max+1")
    sigma = ctypes.c_double(0.0)
    khat = np.empty_like(k) if full else None
    ktil = np.empty_like(k) if full else None
    _a._check(_lib().arkcos_split_error(k.ctypes.data, b.ctypes.data, int(k.size) - 1, int(l_cut), int(bool(compensate)),
                                        float(alpha), ctypes.byref(sigma), khat.ctypes.data if full else None,
                                        ktil.ctypes.data if full else None), "arkcos_split_error")
    return (sigma.value, khat, ktil) if full else sigma.value


def split_search(k_l, theta_cut_arcmin, b_l_cand, bound: float, compensate: bool = True, alpha: float = 5.0,
                 cost: Optional[dict] = None) -> Tuple[int, int, float, float]:
    """-> (best candidate index or -1, best l_cut, time of the parallel halves [s], its sigma)."""
    k = np.ascontiguousarray(k_l, dtype=np.float64)
    th = np.ascontiguousarray(theta_cut_arcmin, dtype=np.float64)
    b = np.ascontiguousarray(b_l_cand, dtype=np.float64)
    if b.shape != (th.size, k.size):
        raise ValueError("b_l_cand must be [n_cand][l_max+1]")
    cm = CostModel(**(cost or PAPER_COST))
    bc, bl = ctypes.c_int(-1), ctypes.c_int(-1)
    bt, bs = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _a._check(_lib().arkcos_split_search(k.ctypes.data, int(k.size) - 1, int(th.size), th.ctypes.data, b.ctypes.data,
                                         int(bool(compensate)), float(alpha), float(bound), ctypes.byref(cm),
                                         ctypes.byref(bc), ctypes.byref(bl), ctypes.byref(bt), ctypes.byref(bs)),
              "arkcos_split_search")
    return bc.value, bl.value, bt.value, bs.value
