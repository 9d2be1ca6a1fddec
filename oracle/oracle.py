"""ctypes loader for the FP64 CPU oracle (oracle/arkcos_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It builds `oracle/liboracle.so` with gcc on first use (plain C, -O2, OpenMP, no
fast-math) and exposes `convolve`, `ring_area`.  It imports nothing from the CUDA package.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "arkcos_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc if the .so is missing or older than the source."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-fno-fast-math",
                   "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True, capture_output=True, text=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_convolve.restype = ctypes.c_int
        lib.oracle_convolve.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p,
            ctypes.POINTER(ctypes.c_ulonglong), ctypes.c_int]
        lib.oracle_convolve_biased.restype = ctypes.c_int
        lib.oracle_convolve_biased.argtypes = [
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_double,
            ctypes.c_int, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p,
            ctypes.POINTER(ctypes.c_ulonglong), ctypes.c_int]
        lib.oracle_ring_area.restype = ctypes.c_int
        lib.oracle_ring_area.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
        lib.oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def ring_area(n_theta: int, n_phi: int) -> np.ndarray:
    a = np.empty(n_theta, dtype=np.float64)
    rc = _load().oracle_ring_area(n_theta, n_phi, a.ctypes.data)
    if rc != 0:
        raise ValueError(f"oracle_ring_area rc={rc}")
    return a


def convolve(map_in: np.ndarray, table: np.ndarray, theta_cut: float, *, level: int = 1,
             pixels: Optional[np.ndarray] = None, n_threads: int = 0,
             return_pairs: bool = False, m_split: int = 0, theta_split: float = 0.0):
    """out = map (*) K(theta <= theta_cut), FP64.

    m_split > 0: two-zone table: node m_split sits at theta_split, nodes are uniform on
    either side of it.

    map_in  [n_theta][n_phi], any float dtype (promoted exactly to FP64)
    table   K at theta_m = m*theta_cut/(n_table-1), FP64
    pixels  optional flat output-pixel indices; result has that shape.  None: the whole map.
    """
    x = np.ascontiguousarray(map_in, dtype=np.float64)
    if x.ndim != 2:
        raise ValueError("map must be [n_theta][n_phi]")
    n_theta, n_phi = x.shape
    t = np.ascontiguousarray(table, dtype=np.float64)
    if pixels is None:
        pix_ptr, n_pix = None, n_theta * n_phi
        out = np.empty((n_theta, n_phi), dtype=np.float64)
    else:
        pix = np.ascontiguousarray(pixels, dtype=np.int64)
        pix_ptr, n_pix = pix.ctypes.data, pix.size
        out = np.empty(pix.shape, dtype=np.float64)
    pairs = ctypes.c_ulonglong(0)
    rc = _load().oracle_convolve_biased(level, n_theta, n_phi, t.ctypes.data, t.size, float(theta_cut),
                                        int(m_split), float(theta_split),
                                        x.ctypes.data, pix_ptr, n_pix, out.ctypes.data,
                                        ctypes.byref(pairs), int(n_threads))
    if rc != 0:
        raise ValueError(f"oracle_convolve rc={rc}")
    if return_pairs:
        return out, int(pairs.value)
    return out


def ring_pixels(n_phi: int, rings) -> np.ndarray:
    """Flat indices of every pixel of the listed rings (helper for sampled parity checks)."""
    rings = np.asarray(rings, dtype=np.int64)
    return (rings[:, None] * n_phi + np.arange(n_phi, dtype=np.int64)[None, :]).reshape(-1)
