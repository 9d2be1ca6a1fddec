"""Thin ctypes binding of the C-ABI library (include/arkcos.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of `libarkcos.so`; PyTorch is used by callers
for device memory and streams (`tensor.data_ptr()`, `torch.cuda.current_stream().cuda_stream`).
There is no CPU fallback: if the library is missing it is built with nvcc (in-tree), and if that
fails the import error propagates.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

from . import build as _build

OK, EINVAL, ENOMEM, ECUDA, EUNSUPPORTED, EINTERNAL = 0, 1, 2, 3, 4, 5
PLAN_DEFAULT, PLAN_HOST_ONLY, PLAN_CACHE_WEIGHTS = 0, 1, 2
PLAN_ONLY_WIDE, PLAN_ONLY_NARROW = 4, 8      # measurement hooks (include/arkcos_measure.h)
PLAN_WIDE_TENSOR = 32                        # N1(a) experiment: WIDE items on the tensor cores (include/arkcos_measure.h)
PLAN_ALL_WIDE = 64                           # measurement hook: every ring in the WIDE class (include/arkcos_measure.h)
PLAN_SPECTRAL = 16                           # N2, the phi-spectral ring-pair path (include/arkcos_spectral.h)

_c_plan_p = ctypes.c_void_p


class PlanInfo(ctypes.Structure):
    _fields_ = [("n_theta", ctypes.c_int), ("n_phi", ctypes.c_int), ("n_table", ctypes.c_int),
                ("theta_cut", ctypes.c_double), ("ring_halfband", ctypes.c_int),
                ("pair_evals", ctypes.c_ulonglong), ("weights", ctypes.c_ulonglong),
                ("fma_slots", ctypes.c_ulonglong), ("weight_slots", ctypes.c_ulonglong),
                ("n_items", ctypes.c_int), ("n_gen_units", ctypes.c_int),
                ("kernels_per_convolve", ctypes.c_int), ("sm_count", ctypes.c_int),
                ("flags", ctypes.c_uint), ("device_bytes", ctypes.c_ulonglong),
                ("fma_slots_wide", ctypes.c_ulonglong), ("first_narrow_ring", ctypes.c_int)]


class ArkcosError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().arkcos_status_string(status).decode()
        cuda = lib().arkcos_last_cuda_error().decode()
        super().__init__(f"{where}: {msg}" + (f" [{cuda}]" if status == ECUDA and cuda else ""))


_lib = None

# every symbol include/arkcos.h, arkcos_measure.h and arkcos_spectral.h declare: (name, restype, argtypes)
SYMBOLS = [
    ("arkcos_plan_create", ctypes.c_int, [ctypes.POINTER(_c_plan_p), ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                          ctypes.c_int, ctypes.c_double]),
    ("arkcos_plan_create_ex", ctypes.c_int, [ctypes.POINTER(_c_plan_p), ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                             ctypes.c_int, ctypes.c_double, ctypes.c_uint]),
    ("arkcos_plan_create_biased", ctypes.c_int, [ctypes.POINTER(_c_plan_p), ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                                 ctypes.c_int, ctypes.c_double, ctypes.c_int, ctypes.c_double, ctypes.c_uint]),
    ("arkcos_convolve", ctypes.c_int, [_c_plan_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    ("arkcos_convolve_batch", ctypes.c_int, [_c_plan_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]),
    ("arkcos_convolve_host", ctypes.c_int, [_c_plan_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    ("arkcos_plan_reserve_host_io", ctypes.c_int, [_c_plan_p]),
    ("arkcos_plan_reserve_host_io_chunks", ctypes.c_int, [_c_plan_p, ctypes.c_int]),
    ("arkcos_plan_destroy", ctypes.c_int, [_c_plan_p]),
    ("arkcos_status_string", ctypes.c_char_p, [ctypes.c_int]),
    ("arkcos_last_cuda_error", ctypes.c_char_p, []),
    ("arkcos_plan_work", ctypes.c_int, [_c_plan_p, ctypes.POINTER(ctypes.c_ulonglong), ctypes.POINTER(ctypes.c_ulonglong),
                                        ctypes.POINTER(ctypes.c_int)]),
    ("arkcos_plan_get_info", ctypes.c_int, [_c_plan_p, ctypes.POINTER(PlanInfo)]),
    ("arkcos_plan_window", ctypes.c_int, [_c_plan_p, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]),
    ("arkcos_plan_pair_weights", ctypes.c_int, [_c_plan_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_int,
                                                ctypes.POINTER(ctypes.c_int)]),
    ("arkcos_measure_convolve", ctypes.c_int, [_c_plan_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p,
                                               ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_float)]),
    ("arkcos_plan_validate", ctypes.c_int, [_c_plan_p, ctypes.c_char_p, ctypes.c_int]),
    ("arkcos_spectral_workspace_bytes", ctypes.c_int, [_c_plan_p, ctypes.c_int, ctypes.POINTER(ctypes.c_ulonglong)]),
    ("arkcos_convolve_spectral", ctypes.c_int, [_c_plan_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p,
                                                ctypes.c_ulonglong, ctypes.c_void_p]),
    ("arkcos_plan_item", ctypes.c_int, [_c_plan_p, ctypes.c_int, ctypes.POINTER(ctypes.c_int)]),
]


def library_path() -> str:
    return _build.LIB


def lib():
    """Loads (building if needed) libarkcos.so and declares the prototypes.  Fails loudly."""
    global _lib
    if _lib is None:
        path = _build.build_library()
        handle = ctypes.CDLL(path)
        for name, restype, argtypes in SYMBOLS:
            fn = getattr(handle, name)          # AttributeError if the .so lacks a declared symbol
            fn.restype = restype
            fn.argtypes = argtypes
        _lib = handle
    return _lib


def _check(status: int, where: str):
    if status != OK:
        raise ArkcosError(status, where)


def _ptr(t) -> int:
    """Device/host pointer of a torch tensor or numpy array (contiguous FP32)."""
    if isinstance(t, np.ndarray):
        if t.dtype != np.float32 or not t.flags["C_CONTIGUOUS"]:
            raise TypeError("expected a C-contiguous float32 array")
        return t.ctypes.data
    if str(t.dtype) != "torch.float32" or not t.is_contiguous():
        raise TypeError("expected a contiguous float32 tensor")
    return t.data_ptr()


class Plan:
    """arkcos_plan_create / arkcos_plan_destroy with the same argument meaning as the C ABI."""

    def __init__(self, n_theta: int, n_phi: int, k_table, theta_cut: float, flags: int = PLAN_DEFAULT,
                 m_split: int = 0, theta_split: float = 0.0):
        """m_split > 0: arkcos_plan_create_biased (two-zone table, node m_split at theta_split)."""
        table = np.ascontiguousarray(k_table, dtype=np.float64)
        self._h = _c_plan_p()
        if m_split:
            _check(lib().arkcos_plan_create_biased(ctypes.byref(self._h), int(n_theta), int(n_phi), table.ctypes.data,
                                                   int(table.size), float(theta_cut), int(m_split), float(theta_split),
                                                   int(flags)), "arkcos_plan_create_biased")
        else:
            _check(lib().arkcos_plan_create_ex(ctypes.byref(self._h), int(n_theta), int(n_phi), table.ctypes.data,
                                               int(table.size), float(theta_cut), int(flags)), "arkcos_plan_create")
        self.n_theta, self.n_phi = int(n_theta), int(n_phi)

    # -- hot path -----------------------------------------------------------------------------
    def convolve(self, d_in, d_out, stream: int = 0):
        _check(lib().arkcos_convolve(self._h, _ptr(d_in), _ptr(d_out), stream), "arkcos_convolve")

    def convolve_batch(self, d_in, d_out, n_maps: int, stream: int = 0):
        _check(lib().arkcos_convolve_batch(self._h, _ptr(d_in), _ptr(d_out), int(n_maps), stream),
               "arkcos_convolve_batch")

    def convolve_host(self, h_in, h_out, stream: int = 0):
        _check(lib().arkcos_convolve_host(self._h, _ptr(h_in), _ptr(h_out), stream), "arkcos_convolve_host")

    def spectral_workspace_bytes(self, n_maps: int = 1) -> int:
        b = ctypes.c_ulonglong(0)
        _check(lib().arkcos_spectral_workspace_bytes(self._h, int(n_maps), ctypes.byref(b)), "arkcos_spectral_workspace_bytes")
        return int(b.value)

    def convolve_spectral(self, d_in, d_out, d_work, n_maps: int = 1, stream: int = 0):
        """d_work: a device tensor (any dtype) of at least spectral_workspace_bytes(n_maps) bytes, owned by the caller."""
        _check(lib().arkcos_convolve_spectral(self._h, _ptr(d_in), _ptr(d_out), int(n_maps), d_work.data_ptr(),
                                              int(d_work.numel() * d_work.element_size()), stream), "arkcos_convolve_spectral")

    def reserve_host_io(self, n_chunks: int = 0):
        _check(lib().arkcos_plan_reserve_host_io_chunks(self._h, int(n_chunks)), "arkcos_plan_reserve_host_io")

    def measure_convolve(self, d_in, d_out, stream: int = 0, n_maps: int = 1) -> Tuple[float, float]:
        a, b = ctypes.c_float(0), ctypes.c_float(0)
        _check(lib().arkcos_measure_convolve(self._h, _ptr(d_in), _ptr(d_out), int(n_maps), stream, ctypes.byref(a), ctypes.byref(b)),
               "arkcos_measure_convolve")
        return float(a.value), float(b.value)

    def items(self):
        """[(kind, ring, nrings, k0, n_out_phi, splits)] of the convolution launch (arkcos_plan_item)."""
        out = []
        f = (ctypes.c_int * 6)()
        for k in range(self.info().n_items):
            _check(lib().arkcos_plan_item(self._h, k, f), "arkcos_plan_item")
            out.append(tuple(int(v) for v in f))
        return out

    def validate(self) -> Tuple[int, str]:
        buf = ctypes.create_string_buffer(256)
        status = lib().arkcos_plan_validate(self._h, buf, 256)
        return int(status), buf.value.decode()

    # -- introspection ------------------------------------------------------------------------
    def work(self) -> Tuple[int, int, int]:
        pe, w, r = ctypes.c_ulonglong(0), ctypes.c_ulonglong(0), ctypes.c_int(0)
        _check(lib().arkcos_plan_work(self._h, ctypes.byref(pe), ctypes.byref(w), ctypes.byref(r)), "arkcos_plan_work")
        return int(pe.value), int(w.value), int(r.value)

    def info(self) -> PlanInfo:
        info = PlanInfo()
        _check(lib().arkcos_plan_get_info(self._h, ctypes.byref(info)), "arkcos_plan_get_info")
        return info

    def window(self, i: int, j: int) -> int:
        d = ctypes.c_int(0)
        _check(lib().arkcos_plan_window(self._h, int(i), int(j), ctypes.byref(d)), "arkcos_plan_window")
        return int(d.value)

    def pair_weights(self, i: int, j: int) -> np.ndarray:
        cap = self.n_phi // 2 + 1
        buf = np.empty(cap, dtype=np.float32)
        n = ctypes.c_int(0)
        _check(lib().arkcos_plan_pair_weights(self._h, int(i), int(j), buf.ctypes.data, cap, ctypes.byref(n)),
               "arkcos_plan_pair_weights")
        return buf[: n.value].copy()

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().arkcos_plan_destroy(self._h)
            self._h = _c_plan_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()
