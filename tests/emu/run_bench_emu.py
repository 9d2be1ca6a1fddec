"""Runs bench.py's own code (argument parsing, measure(), the e2e leg through arkcos_convolve_host, build_line, the
cpu_baseline and reference legs) WITHOUT a GPU: the C-ABI library is the host-emulated one (tests/emu/run_emu_api.py)
and the few torch.cuda calls bench.py makes are replaced by host stand-ins ("device" tensors live in the emulated
cudaMalloc memory, events read the wall clock).  Test infrastructure only; executed in a subprocess by
tests/test_bench_emu.py.  The numbers it prints are meaningless; the point is that every line of bench.py has run and
that the JSON line carries the keys the measurement contract asks for before the first run on hardware.

    python tests/emu/run_bench_emu.py <bench.py arguments>"""
import contextlib
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
_argv = sys.argv[1:]
sys.argv = sys.argv[:1]

import torch  # noqa: E402

from tests.emu import run_emu_api as R  # noqa: E402  (builds and loads the emulated library; arkcos._lib points at it)


def _to_dev(t):
    a = np.ascontiguousarray(t.detach().numpy())
    return torch.from_numpy(R.dev(a, dtype=a.dtype))


def _like(t, value):
    d = R.dev(tuple(t.shape), dtype=np.float32)
    d[...] = value
    return torch.from_numpy(d)


_empty = torch.empty


def _empty_dev(*a, **k):
    on_device = k.pop("device", None) is not None
    t = _empty(*a, **k)
    if on_device and t.dtype == torch.uint8:
        return torch.from_numpy(R.dev((max(1, t.numel()),), dtype=np.uint8))
    return t


class _Stream:
    cuda_stream = 0

    def synchronize(self):
        pass


class _Event:
    def __init__(self, **k):
        self.t = 0.0

    def record(self, stream=None):
        self.t = time.perf_counter()

    def elapsed_time(self, other):
        return max(1e-3, 1e3 * (other.t - self.t))


torch.Tensor.to = lambda self, *a, **k: _to_dev(self)
torch.Tensor.pin_memory = lambda self, *a, **k: self
torch.empty_like = lambda t, **k: _like(t, 0.0)
torch.empty = _empty_dev
torch.device = lambda *a, **k: "cuda:0"
torch.cuda.is_available = lambda: True
torch.cuda.set_device = lambda *a, **k: None
torch.cuda.synchronize = lambda *a, **k: None
torch.cuda.Stream = lambda *a, **k: _Stream()
torch.cuda.stream = lambda s: contextlib.nullcontext()
torch.cuda.Event = _Event
torch.cuda.get_device_name = lambda *a, **k: "host emulation"

import bench  # noqa: E402

if __name__ == "__main__":
    sys.argv = ["bench.py"] + _argv
    sys.exit(bench.main())
