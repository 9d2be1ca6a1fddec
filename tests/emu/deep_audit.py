"""Deep audit of the host emulation (test infrastructure; not part of the pytest suite because it takes ~10 minutes
on 8 cores): about one in ten work items of the REAL schedule of every full-size BASELINE workload - the launch
bench.py times, with the workloads' own maps and tables - runs through the emulated S2 generator and both
convolution kernels (plus the tensor-core WIDE kernel on three workloads) and is compared with the oracle.

    python tests/emu/deep_audit.py [--jobs 8] > profiles/<name>.txt

One line per workload: fraction of the map written by the emulated items, rel-rms and max error against the oracle
on <= 60000 of the written pixels, PASS/FAIL at the north_star tolerance (1e-6 / 1e-5 x rms)."""
import argparse
import math
import os
import pathlib
import sys
import tempfile
import time
from concurrent.futures import ProcessPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

# (config, index in the config, every n-th work item, tensor-core WIDE kernel)
JOBS = [(1, 0, 3, False), (2, 0, 13, False), (3, 0, 7, False), (3, 1, 9, False), (3, 2, 11, False), (3, 3, 13, False),
        (4, 0, 11, False), (4, 1, 13, False), (4, 2, 23, False), (4, 3, 47, False),
        (2, 0, 29, True), (3, 3, 31, True), (4, 3, 101, True)]


def job(args):
    cfg, k, stride, tensor = args
    os.environ["OMP_NUM_THREADS"] = "1"
    from oracle import oracle
    from paper_1211_3556_b200 import workloads as wl
    from tests.test_emu_parity import EMU_BIN, emulate
    w = wl.config(cfg)[k]
    x32, table = w.map_f32(), w.table()
    env = {"EMU_ITEM_STRIDE": str(stride)}
    if tensor:
        env["EMU_WIDE_TENSOR"] = "1"
    t0 = time.time()
    with tempfile.TemporaryDirectory() as d:
        got, log = emulate(EMU_BIN, pathlib.Path(d), x32, table, w.theta_cut, env=env, only="only_wide" if tensor else None)
    written = ~np.isnan(got)
    pix = np.flatnonzero(written.reshape(-1))
    pix = pix[:: max(1, len(pix) // 60000)]
    expect = oracle.convolve(x32, table, w.theta_cut, level=1, pixels=pix)
    rms = math.sqrt((got[written] ** 2).mean())
    err = got.reshape(-1)[pix] - expect
    rel, mx = math.sqrt((err ** 2).mean()) / rms, float(np.abs(err).max()) / rms
    items = log.strip().split("items ")[-1].split(" smem")[0]
    return (f"{w.name:34s} every {stride:3d}th item  wide path {'tensor' if tensor else 'ffma  '}  items {items:22s} map written {written.mean():.3f}  "
            f"rel-rms {rel:.2e}  max/rms {mx:.2e}  {'PASS' if rel <= 1e-6 and mx <= 1e-5 else 'FAIL'}  ({time.time() - t0:.0f} s)")


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--jobs", type=int, default=8)
    a = ap.parse_args()
    from tests.test_emu_parity import build_emu_binary
    build_emu_binary()
    with ProcessPoolExecutor(a.jobs) as ex:
        for line in ex.map(job, JOBS):
            print(line, flush=True)
