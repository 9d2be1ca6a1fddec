"""Deep audit of the host emulation (test infrastructure; not part of the pytest suite: ~20 minutes on 8 cores).

    python tests/emu/deep_audit.py [--jobs 8] [--parts 8] > profiles/<name>.txt

EVERY work item of the REAL schedule of every full-size BASELINE workload - the launch bench.py times, with the
workloads' own maps and tables - runs through the emulated S2 generator and both convolution kernels (`--parts`
emulation processes per workload, each taking every parts-th item of the launch); the parts are merged, every output
pixel must have been written by exactly one work item, and <= 60000 evenly spaced pixels of the map are compared with
the oracle.  Three workloads are repeated with the WIDE items on the tensor-core kernel (N1(a); WIDE rings only).
One line per run: rel-rms and max error, PASS/FAIL at the north_star tolerance (1e-6 / 1e-5 x rms)."""
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

# (config, index, tensor-core WIDE kernel); config 9 = the paper's own regime (workloads.paper_regime_workload():
# theta_cut = 240', R = 91, the residual kernel on the paper's two-zone table; 2.9e12 evaluations, so only every
# 8th part of the launch runs and "exactly once" becomes "at most once")
RUNS = [(1, 0, False), (2, 0, False), (3, 0, False), (3, 1, False), (3, 2, False), (3, 3, False),
        (4, 0, False), (4, 1, False), (4, 2, False), (4, 3, False), (2, 0, True), (3, 3, True), (4, 3, True), (9, 0, False), (9, 0, True)]
PAPER_PARTS = int(os.environ.get("ARKCOS_AUDIT_PAPER_PARTS", "64"))   # the paper-regime launch is cut into this many parts of which the first --parts run


def workload(cfg, k):
    from paper_1211_3556_b200 import workloads as wl
    if cfg != 9:
        w = wl.config(cfg)[k]
        return w, w.table(), {}
    w = wl.paper_regime_workload()
    m_split, t_split = (w.n_table - 1) // 2, w.theta_cut / 16.0
    table = wl.residual_profile(wl.biased_nodes(w.theta_cut, w.n_table, m_split, t_split), w.sigma, w.l_band)
    return w, table, {"m_split": m_split, "theta_split": t_split}


def part(args):
    cfg, k, tensor, parts, offset, outdir = args
    os.environ["OMP_NUM_THREADS"] = "1"
    from tests.test_emu_parity import EMU_BIN, emulate
    w, table, biased = workload(cfg, k)
    env = {"EMU_ITEM_STRIDE": str(PAPER_PARTS if cfg == 9 else parts), "EMU_ITEM_OFFSET": str(offset)}
    if tensor:
        env["EMU_WIDE_TENSOR"] = "1"
    if biased:
        env["EMU_M_SPLIT"], env["EMU_THETA_SPLIT"] = str(biased["m_split"]), repr(biased["theta_split"])
    t0 = time.time()
    with tempfile.TemporaryDirectory() as d:
        got, log = emulate(EMU_BIN, pathlib.Path(d), w.map_f32(), table, w.theta_cut, env=env, only="only_wide" if tensor else None, timeout=4 * 3600)
    path = os.path.join(outdir, f"{cfg}_{k}_{int(tensor)}_{offset}.npy")
    np.save(path, got.astype(np.float32))
    items = log.strip().split("items ")[-1].split(" smem")[0]
    return cfg, k, tensor, path, items, time.time() - t0


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--jobs", type=int, default=8)
    ap.add_argument("--parts", type=int, default=8)
    ap.add_argument("--only", default="", help="comma-separated runs (default: all): a config number, with a trailing t for its tensor-core run; 9 = the paper's regime")
    a = ap.parse_args()
    from oracle import oracle
    from tests.test_emu_parity import build_emu_binary
    build_emu_binary()
    with tempfile.TemporaryDirectory() as outdir, ProcessPoolExecutor(a.jobs) as ex:
        for cfg, k, tensor in RUNS:
            if a.only and f"{cfg}{'t' if tensor else ''}" not in a.only.split(","):
                continue
            w, table, biased = workload(cfg, k)
            t0 = time.time()
            res = list(ex.map(part, [(cfg, k, tensor, a.parts, o, outdir) for o in range(a.parts)]))
            count = np.zeros((w.n_theta, w.n_phi), dtype=np.int32)
            total = np.zeros((w.n_theta, w.n_phi), dtype=np.float64)
            n_items = [0, 0]
            for _, _, _, path, items, _ in res:
                g = np.load(path); os.unlink(path)
                wr = ~np.isnan(g)
                count += wr
                total[wr] += g[wr]
                tok = items.split()
                n_items[0] += int(tok[1]); n_items[1] += int(tok[3])
            once = bool(((count == 1) | ((count == 0) if (tensor or cfg == 9) else False)).all())   # tensor runs cover the WIDE rings only
            pix = np.flatnonzero(count.reshape(-1) == 1)
            pix = pix[:: max(1, len(pix) // 60000)]
            if cfg == 9:
                pix = pix[:: 10]
            expect = oracle.convolve(w.map_f32(), table, w.theta_cut, level=1, pixels=pix, **biased)
            rms = math.sqrt((total[count == 1] ** 2).mean())
            err = total.reshape(-1)[pix] - expect
            rel, mx = math.sqrt((err ** 2).mean()) / rms, float(np.abs(err).max()) / rms
            ok = once and rel <= 1e-6 and mx <= 1e-5
            print(f"{w.name:34s} wide path {'tensor' if tensor else 'ffma  '}  work items wide {n_items[0]:5d} narrow {n_items[1]:5d} ({'all' if cfg != 9 else '%d/%d' % (a.parts, PAPER_PARTS)} of the launch"
                  f"{'; WIDE rings only' if tensor else ''})  map written {float((count == 1).mean()):.3f}  exactly once {once}  "
                  f"rel-rms {rel:.2e}  max/rms {mx:.2e}  {'PASS' if ok else 'FAIL'}  ({time.time() - t0:.0f} s)", flush=True)
