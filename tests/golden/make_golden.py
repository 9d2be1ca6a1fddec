"""Writes tests/golden/*.txt.  Calls ONLY the CPU oracle (oracle/) and the seeded input generators.

The paper prints no convolution output values, so these files hold the ORACLE's values
on seeded inputs - a regression pin of the oracle against itself over time, and sampled expected
values for the GPU parity tests.  No value here comes from the CUDA path.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle  # noqa: E402
from paper_1211_3556_b200 import workloads as wl  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))


def sample_pixels(w, n, seed):
    """Pole rings, equator, and seeded random pixels."""
    rng = np.random.default_rng(seed)
    rings = [0, 1, 2, w.n_theta // 2 - 1, w.n_theta // 2, w.n_theta - 2, w.n_theta - 1]
    pix = [r * w.n_phi + k for r in rings for k in (0, 1, w.n_phi // 2, w.n_phi - 1)]
    pix += list(rng.integers(0, w.n_pix, size=n - len(pix)))
    return np.array(sorted(set(int(p) for p in pix)), dtype=np.int64)


def write(name, w, pix, vals, note):
    path = os.path.join(HERE, name)
    with open(path, "w") as f:
        f.write(f"# {note}\n")
        f.write(f"# workload {w.name}: n_theta={w.n_theta} n_phi={w.n_phi} theta_cut={w.theta_cut!r} "
                f"n_table={w.n_table} kernel={w.kernel} sigma={w.sigma!r} map_seed={w.map_seeds[0]}\n")
        f.write("# source: oracle.convolve(level=1) on the FP32-rounded map (what the GPU receives); "
                "written by tests/golden/make_golden.py\n")
        f.write("# columns: flat_pixel_index  oracle_value(FP64, %.17g)\n")
        for p, v in zip(pix, vals):
            f.write(f"{int(p)} {float(v):.17g}\n")
    print("wrote", path, len(pix))


def main():
    w = wl.config(0)[0]
    pix = sample_pixels(w, 96, 1000)
    vals = oracle.convolve(w.map_f32(), w.table(), w.theta_cut, level=1, pixels=pix)
    write("cfg0_samples.txt", w, pix, vals, "BASELINE.json configs[0], 96 sampled output pixels")

    w = wl.config(1)[0]
    pix = sample_pixels(w, 160, 1001)
    vals = oracle.convolve(w.map_f32(), w.table(), w.theta_cut, level=1, pixels=pix)
    write("cfg1_samples.txt", w, pix, vals, "BASELINE.json configs[1], 160 sampled output pixels")


if __name__ == "__main__":
    main()
