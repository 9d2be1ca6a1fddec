"""GPU parity of the EXPERIMENTAL paired-rows narrow path (ARKCOS_PLAN_PAIR_ROWS, kernel k_convolve_pairs).
Kept in a file that sorts last: the default path's parity tests run before it."""
import math

import numpy as np
import pytest

from oracle import oracle
from paper_1211_3556_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg", [0, 1])
def test_paired_rows_matches_oracle_and_default_path(cfg):
    import torch
    from paper_1211_3556_b200 import arkcos
    assert torch.cuda.is_available()
    w = wl.config(cfg)[0]
    x32, table = w.map_f32(), w.table()
    outs = []
    for flags in (arkcos.PLAN_PAIR_ROWS, arkcos.PLAN_DEFAULT):
        with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut, flags=flags) as plan:
            d_in = torch.from_numpy(x32).cuda()
            d_out = torch.full_like(d_in, float("nan"))
            plan.convolve(d_in, d_out, torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            outs.append(d_out.cpu().numpy().astype(np.float64))
    if cfg == 0:
        expect = oracle.convolve(x32, table, w.theta_cut, level=1)
    else:                                   # cfg1: the oracle on a sample of rings (poles, mid latitudes, equator)
        rings = [0, 1, 7, 100, 255, 400, 511, 512, 700, 1016, 1023]
        pix = oracle.ring_pixels(w.n_phi, rings)
        expect = oracle.convolve(x32, table, w.theta_cut, level=1, pixels=pix).reshape(len(rings), w.n_phi)
        outs = [o[rings] for o in outs]
    rms = math.sqrt((expect ** 2).mean())
    for got in outs:
        assert np.isfinite(got).all()
        assert math.sqrt(((got - expect) ** 2).mean()) / rms <= 1e-6 and float(np.abs(got - expect).max()) / rms <= 1e-5
