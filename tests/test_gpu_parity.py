"""GPU parity: the CUDA path (through the C ABI) against the FP64 CPU oracle, element by element on
the same seeded inputs.  Tolerance (BASELINE.json north_star): relative rms <= 1e-6 and
max |gpu - oracle| <= 1e-5 x rms(output).  Run on the B200 box:  pytest tests -m gpu
"""
import math

import numpy as np
import pytest

from oracle import oracle
from paper_1211_3556_b200 import workloads as wl
from tests import helpers as H

pytestmark = pytest.mark.gpu

REL_RMS_TOL = 1e-6
MAX_ABS_TOL = 1e-5
DEG = math.pi / 180.0


@pytest.fixture(scope="module")
def torch():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def arkcos(torch):
    from paper_1211_3556_b200 import arkcos as a
    a.lib()
    return a


def gpu_convolve(torch, arkcos, x32, table, cut, flags=0):
    nt, nph = x32.shape
    with arkcos.Plan(nt, nph, table, cut, flags=flags) as plan:
        d_in = torch.from_numpy(x32).cuda()
        d_out = torch.full_like(d_in, float("nan"))
        plan.convolve(d_in, d_out, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return d_out.cpu().numpy()


def assert_parity(got, expect, scale_rms=None, what=""):
    got = np.asarray(got, dtype=np.float64); expect = np.asarray(expect, dtype=np.float64)
    assert np.isfinite(got).all(), f"{what}: non-finite GPU output"
    rms = math.sqrt((expect ** 2).mean()) if scale_rms is None else scale_rms
    err = got - expect
    rel = math.sqrt((err ** 2).mean()) / rms
    mx = np.abs(err).max() / rms
    assert rel <= REL_RMS_TOL and mx <= MAX_ABS_TOL, f"{what}: rel-rms {rel:.3e} max/rms {mx:.3e}"
    return rel, mx


# ------------------------------------------------------------------ configs[0]: whole map -------
def test_config0_full_map(torch, arkcos):
    w = wl.config(0)[0]
    x64 = w.map(); x32 = w.map_f32(); table = w.table()
    got = gpu_convolve(torch, arkcos, x32, table, w.theta_cut)
    expect32 = oracle.convolve(x32, table, w.theta_cut, level=1)      # same (rounded) input as the GPU
    assert_parity(got, expect32, what="cfg0 vs oracle(FP32-rounded input)")
    # against the oracle on the FP64 input the rounding of the INPUT adds <= ~6e-8
    expect64 = oracle.convolve(x64, table, w.theta_cut, level=1)
    rms = math.sqrt((expect64 ** 2).mean())
    assert math.sqrt(((got - expect64) ** 2).mean()) / rms < 2e-7 + REL_RMS_TOL


def test_config0_golden_samples(torch, arkcos):
    from tests.test_golden import load_golden
    w = wl.config(0)[0]
    pix, expect = load_golden("cfg0_samples.txt")
    got = gpu_convolve(torch, arkcos, w.map_f32(), w.table(), w.theta_cut).reshape(-1)[pix]
    full_rms = math.sqrt((oracle.convolve(w.map_f32(), w.table(), w.theta_cut) ** 2).mean())
    assert_parity(got, expect, scale_rms=full_rms, what="cfg0 golden")


# ------------------------------------------------------------------ edge cases, tiny grids ------
@pytest.mark.parametrize("n_theta,n_phi,cut_deg", [
    (1, 4, 10.0), (1, 4, 180.0), (2, 8, 95.0), (3, 8, 61.0), (7, 12, 100.0), (9, 16, 50.0), (10, 20, 180.0),
    (16, 32, 7.0), (16, 32, 3.0), (33, 64, 21.0), (20, 1028, 9.5), (64, 516, 4.0), (5, 2052, 40.1), (12, 4100, 50.0)])
def test_small_grids_against_level0(torch, arkcos, n_theta, n_phi, cut_deg):
    """Odd n_theta (self-mirrored middle ring), n_phi not a multiple of the 512 tile (ragged tail),
    theta_cut = pi (every window is a whole ring), theta_cut < dtheta (R = 0), sign-changing kernel.
    Cuts are chosen off exact ties: 40 deg on 5 x 2052 puts equator tap d = 228 at gamma == theta_cut
    exactly, where FP64 rounding (not the method) decides inclusion (R3)."""
    rng = np.random.default_rng(n_theta * 7919 + n_phi)
    cut = cut_deg * DEG
    table = rng.standard_normal(37)
    x32 = rng.standard_normal((n_theta, n_phi)).astype(np.float32)
    got = gpu_convolve(torch, arkcos, x32, table, cut)
    level = 0 if n_theta * n_phi <= 4096 else 1
    expect = oracle.convolve(x32, table, cut, level=level)
    assert_parity(got, expect, what=f"{n_theta}x{n_phi} cut {cut_deg}")


def test_delta_map_matches_oracle_exactly_outside_support(torch, arkcos):
    w = wl.config(0)[0]
    x32 = np.zeros((w.n_theta, w.n_phi), dtype=np.float32); x32[5, 100] = 1.0
    got = gpu_convolve(torch, arkcos, x32, w.table(), w.theta_cut)
    expect = oracle.convolve(x32, w.table(), w.theta_cut)
    assert ((got == 0.0) == (expect == 0.0)).all()              # same support, tap for tap
    np.testing.assert_allclose(got, expect, rtol=2e-7, atol=0)   # one product, one FP32 rounding


# ------------------------------------------------------------------ step S2: the weights --------
def test_generated_weights_match_definition(torch, arkcos):
    """w_ij[d] = A_j K(gamma_ij(d)) with gamma from atan2 and K from numpy.interp (tests/helpers.py)."""
    w = wl.config(0)[0]
    table = w.table()
    theta, phi = H.centres(w.n_theta, w.n_phi)
    area = H.area_by_sine(w.n_theta, w.n_phi)
    nodes = np.linspace(0.0, w.theta_cut, w.n_table)
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut) as plan:
        for (i, j) in [(0, 0), (0, 2), (1, 0), (31, 31), (31, 34), (40, 38), (63, 63), (63, 61), (20, 23)]:
            got = plan.pair_weights(i, j)
            dwin = plan.window(i, j)
            dmax = w.n_phi // 2 if dwin == w.n_phi else dwin
            assert len(got) == dmax + 1
            u = np.array([math.sin(theta[i]), 0.0, math.cos(theta[i])])
            d = np.arange(dmax + 1)
            v = np.stack([math.sin(theta[j]) * np.cos(phi[d]), math.sin(theta[j]) * np.sin(phi[d]),
                          np.full(d.size, math.cos(theta[j]))], axis=-1)
            g = H.angle_atan2(u[None, :], v)
            expect = area[j] * np.interp(g, nodes, table)
            np.testing.assert_allclose(got, expect, rtol=1.2e-7, atol=1e-12 * np.abs(expect).max())


# ------------------------------------------------------------------ API behaviour ----------------
def test_cached_batch_host_and_repeat_calls_are_bit_identical(torch, arkcos):
    w = wl.config(0)[0]
    table = w.table()
    maps = np.stack([wl.white_map(w.n_theta, w.n_phi, s) for s in (40, 41, 42)])
    stream = torch.cuda.current_stream().cuda_stream
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut) as plan, \
            arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut, flags=arkcos.PLAN_CACHE_WEIGHTS) as cached:
        assert plan.info().kernels_per_convolve == 3 and cached.info().kernels_per_convolve == 2   # (S2,) S3w, S3
        d_in = torch.from_numpy(maps).cuda()
        single = torch.empty_like(d_in); again = torch.empty_like(d_in); batch = torch.empty_like(d_in)
        c_out = torch.empty_like(d_in)
        for m in range(3):
            plan.convolve(d_in[m], single[m], stream)
            plan.convolve(d_in[m], again[m], stream)
            cached.convolve(d_in[m], c_out[m], stream)
        plan.convolve_batch(d_in, batch, 3, stream)
        torch.cuda.synchronize()
        assert torch.equal(single, again) and torch.equal(single, batch) and torch.equal(single, c_out)
        h_out = np.empty_like(maps[0])
        plan.convolve_host(maps[0], h_out, stream)
        assert (h_out == single[0].cpu().numpy()).all()
        gen_ms, conv_ms = plan.measure_convolve(d_in[0], again[0], stream)
        assert gen_ms > 0 and conv_ms > 0 and torch.equal(again[0], single[0])


def test_convolve_rejects_bad_pointers(torch, arkcos):
    w = wl.config(0)[0]
    with arkcos.Plan(w.n_theta, w.n_phi, w.table(), w.theta_cut) as plan:
        buf = torch.zeros(2 * w.n_pix + 8, dtype=torch.float32, device="cuda")
        a = buf[: w.n_pix]; b = buf[w.n_pix: 2 * w.n_pix]
        plan.convolve(a, b)
        for bad_in, bad_out in [(a, a), (a, buf[4: w.n_pix + 4]), (buf[1: w.n_pix + 1], b), (a, buf[w.n_pix + 1: 2 * w.n_pix + 1])]:
            with pytest.raises(arkcos.ArkcosError) as e:
                plan.convolve(bad_in, bad_out)
            assert e.value.status == arkcos.EINVAL
        lib = arkcos.lib()
        assert lib.arkcos_convolve(plan._h, None, b.data_ptr(), None) == arkcos.EINVAL
        assert lib.arkcos_convolve(None, a.data_ptr(), b.data_ptr(), None) == arkcos.EINVAL
        torch.cuda.synchronize()


# ------------------------------------------------------------------ configs[1]: whole map --------
def test_config1_full_map_and_golden(torch, arkcos):
    from tests.test_golden import load_golden
    w = wl.config(1)[0]
    x32 = w.map_f32(); table = w.table()
    got = gpu_convolve(torch, arkcos, x32, table, w.theta_cut)
    expect = oracle.convolve(x32, table, w.theta_cut, level=1)
    rel, mx = assert_parity(got, expect, what="cfg1 full map")
    pix, gold = load_golden("cfg1_samples.txt")
    assert_parity(got.reshape(-1)[pix], gold, scale_rms=math.sqrt((expect ** 2).mean()), what="cfg1 golden")
    # the 8 seeded Y_lm modes (amp 10) come through scaled by ~b_l: the output is dominated by them
    assert math.sqrt((expect ** 2).mean()) > 1.0


# ------------------------------------------------------------------ full-size configs: sampled ---
ORACLE_PAIR_BUDGET = 4.0e9      # in-support pairs the oracle evaluates per workload (~10 s on the GPU box's 16 cores)


def seam_ks(nph, rng):
    """phi positions at every seam of the kernels' tiling: the lane tile (32), the warp tile (1024) and
    the CTA tile (multiples of 1024 up to 8192), the wrap-around at 0 / n_phi, plus seeded random ones."""
    ks = {0, 1, 2, 3, 4, 15, 16, 17, 31, 32, 33, 63, 64, 511, 512, 513, nph // 2 - 1, nph // 2, nph - 33, nph - 32, nph - 17, nph - 1}
    for m in range(1, nph // 1024 + 1):
        ks |= {m * 1024 - 1, m * 1024, m * 1024 + 1}
    ks |= {int(k) for k in rng.integers(0, nph, size=12)}
    return sorted(k for k in ks if 0 <= k < nph)


def ring_taps(plan, i, nt, nph, r):
    t = 0
    for j in range(max(0, i - r), min(nt, i + r + 1)):
        d = plan.window(i, j)
        t += nph if d == nph else (2 * d + 1 if d >= 0 else 0)
    return t


def probe_pixels(w, plan, seed):
    """Pixels the oracle evaluates for a full-size workload: WHOLE rings (all k) at the seams of the schedule -
    the WIDE/NARROW class boundary, a boundary between two NARROW bands, the equator, and as many of the polar
    rings 0 .. 2R+3 as the pair budget allows - plus, on every other probed ring (all polar rings of both
    hemispheres, band edges, seeded random rings), the phi positions of `seam_ks`; plus random pixels."""
    rng = np.random.default_rng(seed)
    nt, nph = w.n_theta, w.n_phi
    r = plan.work()[2]
    fn = plan.info().first_narrow_ring
    items = plan.items()
    north_bands = sorted({(it[1], it[1] + it[2]) for it in items if it[0] == 1 and it[2] > 0})
    whole, sampled = [], set()
    if 0 < fn < (nt + 1) // 2:
        whole += [fn, fn - 1, nt - 1 - fn, nt - fn]            # class boundary, both hemispheres
    if len(north_bands) >= 2:
        b = north_bands[len(north_bands) // 2]
        whole += [b[0] - 1, b[0], nt - 1 - b[0]]                # last ring of a band / first of the next (+ south mirror)
    whole += [nt // 2 - 1, nt // 2]
    whole += list(range(0, min(nt, 2 * r + 4)))                 # polar rings, heaviest: taken while the budget lasts
    for b in north_bands[:6]:
        sampled |= {b[0], b[1] - 1, nt - 1 - b[0], nt - b[1]}
    sampled |= set(range(0, min(nt, 2 * r + 4))) | set(range(max(0, nt - 2 * r - 4), nt))
    sampled |= {nt // 4, nt // 3, fn + 1, max(0, fn - 2)} | {int(x) for x in rng.integers(0, nt, size=24)}
    ks = seam_ks(nph, rng)
    budget = ORACLE_PAIR_BUDGET - 2e8
    pix, seen_whole = [], []
    for i in whole:
        if not (0 <= i < nt) or i in seen_whole:
            continue
        cost = ring_taps(plan, i, nt, nph, r) * nph
        if cost > budget:
            continue
        budget -= cost
        seen_whole.append(i)
        pix += [i * nph + k for k in range(nph)]
    for i in sorted(sampled):
        if 0 <= i < nt and i not in seen_whole:
            pix += [i * nph + k for k in ks]
    pix += [int(p) for p in rng.integers(0, nt * nph, size=600)]
    return np.array(sorted(set(pix)), dtype=np.int64), seen_whole


FULL_SIZE = [(2, 0), (3, 0), (3, 1), (3, 2), (3, 3), (4, 0), (4, 1), (4, 2), (4, 3)]


@pytest.mark.parametrize("cfg,k", FULL_SIZE)
def test_full_size_configs_on_sampled_pixels(torch, arkcos, cfg, k):
    """Every workload of BASELINE configs[2..4] at full size, in the launch configuration bench.py times; the
    oracle evaluates whole rings at the schedule's seams and sampled pixels elsewhere, one by one."""
    w = wl.config(cfg)[k]
    x32 = w.map_f32(); table = w.table()
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut) as plan:
        d_in = torch.from_numpy(x32).cuda()
        d_out = torch.full_like(d_in, float("nan"))
        plan.convolve(d_in, d_out, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        got_full = d_out.cpu().numpy()
        pix, whole = probe_pixels(w, plan, 2000 + cfg * 10 + k)
    assert np.isfinite(got_full).all()
    assert len(whole) >= 3, whole
    expect = oracle.convolve(x32, table, w.theta_cut, level=1, pixels=pix)
    scale = math.sqrt((got_full.astype(np.float64) ** 2).mean())     # global output rms
    assert_parity(got_full.reshape(-1)[pix], expect, scale_rms=scale, what=f"{w.name} (whole rings {whole})")
    # properties that hold at any size: phi-shift equivariance of the GPU operator itself
    shift = 1000
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut, flags=arkcos.PLAN_CACHE_WEIGHTS) as plan:
        d_in = torch.from_numpy(np.roll(x32, shift, axis=1).copy()).cuda()
        d_out = torch.empty_like(d_in)
        plan.convolve(d_in, d_out)
        torch.cuda.synchronize()
        rolled = d_out.cpu().numpy()
    assert np.abs(rolled - np.roll(got_full, shift, axis=1)).max() <= 2e-6 * scale


def test_config4_batch_of_8_maps(torch, arkcos):
    """configs[4] as BASELINE states it: a batch of 8 maps (seeds 10-17) through arkcos_convolve_batch, each map
    checked against the oracle on sampled pixels, and against a single-map arkcos_convolve bit for bit."""
    w = wl.config(4)[0]
    table = w.table()
    maps = np.stack([w.map_f32(m) for m in range(8)])
    rng = np.random.default_rng(4108)
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut) as plan:
        d_in = torch.from_numpy(maps).cuda()
        d_out = torch.full_like(d_in, float("nan"))
        plan.convolve_batch(d_in, d_out, 8, torch.cuda.current_stream().cuda_stream)
        single = torch.full_like(d_in[5], float("nan"))
        plan.convolve(d_in[5], single, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        got = d_out.cpu().numpy()
        assert torch.equal(single, d_out[5])
        r = plan.work()[2]
    assert np.isfinite(got).all()
    ks = seam_ks(w.n_phi, rng)
    rings = sorted(set(range(0, 2 * r + 4)) | {w.n_theta - 1, w.n_theta // 2, 1000, 3000} | {int(x) for x in rng.integers(0, w.n_theta, 8)})
    pix = np.array(sorted({i * w.n_phi + k for i in rings for k in ks} | {int(p) for p in rng.integers(0, w.n_pix, 300)}), dtype=np.int64)
    for m in range(8):
        expect = oracle.convolve(maps[m], table, w.theta_cut, level=1, pixels=pix)
        scale = math.sqrt((got[m].astype(np.float64) ** 2).mean())
        assert_parity(got[m].reshape(-1)[pix], expect, scale_rms=scale, what=f"{w.name} map {m} (seed {w.map_seeds[m]})")


def test_interleaved_plans_of_different_shared_memory_size(torch, arkcos):
    """The dynamic shared-memory attribute belongs to the kernel, not to a plan: a small plan created
    after a large one must not break the large one's launches, and vice versa."""
    rng = np.random.default_rng(77)
    big = (256, 2048, 2.1 * DEG)       # narrow band marching, R = 2: ~190 KB of dynamic shared memory
    small = (16, 32, 7.0 * DEG)
    tabs = {big: rng.standard_normal(64), small: rng.standard_normal(37)}
    xs = {g: rng.standard_normal(g[:2]).astype(np.float32) for g in (big, small)}
    expect = {g: oracle.convolve(xs[g], tabs[g], g[2], level=1) for g in (big, small)}
    plans = []
    try:
        for g in (big, small, big, small):
            plans.append((g, arkcos.Plan(g[0], g[1], tabs[g], g[2])))
        for g, plan in plans + plans[::-1]:
            d_in = torch.from_numpy(xs[g]).cuda()
            d_out = torch.full_like(d_in, float("nan"))
            plan.convolve(d_in, d_out, torch.cuda.current_stream().cuda_stream)
            torch.cuda.synchronize()
            assert_parity(d_out.cpu().numpy(), expect[g], what=f"interleaved plan {g}")
    finally:
        for _, plan in plans:
            plan.destroy()


def test_one_plan_on_two_streams_concurrently(torch, arkcos):
    """a plan may be used concurrently from several streams.  On-the-fly plans rewrite the weight
    buffer in every call with bit-identical values; calls interleaved on two non-blocking streams must give the
    single-stream result bit for bit."""
    w = wl.config(1)[0]
    table = w.table()
    maps = [wl.white_map(w.n_theta, w.n_phi, s) for s in (50, 51)]
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut) as plan:
        d_in = [torch.from_numpy(m).cuda() for m in maps]
        ref = [torch.empty_like(d_in[0]) for _ in range(2)]
        for m in range(2):
            plan.convolve(d_in[m], ref[m], torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        outs = [[torch.full_like(d_in[0], float("nan")) for _ in range(6)] for _ in range(2)]
        torch.cuda.synchronize()        # the NaN fills run on the default stream, which the side streams do not wait for
        for rep in range(6):
            for m in range(2):
                plan.convolve(d_in[m], outs[m][rep], streams[m].cuda_stream)
        torch.cuda.synchronize()
        for m in range(2):
            for rep in range(6):
                assert torch.equal(outs[m][rep], ref[m]), (m, rep)
