"""N2, the phi-spectral ring-pair path (include/arkcos_spectral.h, csrc/arkcos_spectral.cuh) against the FP64 oracle.

CPU: the kernels' source runs in the host emulation (tests/emu/emu_spectral.cpp) - plan-time FP64 weight spectra,
half-length Stockham FFT + real split, per-mode ring-pair products, inverse - at the north_star tolerance.
GPU (`-m gpu`): the same through the C ABI, and against the direct path of the same plan."""
import math
import os
import subprocess

import numpy as np
import pytest

from oracle import oracle
from paper_1211_3556_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
EMU_DIR = os.path.join(ROOT, "tests", "emu")
CSRC = os.path.join(ROOT, "paper_1211_3556_b200", "csrc")
DEG = math.pi / 180.0


@pytest.fixture(scope="module")
def emu_spectral(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("emu") / "emu_spectral")
    cmd = ["g++", "-std=c++20", "-O1", "-g", "-fsanitize=address", "-fno-omit-frame-pointer", "-pthread", "-DARKCOS_HOST_EMU",
           "-Wno-unknown-pragmas", "-I", os.path.join(EMU_DIR, "stub"), "-I", EMU_DIR, "-I", CSRC, os.path.join(EMU_DIR, "emu_spectral.cpp"),
           os.path.join(CSRC, "arkcos_schedule.cpp"), "-o", out]
    res = subprocess.run(cmd, capture_output=True, text=True)
    assert res.returncode == 0, res.stderr[-3000:]
    return out


def emulate(emu, tmp_path, x32, table, cut):
    n_theta, n_phi = x32.shape
    t, i, o = (str(tmp_path / n) for n in ("table.f64", "in.f32", "out.f32"))
    np.ascontiguousarray(table, dtype=np.float64).tofile(t)
    np.ascontiguousarray(x32, dtype=np.float32).tofile(i)
    res = subprocess.run([emu, str(n_theta), str(n_phi), repr(float(cut)), str(table.size), t, i, o], capture_output=True, text=True, timeout=900)
    assert res.returncode == 0, (res.stdout + res.stderr)[-3000:]
    return np.fromfile(o, dtype=np.float32).reshape(n_theta, n_phi).astype(np.float64)


def errors(got, expect):
    rms = math.sqrt((expect ** 2).mean())
    return math.sqrt(((got - expect) ** 2).mean()) / rms, float(np.abs(got - expect).max()) / rms


@pytest.mark.parametrize("n_theta,n_phi,cut_deg,kernel", [
    (64, 128, 9.0, "gauss"),        # configs[0]: whole-ring windows at the poles, narrow ones at the equator
    (33, 64, 17.0, "gauss"),        # odd n_theta: the equator ring is its own mirror
    (9, 16, 50.0, "random"),        # the smallest ring length the path takes; every window is wide
    (80, 2048, 4.3, "oscillating"),
    (12, 8192, 41.3, "gauss"),      # the ring length of configs[2] / configs[4]: FP32 FFT error at n = 8192
])
def test_emulated_spectral_path_matches_oracle(emu_spectral, tmp_path, n_theta, n_phi, cut_deg, kernel):
    cut = cut_deg * DEG
    th = np.linspace(0.0, cut, 2048)
    table = {"gauss": np.exp(-0.5 * (th / (cut / 3.0)) ** 2),
             "oscillating": np.cos(7.0 * th / cut) * np.exp(-0.5 * (th / (0.4 * cut)) ** 2) * 50.0,
             "random": np.random.default_rng(3).standard_normal(37)}[kernel]
    x32 = np.random.default_rng(4000 + n_theta).standard_normal((n_theta, n_phi)).astype(np.float32)
    got = emulate(emu_spectral, tmp_path, x32, table, cut)
    assert not np.isnan(got).any()
    rel, mx = errors(got, oracle.convolve(x32, table, cut, level=1))
    assert rel <= 1e-6 and mx <= 1e-5, (rel, mx)


def test_spectral_plan_argument_rules():
    from paper_1211_3556_b200 import arkcos
    t = np.ones(8)
    for n_phi in (12, 8, 32768):               # not a power of two / below 16 / above the shared-memory limit
        with pytest.raises(arkcos.ArkcosError) as e:
            arkcos.Plan(8, n_phi, t, 0.5, flags=arkcos.PLAN_HOST_ONLY | arkcos.PLAN_SPECTRAL)
        assert e.value.status == arkcos.EUNSUPPORTED
    with arkcos.Plan(8, 16, t, 0.5, flags=arkcos.PLAN_HOST_ONLY) as p:     # plan without the flag
        with pytest.raises(arkcos.ArkcosError) as e:
            p.spectral_workspace_bytes(1)
        assert e.value.status == arkcos.EUNSUPPORTED
    with arkcos.Plan(8, 16, t, 0.5, flags=arkcos.PLAN_HOST_ONLY | arkcos.PLAN_SPECTRAL) as p:
        assert p.spectral_workspace_bytes(3) == 3 * 8 * 9 * 8


# ------------------------------------------------------------------ GPU ---------------------------
def _gpu_both(torch, arkcos, x32, table, cut, n_maps=1):
    nt, nph = x32.shape[-2:]
    with arkcos.Plan(nt, nph, table, cut, flags=arkcos.PLAN_SPECTRAL) as plan:
        d_in = torch.from_numpy(x32).cuda()
        spec = torch.full_like(d_in, float("nan")); direct = torch.full_like(d_in, float("nan"))
        work = torch.empty(plan.spectral_workspace_bytes(n_maps), dtype=torch.uint8, device="cuda")
        st = torch.cuda.current_stream().cuda_stream
        plan.convolve_spectral(d_in, spec, work, n_maps, st)
        plan.convolve_batch(d_in, direct, n_maps, st)
        torch.cuda.synchronize()
        return spec.cpu().numpy().astype(np.float64), direct.cpu().numpy().astype(np.float64)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", [0, 1])
def test_gpu_spectral_path_matches_oracle_and_direct_path(cfg):
    import torch
    from paper_1211_3556_b200 import arkcos
    assert torch.cuda.is_available()
    w = wl.config(cfg)[0]
    x32, table = w.map_f32(), w.table()
    spec, direct = _gpu_both(torch, arkcos, x32, table, w.theta_cut)
    expect = oracle.convolve(x32, table, w.theta_cut, level=1)
    rel, mx = errors(spec, expect)
    assert np.isfinite(spec).all() and rel <= 1e-6 and mx <= 1e-5, (rel, mx)
    rel, mx = errors(spec, direct)
    assert rel <= 1e-6 and mx <= 1e-5, (rel, mx)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,k", [(2, 0), (4, 3)])
def test_gpu_spectral_path_full_size_sampled(cfg, k):
    """configs[2] and configs[4]-40' at full size: whole polar rings, the equator and random pixels against the
    oracle; everything against the direct path."""
    import torch
    from paper_1211_3556_b200 import arkcos
    w = wl.config(cfg)[k]
    x32, table = w.map_f32(), w.table()
    spec, direct = _gpu_both(torch, arkcos, x32, table, w.theta_cut)
    assert np.isfinite(spec).all()
    scale = math.sqrt((direct ** 2).mean())
    d = spec - direct
    assert math.sqrt((d ** 2).mean()) / scale <= 1e-6 and np.abs(d).max() / scale <= 1e-5
    rng = np.random.default_rng(77 + cfg)
    rings = [0, 1, w.n_theta // 2, w.n_theta - 1]
    pix = np.concatenate([oracle.ring_pixels(w.n_phi, rings)[:: (1 if cfg == 2 else 4)], rng.integers(0, w.n_pix, 500)]).astype(np.int64)
    expect = oracle.convolve(x32, table, w.theta_cut, level=1, pixels=pix)
    err = spec.reshape(-1)[pix] - expect
    assert math.sqrt((err ** 2).mean()) / scale <= 1e-6 and np.abs(err).max() / scale <= 1e-5
