"""Host emulation of the CUDA kernels against the FP64 oracle (no GPU needed).

tests/emu/ compiles the product's kernel source (csrc/arkcos_kernels.cuh + arkcos_schedule.cpp) for the
host - one OS thread per CUDA thread, checked shared memory, cp.async performed at its wait - and runs
generator + convolution for a whole plan.  This checks the INDEX LOGIC of the kernels (windows, lane-tile
layout, wrap-around, band marching, tap splits, weight layout) with the north_star tolerance; the compiled
SASS is checked by the `gpu` parity tests.  The emulator evaluates the same FP32 fmaf in the same order as
the kernel, so the error it shows is the kernel's accumulation error.
"""
import math
import os
import subprocess

import numpy as np
import pytest

from oracle import oracle

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
EMU_DIR = os.path.join(ROOT, "tests", "emu")
CSRC = os.path.join(ROOT, "paper_1211_3556_b200", "csrc")
EMU_BIN = os.path.join(EMU_DIR, "emu_arkcos")


def build_emu_binary():
    srcs = [os.path.join(EMU_DIR, "emu_main.cpp"), os.path.join(CSRC, "arkcos_schedule.cpp")]
    deps = srcs + [os.path.join(CSRC, "arkcos_kernels.cuh"), os.path.join(CSRC, "arkcos_tensor.cuh"), os.path.join(CSRC, "arkcos_internal.h"),
                   os.path.join(EMU_DIR, "stub", "cuda_runtime.h"), os.path.join(EMU_DIR, "emu_runtime.h")]
    if not os.path.exists(EMU_BIN) or any(os.path.getmtime(d) > os.path.getmtime(EMU_BIN) for d in deps):
        cmd = ["g++", "-std=c++20", "-O1", "-g", "-fsanitize=address", "-fno-omit-frame-pointer", "-pthread",
               "-DARKCOS_HOST_EMU", "-Wno-unknown-pragmas", "-I", os.path.join(EMU_DIR, "stub"), "-I", CSRC] + srcs + ["-o", EMU_BIN]
        res = subprocess.run(cmd, capture_output=True, text=True)
        assert res.returncode == 0, res.stderr[-3000:]
    return EMU_BIN


@pytest.fixture(scope="module")
def emu_bin():
    return build_emu_binary()


def emulate(emu, tmp_path, x32, table, theta_cut, only=None, env=None, timeout=600):
    n_theta, n_phi = x32.shape
    t, i, o = (str(tmp_path / n) for n in ("table.f64", "in.f32", "out.f32"))
    np.ascontiguousarray(table, dtype=np.float64).tofile(t)
    np.ascontiguousarray(x32, dtype=np.float32).tofile(i)
    cmd = [emu, str(n_theta), str(n_phi), repr(float(theta_cut)), str(table.size), t, i, o] + ([only] if only else [])
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, env=dict(os.environ, **(env or {})))
    assert res.returncode == 0, (res.stdout + res.stderr)[-3000:]
    return np.fromfile(o, dtype=np.float32).reshape(n_theta, n_phi).astype(np.float64), res.stdout


def gaussian_table(sigma, theta_cut, n):
    th = np.linspace(0.0, theta_cut, n)
    return np.exp(-0.5 * (th / sigma) ** 2) / (2.0 * math.pi * sigma * sigma)


# (n_theta, n_phi, sigma [deg], cut [sigma]): chosen so that theta_cut / dtheta is not an integer (DESIGN R3)
CASES = [
    (64, 128, 3.0, 3.0),      # configs[0]: wide polar rings + one narrow band per hemisphere, ragged warp tile
    (65, 128, 3.0, 3.0),      # odd n_theta: the equator ring is its own mirror
    (200, 512, 1.27, 3.0),    # R = 4, several narrow passes
    (96, 1024, 1.43, 2.5),    # R = 1, whole warp tile
    (301, 256, 0.9, 4.1),     # R = 6, odd n_theta, narrow windows up to the +-32 limit
]


def test_emulated_eager_cp_async(emu_bin, tmp_path):
    """cp.async copies performed at issue (EMU_EAGER): a copy into a row slot, weight block or stage buffer that is
    still being read would corrupt the result.  Several narrow passes and multi-stage wide rows."""
    n_theta, n_phi, sigma = 200, 512, math.radians(1.27)
    cut = 3.0 * sigma
    table = gaussian_table(sigma, cut, 1024)
    x32 = np.random.default_rng(31).standard_normal((n_theta, n_phi)).astype(np.float32)
    env = {"EMU_EAGER": "1"}
    got, log = emulate(emu_bin, tmp_path, x32, table, cut, env=env)
    expect = oracle.convolve(x32, table, cut, level=1)
    rms = math.sqrt((expect ** 2).mean())
    assert not np.isnan(got).any(), log
    assert math.sqrt(((got - expect) ** 2).mean()) / rms <= 1e-6 and float(np.abs(got - expect).max()) / rms <= 1e-5, log


@pytest.mark.parametrize("n_theta,n_phi,sigma_deg,cut_sigmas", CASES)
def test_emulated_kernels_match_oracle(emu_bin, tmp_path, n_theta, n_phi, sigma_deg, cut_sigmas):
    sigma = math.radians(sigma_deg)
    cut = cut_sigmas * sigma
    assert abs(cut / (math.pi / n_theta) - round(cut / (math.pi / n_theta))) > 1e-3
    table = gaussian_table(sigma, cut, 1024)
    x32 = np.random.default_rng(1000 + n_theta).standard_normal((n_theta, n_phi)).astype(np.float32)
    got, log = emulate(emu_bin, tmp_path, x32, table, cut)
    if (n_theta, n_phi) == (301, 256):      # this case must exercise the single-buffered weight tables of conv_narrow
        import re
        assert int(re.search(r"single-buffered narrow items (\d+)", log).group(1)) > 0, log
    assert not np.isnan(got).any(), "an output was never written or consumed unstaged shared memory\n" + log
    expect = oracle.convolve(x32, table, cut, level=1)
    rms = math.sqrt((expect ** 2).mean())
    rel = math.sqrt(((got - expect) ** 2).mean()) / rms
    mx = float(np.abs(got - expect).max()) / rms
    assert rel <= 1e-6 and mx <= 1e-5, (rel, mx, log)


def test_emulated_two_phi_tiles_and_oscillating_kernel(emu_bin, tmp_path):
    """n_phi = 2048: two warp tiles per ring (F = 2 narrow sub-tiles, wrap-around across the tile seam), with a
    sign-changing kernel so that a misplaced tap cannot hide behind a smooth weight profile."""
    n_theta, n_phi = 80, 2048
    cut = math.radians(4.3)
    th = np.linspace(0.0, cut, 2048)
    table = np.cos(7.0 * th / cut) * np.exp(-0.5 * (th / (0.4 * cut)) ** 2) * 50.0
    x32 = np.random.default_rng(7).standard_normal((n_theta, n_phi)).astype(np.float32)
    got, log = emulate(emu_bin, tmp_path, x32, table, cut)
    expect = oracle.convolve(x32, table, cut, level=1)
    rms = math.sqrt((expect ** 2).mean())
    assert not np.isnan(got).any(), log
    assert math.sqrt(((got - expect) ** 2).mean()) / rms <= 1e-6 and float(np.abs(got - expect).max()) / rms <= 1e-5, log


@pytest.mark.parametrize("n_theta,cut_deg,stride,expect_narrow", [(400, 1.3, 9, True), (64, 9.0, 7, False)])
def test_emulated_launch_shapes_of_the_timed_configs(emu_bin, tmp_path, n_theta, cut_deg, stride, expect_narrow):
    """n_phi = 8192, the ring length of configs[2] and configs[4]: WIDE items with F = 8 sub-tiles / S = 1, NARROW
    items with the widest tile.  Every `stride`-th work item is run (EMU_ITEM_STRIDE); the outputs of the
    skipped items stay NaN and only the written ones are compared.  An oscillating kernel, so a misplaced tap shows."""
    import re
    n_phi = 8192
    cut = math.radians(cut_deg)
    th = np.linspace(0.0, cut, 2048)
    table = np.cos(5.0 * th / cut) * np.exp(-0.5 * (th / (0.45 * cut)) ** 2) * 30.0
    x32 = np.random.default_rng(8192 + n_theta).standard_normal((n_theta, n_phi)).astype(np.float32)
    got, log = emulate(emu_bin, tmp_path, x32, table, cut, env={"EMU_ITEM_STRIDE": str(stride)})
    assert (int(re.search(r"items wide \d+ narrow (\d+)", log).group(1)) > 0) == expect_narrow, log
    written = ~np.isnan(got)
    rings = np.nonzero(written.any(axis=1))[0]
    assert len(rings) >= 6 and written.mean() > 0.4 / stride, log
    pix = np.flatnonzero(written.reshape(-1))
    pix = pix[:: max(1, len(pix) // 60000)]                     # bounded oracle work
    expect = oracle.convolve(x32, table, cut, level=1, pixels=pix)
    full_rms = math.sqrt((expect ** 2).mean())
    err = got.reshape(-1)[pix] - expect
    assert math.sqrt((err ** 2).mean()) / full_rms <= 1e-6 and float(np.abs(err).max()) / full_rms <= 1e-5, log


@pytest.mark.parametrize("n_theta,n_phi,cut_in_dtheta,stride,single", [(320, 640, 12.52, 2, False), (384, 768, 15.17, 3, True)])
def test_emulated_medium_ring_bands_march(emu_bin, tmp_path, n_theta, n_phi, cut_in_dtheta, stride, single):
    """R = 12 and R = 15, the ring half bands of configs[3] at 2 x FWHM and configs[4] at 40': the
    equatorial rings take the band-marching NARROW path (2R + 16 row slots, one CTA per SM), the polar-most band of
    the R = 15 case with single-buffered weight tables.  A sign-changing kernel; every `stride`-th work item."""
    import re
    cut = cut_in_dtheta * math.pi / n_theta
    th = np.linspace(0.0, cut, 2048)
    table = np.cos(3.0 * th / cut) * np.exp(-0.5 * (th / (cut / 3.0)) ** 2)
    x32 = np.random.default_rng(n_theta).standard_normal((n_theta, n_phi)).astype(np.float32)
    got, log = emulate(emu_bin, tmp_path, x32, table, cut, env={"EMU_ITEM_STRIDE": str(stride)})
    assert int(re.search(r"items wide \d+ narrow (\d+)", log).group(1)) > 0, log
    assert (int(re.search(r"single-buffered narrow items (\d+)", log).group(1)) > 0) == single, log
    written = ~np.isnan(got)
    pix = np.flatnonzero(written.reshape(-1))
    assert written.mean() > 0.2
    pix = pix[:: max(1, len(pix) // 40000)]
    expect = oracle.convolve(x32, table, cut, level=1, pixels=pix)
    rms = math.sqrt((expect ** 2).mean())
    err = got.reshape(-1)[pix] - expect
    assert math.sqrt((err ** 2).mean()) / rms <= 1e-6 and float(np.abs(err).max()) / rms <= 1e-5, log


@pytest.mark.parametrize("n_theta,n_phi,cut_deg", [
    (1, 4, 10.0), (1, 4, 180.0), (2, 8, 95.0), (3, 8, 61.0), (7, 12, 100.0), (9, 16, 50.0), (10, 20, 180.0),
    (16, 32, 7.0), (16, 32, 3.0), (33, 64, 21.0), (20, 1028, 9.5), (64, 516, 4.0), (5, 2052, 40.1), (12, 4100, 50.0)])
def test_emulated_edge_case_grids_of_the_gpu_suite(emu_bin, tmp_path, n_theta, n_phi, cut_deg):
    """The very grids, seeds and tables of tests/test_gpu_parity.py::test_small_grids_against_level0 (single ring,
    theta_cut = pi, R = 0, odd n_theta, n_phi not a multiple of the tiles), so that the cases the GPU suite will
    run have run in the emulation first."""
    rng = np.random.default_rng(n_theta * 7919 + n_phi)
    cut = math.radians(cut_deg)
    table = rng.standard_normal(37)
    x32 = rng.standard_normal((n_theta, n_phi)).astype(np.float32)
    got, log = emulate(emu_bin, tmp_path, x32, table, cut)
    assert not np.isnan(got).any(), log
    expect = oracle.convolve(x32, table, cut, level=0 if n_theta * n_phi <= 4096 else 1)
    rms = math.sqrt((expect ** 2).mean())
    assert math.sqrt(((got - expect) ** 2).mean()) / rms <= 1e-6 and float(np.abs(got - expect).max()) / rms <= 1e-5, log


@pytest.mark.parametrize("cfg,k,stride", [(1, 0, 16), (2, 0, 97), (3, 0, 59), (3, 1, 61), (3, 2, 61), (3, 3, 67), (4, 0, 89), (4, 1, 97),
                                          (4, 2, 101), (4, 3, 211)])
def test_emulated_subsets_of_the_full_size_schedules(emu_bin, tmp_path, cfg, k, stride):
    """The REAL schedules of BASELINE configs[1..4] (full-size grids, the workloads' own maps and tables): every
    `stride`-th work item of the launch bench.py times runs in the emulation - the heaviest polar WIDE item, WIDE and
    NARROW items of every band, single- and double-buffered weight tables - and its outputs are compared with the oracle."""
    from paper_1211_3556_b200 import workloads as wl
    w = wl.config(cfg)[k]
    x32, table = w.map_f32(), w.table()
    got, log = emulate(emu_bin, tmp_path, x32, table, w.theta_cut, env={"EMU_ITEM_STRIDE": str(stride)})
    written = ~np.isnan(got)
    assert written.any(), log
    pix = np.flatnonzero(written.reshape(-1))
    pix = pix[:: max(1, len(pix) // 30000)]
    expect = oracle.convolve(x32, table, w.theta_cut, level=1, pixels=pix)
    rms = math.sqrt((got[written] ** 2).mean())
    err = got.reshape(-1)[pix] - expect
    assert math.sqrt((err ** 2).mean()) / rms <= 1e-6 and float(np.abs(err).max()) / rms <= 1e-5, log


def emulate_whole_launch(emu_bin, tmp_path, w, parts):
    """Every work item of the launch in `parts` concurrent emulation processes (each takes every parts-th item);
    returns the merged map after checking that every output pixel was written by exactly one work item."""
    from concurrent.futures import ThreadPoolExecutor
    x32, table = w.map_f32(), w.table()
    dirs = [tmp_path / f"part{o}" for o in range(parts)]
    for d in dirs:
        d.mkdir()
    with ThreadPoolExecutor(parts) as ex:
        outs = list(ex.map(lambda o: emulate(emu_bin, dirs[o], x32, table, w.theta_cut,
                                             env={"EMU_ITEM_STRIDE": str(parts), "EMU_ITEM_OFFSET": str(o)})[0].astype(np.float32), range(parts)))
    count = np.zeros(x32.shape, dtype=np.int32)
    got = np.zeros(x32.shape, dtype=np.float64)
    for o in outs:
        wr = ~np.isnan(o)
        count += wr
        got[wr] += o[wr]
    assert (count == 1).all()
    return got


def test_emulated_config1_whole_map(emu_bin, tmp_path):
    """BASELINE configs[1] (1024 x 2048, FWHM 30', 8.95e8 kernel-pixel evaluations) COMPLETE: every work item of the
    launch through the emulated generator and both convolution kernels, the whole map against the oracle and the
    committed golden samples - the same assertions tests/test_gpu_parity.py::test_config1_full_map_and_golden makes on
    the device."""
    from paper_1211_3556_b200 import workloads as wl
    from tests.test_golden import load_golden
    w = wl.config(1)[0]
    got = emulate_whole_launch(emu_bin, tmp_path, w, 4)
    expect = oracle.convolve(w.map_f32(), w.table(), w.theta_cut, level=1)
    rms = math.sqrt((expect ** 2).mean())
    err = got - expect
    assert math.sqrt((err ** 2).mean()) / rms <= 1e-6 and float(np.abs(err).max()) / rms <= 1e-5
    pix, gold = load_golden("cfg1_samples.txt")
    assert float(np.abs(got.reshape(-1)[pix] - gold).max()) / rms <= 1e-5


def test_emulated_config2_planck_whole_map(emu_bin, tmp_path):
    """BASELINE configs[2], the Planck-resolution workload north_star's target is quoted on (4096 x 8192, 1.73e10
    kernel-pixel evaluations), COMPLETE: all 1610 work items of the launch bench.py times, in 8 emulation processes;
    60 000 evenly spaced pixels and the two polar rings against the oracle.  (tests/emu/deep_audit.py does the same for
    every BASELINE workload; profiles/r2_emulation_deep_audit.txt.)"""
    from paper_1211_3556_b200 import workloads as wl
    w = wl.config(2)[0]
    got = emulate_whole_launch(emu_bin, tmp_path, w, 8)
    pix = np.unique(np.concatenate([np.arange(0, w.n_pix, w.n_pix // 60000), np.arange(0, w.n_phi, 8), (w.n_theta - 1) * w.n_phi + np.arange(3, w.n_phi, 8)]))
    expect = oracle.convolve(w.map_f32(), w.table(), w.theta_cut, level=1, pixels=pix)
    rms = math.sqrt((got ** 2).mean())
    err = got.reshape(-1)[pix] - expect
    assert math.sqrt((err ** 2).mean()) / rms <= 1e-6 and float(np.abs(err).max()) / rms <= 1e-5


@pytest.mark.parametrize("mode,must_fail", [(1, True), (2, False), (3, True), (4, False), (5, True), (6, True)])
def test_emulation_hazard_checker_catches_missing_barriers(emu_bin, mode, must_fail):
    """The emulation's shared-memory hazard checker (the CPU counterpart of compute-sanitizer racecheck for cp.async
    writes and ld.shared reads): a read of another warp's cp.async data without a CTA barrier, and a cp.async into a
    word a lane of the same warp has read without a warp barrier, must be reported; with the barrier they must pass.
    Every other emulation test in this file runs with the checker on.  Modes 5 and 6: the fiber scheduler reports a
    barrier that can never complete (divergent __syncwarp / __syncthreads; a warp-collective mma executed by 31 lanes) -
    on the device these would hang the kernel."""
    res = subprocess.run([emu_bin, "selftest", str(mode)], capture_output=True, text=True, timeout=60)
    if must_fail:
        what = "shared-memory hazard" if mode <= 4 else ("DEADLOCK" if mode == 5 else "partial warp")
        assert res.returncode == 3 and what in res.stderr, (res.returncode, res.stdout, res.stderr)
    else:
        assert res.returncode == 0, res.stderr


def bank_report(path):
    """{(kernel, access kind, bytes): [instructions, wavefronts, conflict-free wavefronts, worst factor of a site]}"""
    agg = {}
    for line in open(path).read().splitlines():
        kernel, kind, nbytes, instrs, waves, ideal, worst = line.split()
        a = agg.setdefault((kernel, kind, int(nbytes)), [0, 0, 0, 0])
        a[0] += int(instrs); a[1] += int(waves); a[2] += int(ideal); a[3] = max(a[3], int(worst))
    return agg


def test_emulated_bank_conflict_accounting_on_known_patterns(emu_bin, tmp_path):
    """The emulation's shared-memory bank model (32 banks x 4 bytes; a 16-byte access is served a quarter warp at a
    time, an 8-byte access a half warp; different words of one bank serialise, equal words broadcast) on four known
    patterns, one of them the 144-byte lane stride with 8-byte loads that ncu showed as 2-way conflicts in round 1."""
    rep = str(tmp_path / "banks.txt")
    res = subprocess.run([emu_bin, "selftest", "7"], capture_output=True, text=True, timeout=60, env=dict(os.environ, EMU_BANKS=rep))
    assert res.returncode == 0, res.stderr
    rows = sorted((int(l.split()[2]), int(l.split()[4]), int(l.split()[5])) for l in open(rep).read().splitlines())
    assert rows == [(8, 4, 2), (16, 4, 4), (16, 4, 4), (16, 32, 4)], rows      # (bytes, wavefronts, conflict-free wavefronts) per site


@pytest.mark.parametrize("tensor", [False, True])
def test_emulated_shared_memory_loads_are_bank_conflict_free(emu_bin, tmp_path, tensor):
    """What ncu reports as l1tex__data_bank_conflicts_pipe_lsu_mem_shared, from the addresses the emulation sees, on
    a grid that has WIDE and NARROW items: every ld.shared of the three convolution kernels (window loads, weights,
    run descriptors, the tensor path's fragments) takes exactly its conflict-free number of wavefronts.  The cp.async
    destinations of the NARROW row staging are 2-way (lane tiles of 4 chunks + 1 pad: chunks 0 and 8 of a quarter
    warp share banks); they are 5 instructions per lane and staged row, against ~2700 issue slots of the pass."""
    rng = np.random.default_rng(5)
    cut = 1.3 * math.pi / 180.0
    table = gaussian_table(cut / 3.0, cut, 257)
    x32 = rng.standard_normal((64, 2048)).astype(np.float32)
    rep = str(tmp_path / "banks.txt")
    env = {"EMU_BANKS": rep}
    if tensor:
        env["EMU_WIDE_TENSOR"] = "1"
    emulate(emu_bin, tmp_path, x32, table, cut, env=env, only="only_wide" if tensor else None)
    agg = bank_report(rep)
    kernels = {k[0] for k in agg}
    assert kernels >= ({"k_convolve_wide_tc"} if tensor else {"k_convolve_wide", "k_convolve_narrow"}), kernels
    for (kernel, kind, nbytes), (instrs, waves, ideal, worst) in agg.items():
        if kind == "ld.shared" and kernel.startswith("k_convolve"):
            assert instrs > 0 and waves == ideal and worst == 1, (kernel, kind, nbytes, waves, ideal)
        if kind == "cp.async":
            assert waves <= 2 * ideal, (kernel, waves, ideal)
