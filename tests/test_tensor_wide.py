"""N1(a) - the WIDE work items on the tensor cores (csrc/arkcos_tensor.cuh, flag ARKCOS_PLAN_WIDE_TENSOR):
a banded-Toeplitz GEMM per stage with warp-level mma.m16n8k8 TF32 instructions and a 3-term hi/lo split.

CPU (`-m "not gpu"`): the kernel source in the host emulation (fragment-exact emulation of the mma instruction,
truncating accumulation) against the oracle at the north_star tolerance; the fragment layout the emulation uses
against the one CuTe documents; the compiled SASS (HMMA.1688.F32.TF32, no spills).
GPU (`-m gpu`): against the oracle and against the default FFMA path."""
import math
import os
import re
import shutil
import subprocess

import numpy as np
import pytest

from oracle import oracle
from paper_1211_3556_b200 import workloads as wl
from tests.test_emu_parity import emu_bin, emulate, gaussian_table  # noqa: F401

DEG = math.pi / 180.0


def check(got, x32, table, cut, max_pix=30000):
    written = ~np.isnan(got)
    assert written.any()
    pix = np.flatnonzero(written.reshape(-1))
    pix = pix[:: max(1, len(pix) // max_pix)]
    expect = oracle.convolve(x32, table, cut, level=1, pixels=pix)
    rms = math.sqrt((got[written] ** 2).mean())
    err = got.reshape(-1)[pix] - expect
    rel, mx = math.sqrt((err ** 2).mean()) / rms, float(np.abs(err).max()) / rms
    assert rel <= 1e-6 and mx <= 1e-5, (rel, mx)
    return written


@pytest.mark.parametrize("n_theta,n_phi,cut_deg,kernel", [
    (16, 64, 20.0, "gauss"),        # F = 1, eight tap splits (S = 8): the fragment-space reduction
    (24, 256, 9.0, "osc"),
    (9, 1500, 31.0, "osc"),         # ragged tiles (1500 = 1024 + 476), odd n_theta, several stages per row
    (4, 4096, 50.0, "osc"),         # whole-ring windows (4096 taps = 8 stages of 512), F = 4
    (5, 36, 179.0, "osc"),          # the input window wraps around the ring many times
])
def test_emulated_tensor_wide_kernel_matches_oracle(emu_bin, tmp_path, n_theta, n_phi, cut_deg, kernel):  # noqa: F811
    rng = np.random.default_rng(n_theta * 131 + n_phi)
    cut = cut_deg * DEG
    th = np.linspace(0.0, cut, 257)
    table = gaussian_table(cut / 3.0, cut, 257) if kernel == "gauss" else np.cos(7.0 * th / cut) * np.exp(-th / cut)
    x32 = rng.standard_normal((n_theta, n_phi)).astype(np.float32)
    got, log = emulate(emu_bin, tmp_path, x32, table, cut, only="only_wide", env={"EMU_WIDE_TENSOR": "1"})
    written = check(got, x32, table, cut)
    ref, _ = emulate(emu_bin, tmp_path, x32, table, cut, only="only_wide")
    assert (written == ~np.isnan(ref)).all()                     # same work items write the same outputs
    assert np.abs(got[written] - ref[written]).max() <= 3e-6 * math.sqrt((ref[written] ** 2).mean())


def test_emulated_tensor_wide_kernel_on_a_subset_of_the_planck_schedule(emu_bin, tmp_path):  # noqa: F811
    """configs[2] (4096 x 8192, R = 5): every 151st WIDE item of the launch bench.py times, incl. the heaviest polar one."""
    w = wl.config(2)[0]
    x32, table = w.map_f32(), w.table()
    got, log = emulate(emu_bin, tmp_path, x32, table, w.theta_cut, only="only_wide", env={"EMU_WIDE_TENSOR": "1", "EMU_ITEM_STRIDE": "151"})
    check(got, x32, table, w.theta_cut)


def test_emulated_mma_fragment_layout_matches_cute():
    """The emulation's (and the kernel's) reading of the m16n8k8 TF32 fragment layout, against the thread-value layouts
    CuTe publishes for SM80_16x8x8_F32TF32TF32F32_TN (vendored CUTLASS headers; skipped if they are not installed)."""
    import glob
    import sysconfig
    site = sysconfig.get_paths()["purelib"]
    hits = glob.glob(os.path.join(site, "*", "**", "cute", "atom", "mma_traits_sm80.hpp"), recursive=True)
    if not hits:
        pytest.skip("no CUTLASS headers in site-packages")
    text = open(hits[0]).read()
    blk = text[text.index("MMA_Traits<SM80_16x8x8_F32TF32TF32F32_TN>"):]
    blk = blk[:blk.index("};")]
    row = re.search(r"using SM80_16x8_Row\s*=\s*Layout<(.*?)>;", text, re.S).group(1)

    def strides(expr):
        return [int(x) for x in re.findall(r"_(\d+)", expr[expr.index("Stride"):])]
    sa = strides(re.search(r"using ALayout\s*=\s*Layout<(.*?)>;", blk, re.S).group(1))   # ((4,8),(2,2)) : ((16,1),(8,64)) -> m + 16 k
    sb = strides(re.search(r"using BLayout\s*=\s*Layout<(.*?)>;", blk, re.S).group(1))   # ((4,8),2) : ((8,1),32) -> n + 8 k
    sc = strides(row)                                                                    # ((4,8),(2,2)) : ((32,1),(16,8)) -> m + 16 n
    assert "CLayout = SM80_16x8_Row" in blk
    for lane in range(32):
        g, t = lane >> 2, lane & 3
        for r in range(4):
            off = sa[0] * t + sa[1] * g + sa[2] * (r & 1) + sa[3] * (r >> 1)
            assert (off % 16, off // 16) == (g + 8 * (r & 1), t + 4 * (r >> 1))          # a_r = A[g + 8 (r & 1)][t + 4 (r >> 1)]
            off = sc[0] * t + sc[1] * g + sc[2] * (r & 1) + sc[3] * (r >> 1)
            assert (off % 16, off // 16) == (g + 8 * (r >> 1), 2 * t + (r & 1))          # c_r = C[g + 8 (r >> 1)][2 t + (r & 1)]
        for r in range(2):
            off = sb[0] * t + sb[1] * g + sb[2] * r
            assert (off % 8, off // 8) == (g, t + 4 * r)                                 # b_r = B[t + 4 r][g]


@pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not installed")
def test_sass_of_the_tensor_kernel():
    from paper_1211_3556_b200 import arkcos
    arkcos.lib()
    out = subprocess.run(["cuobjdump", "-sass", arkcos.library_path()], capture_output=True, text=True, check=True).stdout
    part = [p for p in re.split(r"\n\s*Function : ", out)[1:] if "k_convolve_wide_tc" in p.split("\n")[0]]
    assert len(part) == 1
    ops = re.findall(r"/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)", part[0])
    assert ops.count("HMMA.1688.F32.TF32") == 48                  # 8 n-tiles x 2 k blocks x 3 split terms per 16 taps
    assert not any(o.startswith(("LDL", "STL")) for o in ops)
    assert sum(o == "LDS.128" for o in ops) >= 8 and any(o.startswith("LDGSTS") for o in ops)
    assert not any(o.startswith("LD.") for o in ops)              # no generic-address loads: every operand load is an LDS


# ------------------------------------------------------------------------------------------- GPU
def _gpu_convolve(x32, table, cut, flags):
    import torch
    from paper_1211_3556_b200 import arkcos
    with arkcos.Plan(x32.shape[0], x32.shape[1], table, cut, flags=flags) as plan:
        d_in = torch.from_numpy(x32).cuda()
        d_out = torch.full_like(d_in, float("nan"))
        plan.convolve(d_in, d_out, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        return d_out.cpu().numpy(), plan.info().first_narrow_ring


@pytest.mark.gpu
@pytest.mark.parametrize("cfg", [0, 1])
def test_gpu_tensor_wide_path_full_maps(cfg):
    from paper_1211_3556_b200 import arkcos
    w = wl.config(cfg)[0]
    x32, table = w.map_f32(), w.table()
    got, _ = _gpu_convolve(x32, table, w.theta_cut, arkcos.PLAN_WIDE_TENSOR)
    ref, _ = _gpu_convolve(x32, table, w.theta_cut, 0)
    expect = oracle.convolve(x32, table, w.theta_cut, level=1)
    rms = math.sqrt((expect ** 2).mean())
    err = got.astype(np.float64) - expect
    assert np.isfinite(got).all()
    assert math.sqrt((err ** 2).mean()) / rms <= 1e-6 and np.abs(err).max() / rms <= 1e-5
    assert (got != ref).any() and np.abs(got.astype(np.float64) - ref).max() <= 3e-6 * rms


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,k", [(2, 0), (3, 3), (4, 3)])
def test_gpu_tensor_wide_path_full_size_sampled(cfg, k):
    """Full-size workloads (the Planck grid; the widest cuts of configs[3] and configs[4]) on the WIDE rings: whole
    polar rings and sampled pixels against the oracle."""
    from paper_1211_3556_b200 import arkcos
    w = wl.config(cfg)[k]
    x32, table = w.map_f32(), w.table()
    got, fn = _gpu_convolve(x32, table, w.theta_cut, arkcos.PLAN_WIDE_TENSOR)
    assert np.isfinite(got).all() and fn > 0
    rng = np.random.default_rng(7000 + 10 * cfg + k)
    nt, nph = w.n_theta, w.n_phi
    ks = sorted({0, 1, 15, 16, 17, 127, 128, 129, 1023, 1024, 1025, nph // 2, nph - 129, nph - 1} | {int(x) for x in rng.integers(0, nph, 10)})
    rings = sorted({1, 2, 5, fn - 1, nt - fn, nt - 2} | {int(x) for x in rng.integers(0, fn, 12)} | {nt - 1 - int(x) for x in rng.integers(0, fn, 6)})
    pix = [0 * nph + k_ for k_ in range(0, nph, 16)] + [(nt - 1) * nph + k_ for k_ in range(5, nph, 64)]     # the polar rings, densely
    pix += [i * nph + k_ for i in rings for k_ in ks]
    pix = np.array(sorted(set(pix)), dtype=np.int64)
    expect = oracle.convolve(x32, table, w.theta_cut, level=1, pixels=pix)
    scale = math.sqrt((got.astype(np.float64) ** 2).mean())
    err = got.reshape(-1)[pix].astype(np.float64) - expect
    assert math.sqrt((err ** 2).mean()) / scale <= 1e-6 and np.abs(err).max() / scale <= 1e-5, (math.sqrt((err ** 2).mean()) / scale, np.abs(err).max() / scale)
