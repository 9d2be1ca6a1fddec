"""Runs ONE API-level scenario of the GPU suite against tests/emu/libarkcos_emu.so - the whole C-ABI library
(csrc/arkcos_api.cu) compiled for the host with an emulated CUDA runtime (tests/emu/emu_runtime.h).  Test
infrastructure only; executed in a subprocess by tests/test_emu_api.py (a kernel-level failure ends the process).

    python tests/emu/run_emu_api.py <scenario>

"Device" buffers are host memory from the emulated cudaMalloc (red zones, registered as legal cp.async sources),
wrapped as numpy arrays; the ctypes binding is the product's own (paper_1211_3556_b200/arkcos.py) with its library
handle pointed at the emulated library."""
import ctypes
import math
import os
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)
CSRC = os.path.join(ROOT, "paper_1211_3556_b200", "csrc")
LIB = os.path.join(HERE, "libarkcos_emu.so")
DEG = math.pi / 180.0


def build_emu_library():
    srcs = [os.path.join(HERE, "emu_api.cpp"), os.path.join(CSRC, "arkcos_schedule.cpp"), os.path.join(CSRC, "arkcos_split.cpp")]
    deps = srcs + [os.path.join(CSRC, f) for f in ("arkcos_api.cu", "arkcos_kernels.cuh", "arkcos_spectral.cuh", "arkcos_tensor.cuh", "arkcos_internal.h")] + \
        [os.path.join(HERE, "emu_runtime.h"), os.path.join(HERE, "stub", "cuda_runtime.h")]
    if os.path.exists(LIB) and all(os.path.getmtime(d) <= os.path.getmtime(LIB) for d in deps):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["g++", "-std=c++20", "-O1", "-g", "-shared", "-fPIC", "-pthread", "-DARKCOS_HOST_EMU", "-DARKCOS_BUILD", "-Wno-unknown-pragmas",
           "-I", os.path.join(HERE, "stub"), "-I", HERE, "-I", CSRC, "-x", "c++"] + srcs + ["-o", tmp]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stderr[-4000:])
        raise SystemExit(2)
    os.replace(tmp, LIB)
    return LIB


from paper_1211_3556_b200 import arkcos  # noqa: E402
from paper_1211_3556_b200 import workloads as wl  # noqa: E402
from oracle import oracle  # noqa: E402
from tests import helpers as H  # noqa: E402

_emu = ctypes.CDLL(build_emu_library())
for _name, _res, _args in arkcos.SYMBOLS:
    _fn = getattr(_emu, _name)
    _fn.restype, _fn.argtypes = _res, _args
_emu.arkcos_emu_device_alloc.restype, _emu.arkcos_emu_device_alloc.argtypes = ctypes.c_void_p, [ctypes.c_ulonglong]
_emu.arkcos_emu_device_free.argtypes = [ctypes.c_void_p]
_emu.arkcos_emu_launches.restype = ctypes.c_ulonglong
_emu.arkcos_emu_ctas.restype = ctypes.c_ulonglong
arkcos._lib = _emu                       # every Plan below talks to the emulated library
_keep = []


def dev(array_or_shape, dtype=np.float32, fill=None):
    """A "device" array: emulated cudaMalloc memory viewed as numpy (contents copied in, or NaN-filled)."""
    src = None if isinstance(array_or_shape, tuple) else np.ascontiguousarray(array_or_shape, dtype=dtype)
    shape = array_or_shape if src is None else src.shape
    n = int(np.prod(shape))
    ptr = _emu.arkcos_emu_device_alloc(max(1, n) * np.dtype(dtype).itemsize)
    buf = (ctypes.c_char * (n * np.dtype(dtype).itemsize)).from_address(ptr)
    a = np.frombuffer(buf, dtype=dtype).reshape(shape)
    _keep.append(buf)
    if src is not None:
        a[...] = src
    elif fill is not None:
        a[...] = fill
    return a


class Work:                              # the workspace argument of Plan.convolve_spectral (torch-tensor-like)
    def __init__(self, nbytes):
        self.a = dev((nbytes,), dtype=np.uint8)
    def data_ptr(self): return self.a.ctypes.data
    def numel(self): return self.a.size
    def element_size(self): return 1


def parity(got, expect, scale=None, what=""):
    got = np.asarray(got, dtype=np.float64); expect = np.asarray(expect, dtype=np.float64)
    assert np.isfinite(got).all(), f"{what}: non-finite output"
    rms = math.sqrt((expect ** 2).mean()) if scale is None else scale
    rel = math.sqrt(((got - expect) ** 2).mean()) / rms
    mx = np.abs(got - expect).max() / rms
    assert rel <= 1e-6 and mx <= 1e-5, f"{what}: rel-rms {rel:.3e} max/rms {mx:.3e}"


def convolve(x32, table, cut, flags=0, **kw):
    with arkcos.Plan(x32.shape[0], x32.shape[1], table, cut, flags=flags, **kw) as plan:
        d_in = dev(x32); d_out = dev(x32.shape, fill=np.nan)
        plan.convolve(d_in, d_out, 0)
        return d_out.copy()


# ---------------------------------------------------------------------------------------------- scenarios
def sc_config0():
    w = wl.config(0)[0]
    x32, table = w.map_f32(), w.table()
    got = convolve(x32, table, w.theta_cut)
    parity(got, oracle.convolve(x32, table, w.theta_cut, level=1), what="cfg0")
    from tests.test_golden import load_golden
    pix, gold = load_golden("cfg0_samples.txt")
    parity(got.reshape(-1)[pix], gold, scale=math.sqrt((got.astype(np.float64) ** 2).mean()), what="cfg0 golden")


def sc_delta_and_weights():
    w = wl.config(0)[0]
    table = w.table()
    x32 = np.zeros((w.n_theta, w.n_phi), dtype=np.float32); x32[5, 100] = 1.0
    got = convolve(x32, table, w.theta_cut)
    expect = oracle.convolve(x32, table, w.theta_cut)
    assert ((got == 0.0) == (expect == 0.0)).all()
    np.testing.assert_allclose(got, expect, rtol=2e-7, atol=0)
    theta, phi = H.centres(w.n_theta, w.n_phi); area = H.area_by_sine(w.n_theta, w.n_phi)
    nodes = np.linspace(0.0, w.theta_cut, w.n_table)
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut) as plan:
        for (i, j) in [(0, 0), (0, 2), (31, 34), (63, 61), (20, 23)]:
            gw = plan.pair_weights(i, j)
            dwin = plan.window(i, j); dmax = w.n_phi // 2 if dwin == w.n_phi else dwin
            assert len(gw) == dmax + 1
            u = np.array([math.sin(theta[i]), 0.0, math.cos(theta[i])]); d = np.arange(dmax + 1)
            v = np.stack([math.sin(theta[j]) * np.cos(phi[d]), math.sin(theta[j]) * np.sin(phi[d]), np.full(d.size, math.cos(theta[j]))], axis=-1)
            ex = area[j] * np.interp(H.angle_atan2(u[None, :], v), nodes, table)
            np.testing.assert_allclose(gw, ex, rtol=1.2e-7, atol=1e-12 * np.abs(ex).max())


def sc_entry_points_bit_identical():
    w = wl.config(0)[0]
    table = w.table()
    maps = np.stack([wl.white_map(w.n_theta, w.n_phi, s) for s in (40, 41, 42)])
    with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut) as plan, \
            arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut, flags=arkcos.PLAN_CACHE_WEIGHTS) as cached:
        assert plan.info().kernels_per_convolve == 3 and cached.info().kernels_per_convolve == 2
        d_in = dev(maps)
        single, again, batch, c_out = (dev(maps.shape, fill=np.nan) for _ in range(4))
        before = _emu.arkcos_emu_launches()
        for m in range(3):
            plan.convolve(d_in[m], single[m], 0); plan.convolve(d_in[m], again[m], 0); cached.convolve(d_in[m], c_out[m], 0)
        assert _emu.arkcos_emu_launches() - before == 3 * (3 + 3 + 2)
        plan.convolve_batch(d_in, batch, 3, 0)
        assert (single == again).all() and (single == batch).all() and (single == c_out).all()
        for chunks in (0, 3):                          # the host pipeline: one band, and three bands of rings
            with arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut) as hp:
                hp.reserve_host_io(chunks)
                h_out = np.full_like(maps[0], np.nan)
                hp.convolve_host(maps[0], h_out, 0)
                assert (h_out == single[0]).all(), chunks
        gen_ms, conv_ms = plan.measure_convolve(d_in[0], again[0], 0)
        assert gen_ms > 0 and conv_ms > 0 and (again[0] == single[0]).all()
        batch[...] = np.nan
        gen_ms, conv_ms = plan.measure_convolve(d_in, batch, 0, 3)           # what bench.py times for configs[4]
        assert gen_ms > 0 and conv_ms > 0 and (batch == single).all()
        st, why = plan.validate()
        assert st == arkcos.OK, why
        assert len(plan.items()) == plan.info().n_items


def sc_bad_pointers():
    w = wl.config(0)[0]
    with arkcos.Plan(w.n_theta, w.n_phi, w.table(), w.theta_cut) as plan:
        buf = dev((2 * w.n_pix + 8,), fill=0.0)
        a = buf[: w.n_pix]; b = buf[w.n_pix: 2 * w.n_pix]
        plan.convolve(a, b)
        for bad_in, bad_out in [(a, a), (a, buf[4: w.n_pix + 4]), (buf[1: w.n_pix + 1], b), (a, buf[w.n_pix + 1: 2 * w.n_pix + 1])]:
            try:
                plan.convolve(bad_in, bad_out)
            except arkcos.ArkcosError as e:
                assert e.status == arkcos.EINVAL
            else:
                raise AssertionError("bad pointers accepted")
        assert _emu.arkcos_convolve(plan._h, None, b.ctypes.data, None) == arkcos.EINVAL
        assert _emu.arkcos_convolve(None, a.ctypes.data, b.ctypes.data, None) == arkcos.EINVAL


def sc_small_grids():
    for n_theta, n_phi, cut_deg in [(1, 4, 180.0), (3, 8, 61.0), (10, 20, 180.0), (33, 64, 21.0), (20, 1028, 9.5)]:
        rng = np.random.default_rng(n_theta * 7919 + n_phi)
        cut = cut_deg * DEG; table = rng.standard_normal(37)
        x32 = rng.standard_normal((n_theta, n_phi)).astype(np.float32)
        got = convolve(x32, table, cut)
        parity(got, oracle.convolve(x32, table, cut, level=0 if n_theta * n_phi <= 4096 else 1), what=f"{n_theta}x{n_phi}")


def sc_interleaved_plans():
    rng = np.random.default_rng(77)
    big = (96, 512, 5.1 * DEG); small = (16, 32, 7.0 * DEG)
    tabs = {big: rng.standard_normal(64), small: rng.standard_normal(37)}
    xs = {g: rng.standard_normal(g[:2]).astype(np.float32) for g in (big, small)}
    expect = {g: oracle.convolve(xs[g], tabs[g], g[2], level=1) for g in (big, small)}
    plans = [(g, arkcos.Plan(g[0], g[1], tabs[g], g[2])) for g in (big, small, big, small)]
    for g, plan in plans + plans[::-1]:
        d_in = dev(xs[g]); d_out = dev(xs[g].shape, fill=np.nan)
        plan.convolve(d_in, d_out, 0)
        parity(d_out, expect[g], what=f"interleaved {g}")
    for _, plan in plans:
        plan.destroy()


def sc_spectral():
    for (nt, nph, cut_deg) in [(64, 128, 9.0), (33, 64, 17.0)]:
        rng = np.random.default_rng(nt)
        cut = cut_deg * DEG
        th = np.linspace(0.0, cut, 1024); table = np.cos(4.0 * th / cut) * np.exp(-0.5 * (th / (cut / 3.0)) ** 2)
        maps = rng.standard_normal((2, nt, nph)).astype(np.float32)
        with arkcos.Plan(nt, nph, table, cut, flags=arkcos.PLAN_SPECTRAL) as plan:
            d_in = dev(maps); spec = dev(maps.shape, fill=np.nan); direct = dev(maps.shape, fill=np.nan)
            work = Work(plan.spectral_workspace_bytes(2))
            plan.convolve_spectral(d_in, spec, work, 2, 0)
            plan.convolve_batch(d_in, direct, 2, 0)
            try:
                plan.convolve_spectral(d_in, spec, Work(plan.spectral_workspace_bytes(2) - 16), 2, 0)
            except arkcos.ArkcosError as e:
                assert e.status == arkcos.EINVAL
            else:
                raise AssertionError("short workspace accepted")
        for m in range(2):
            ex = oracle.convolve(maps[m], table, cut, level=1)
            parity(spec[m], ex, what=f"spectral {nt}x{nph} map {m}")
            parity(spec[m], direct[m].astype(np.float64), what="spectral vs direct")
    with arkcos.Plan(16, 32, np.ones(8), 0.4) as plan:       # plan without the flag
        try:
            plan.spectral_workspace_bytes(1)
        except arkcos.ArkcosError as e:
            assert e.status == arkcos.EUNSUPPORTED


def sc_biased_table():
    from tests.test_biased_table import CUT, M_SPLIT, N_PHI, N_THETA, T_SPLIT, biased_table
    table = biased_table()
    x32 = np.random.default_rng(11).standard_normal((N_THETA, N_PHI)).astype(np.float32)
    got = convolve(x32, table, CUT, m_split=M_SPLIT, theta_split=T_SPLIT)
    parity(got, oracle.convolve(x32, table, CUT, level=1, m_split=M_SPLIT, theta_split=T_SPLIT), what="biased")
    spec_in = dev(x32); spec_out = dev(x32.shape, fill=np.nan)
    if N_PHI & (N_PHI - 1) == 0:
        with arkcos.Plan(N_THETA, N_PHI, table, CUT, flags=arkcos.PLAN_SPECTRAL, m_split=M_SPLIT, theta_split=T_SPLIT) as plan:
            plan.convolve_spectral(spec_in, spec_out, Work(plan.spectral_workspace_bytes(1)), 1, 0)
        parity(spec_out, got.astype(np.float64), what="biased spectral vs direct")


def sc_class_only_flags():
    w = wl.config(0)[0]
    x32, table = w.map_f32(), w.table()
    full = convolve(x32, table, w.theta_cut)
    wide = convolve(x32, table, w.theta_cut, flags=arkcos.PLAN_ONLY_WIDE)
    narrow = convolve(x32, table, w.theta_cut, flags=arkcos.PLAN_ONLY_NARROW)
    ww, nw = ~np.isnan(wide), ~np.isnan(narrow)
    assert (ww ^ nw).all() and ww.any() and nw.any()             # the two classes partition the map
    assert (np.where(ww, wide, narrow) == full).all()


def sc_wide_tensor():
    """N1(a): ARKCOS_PLAN_WIDE_TENSOR runs the WIDE items through k_convolve_wide_tc (emulated mma.m16n8k8 TF32 with the
    3-term split); same tolerance against the oracle, NARROW rings bit-identical to the default plan, batch entry point."""
    w = wl.config(0)[0]
    x32, table = w.map_f32(), w.table()
    expect = oracle.convolve(x32, table, w.theta_cut, level=1)
    full = convolve(x32, table, w.theta_cut)
    tens = convolve(x32, table, w.theta_cut, flags=arkcos.PLAN_WIDE_TENSOR)
    parity(tens, expect, what="cfg0 wide-tensor")
    narrow_only = convolve(x32, table, w.theta_cut, flags=arkcos.PLAN_ONLY_NARROW)
    nw = ~np.isnan(narrow_only)
    assert nw.any() and (~nw).any()
    assert (tens[nw] == full[nw]).all()                           # the NARROW kernel is not affected
    assert (tens[~nw] != full[~nw]).any()                         # ... and the WIDE rings really took the other kernel
    for n_theta, n_phi, cut_deg in [(3, 8, 61.0), (20, 1028, 9.5)]:
        rng = np.random.default_rng(n_theta * 7919 + n_phi)
        cut = cut_deg * DEG; table = rng.standard_normal(37)
        x = rng.standard_normal((n_theta, n_phi)).astype(np.float32)
        got = convolve(x, table, cut, flags=arkcos.PLAN_WIDE_TENSOR)
        parity(got, oracle.convolve(x, table, cut, level=0 if n_theta * n_phi <= 4096 else 1), what=f"wide-tensor {n_theta}x{n_phi}")
    # every ring WIDE (measurement hook), FFMA and tensor
    for fl in (arkcos.PLAN_ALL_WIDE, arkcos.PLAN_ALL_WIDE | arkcos.PLAN_WIDE_TENSOR):
        with arkcos.Plan(w.n_theta, w.n_phi, w.table(), w.theta_cut, flags=fl | arkcos.PLAN_HOST_ONLY) as hp:
            assert hp.info().first_narrow_ring == (w.n_theta + 1) // 2 and hp.validate()[0] == 0
        parity(convolve(x32, w.table(), w.theta_cut, flags=fl), expect, what=f"cfg0 all-wide flags {fl}")
    maps = np.stack([wl.white_map(w.n_theta, w.n_phi, s) for s in (20, 21)])
    with arkcos.Plan(w.n_theta, w.n_phi, w.table(), w.theta_cut, flags=arkcos.PLAN_WIDE_TENSOR) as plan:
        d_in = dev(maps); d_out = dev(maps.shape, fill=np.nan)
        plan.convolve_batch(d_in, d_out, 2, 0)
        for m in range(2):
            parity(d_out[m], oracle.convolve(maps[m], w.table(), w.theta_cut, level=1), what=f"wide-tensor batch map {m}")


SCENARIOS = {k[3:]: v for k, v in globals().items() if k.startswith("sc_")}

if __name__ == "__main__":
    name = sys.argv[1]
    SCENARIOS[name]()
    assert _emu.arkcos_emu_check_red_zones() == 0, "a red zone of a device allocation was overwritten"
    print(f"ok {name}: {_emu.arkcos_emu_launches()} launches, {_emu.arkcos_emu_ctas()} CTAs emulated")
