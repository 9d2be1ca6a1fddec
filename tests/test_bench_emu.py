"""bench.py's own code on the host-emulated library (tests/emu/run_bench_emu.py): the JSON line of the measurement
contract - metric / value / unit, roofline {bound, achieved, peak, unit, frac, traffic}, cpu_baseline {value, unit,
cores, kind, sample}, e2e {value, unit, h2d_bytes_per_step, d2h_bytes_per_step}, clocks, gpu_launches - is produced
by the code path the GPU box will run, on configs[0].  The values are those of an emulation and are not checked."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
RUNNER = os.path.join(ROOT, "tests", "emu", "run_bench_emu.py")
CFG0 = "cfg0_64x128_gauss3deg"


def run(*args):
    res = subprocess.run([sys.executable, RUNNER, "--workload", CFG0] + list(args), capture_output=True, text=True, timeout=1800, cwd=ROOT)
    assert res.returncode == 0, (res.stdout[-2000:], res.stderr[-4000:])
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout[-2000:]
    return json.loads(lines[0])


def test_bench_line_carries_the_contract_keys():
    line = run("--steps", "2", "--cpu-pixels", "2000")
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "clocks", "gpu_launches"):
        assert key in line, key
    assert line["n_gpus"] == 1 and line["steps"] == 2 and line["warmup"] >= 3 and line["dtype"] == "f32" and line["vs_baseline"] is None
    assert line["config"]["workload"] == CFG0 and "model" not in line["config"]
    roof = line["roofline"]
    assert roof["bound"] == "alu" and roof["unit"] == "TFLOP/s" and abs(roof["frac"] - roof["achieved"] / roof["peak"]) < 1e-12
    assert "traffic" in roof and abs(roof["peak"] - 148 * 128 * 2 * 1965e6 / 1e12) < 0.5      # the SM count comes from the (emulated) device
    assert roof["flops_per_launch"] == 2.0 * line["pair_evals_per_map"]
    cpu = line["cpu_baseline"]
    assert cpu["kind"] == "oracle" and cpu["cores"] >= 1 and cpu["value"] > 0 and "sample" in cpu
    e2e = line["e2e"]
    assert e2e["h2d_bytes_per_step"] == 4 * 64 * 128 == e2e["d2h_bytes_per_step"] and e2e["value"] > 0 and e2e["api"] == "arkcos_convolve_host"
    assert line["gpu_launches"] == 2 * 3            # S2 + the WIDE and the NARROW convolution kernel per step


@pytest.mark.parametrize("args,expect", [
    (("--only", "wide", "--wide-tensor", "--steps", "1"), {"report": "class_only", "only": "wide", "wide_path": "tensor (k_convolve_wide_tc)"}),
    (("--impl", "reference", "--steps", "2", "--warmup", "1", "--ref-pixels", "2000"), {"impl": "reference", "dtype": "f64", "gpu_launches": 0}),
])
def test_other_bench_modes_run(args, expect):
    line = run(*args)
    for k, v in expect.items():
        assert line[k] == v, (k, line.get(k))
    if "--impl" in args:
        assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["value"] == line["value"]


def test_cost_curve_fits_of_the_sweep():
    """bench.py --sweep's fit of GPU time against theta_cut (no device needed): a quadratic curve is recovered by the
    quadratic form and not by the paper's linear form (Eq. 2.3), and the line carries the coefficients in
    the units arkcos_split_search takes."""
    sys.path.insert(0, ROOT)
    import bench
    cuts = [5.0, 10.0, 20.0, 40.0]
    line = bench.cost_curve_line("cfg4", [(c, 0.05 + 3e-3 * c * c) for c in cuts])
    q, l = line["fit_quadratic_ms"], line["fit_linear_ms"]
    assert abs(q["a_per_arcmin2"] - 3e-3) < 1e-12 and abs(q["c"] - 0.05) < 1e-9 and q["rms_resid"] < 1e-9 < l["rms_resid"]
    assert abs(line["split_cost_model_s"]["gpu_a2"] - 3e-6) < 1e-15 and line["theta_cut_arcmin"] == cuts
    json.dumps(line)
