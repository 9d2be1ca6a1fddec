"""The WHOLE C-ABI library on the host: csrc/arkcos_api.cu (plan creation, validation, uploads, launch configuration,
the host pipeline, the spectral plan) compiled against an emulated CUDA runtime (tests/emu/emu_runtime.h,
tests/emu/emu_api.cpp -> tests/emu/libarkcos_emu.so) and driven through the product's own ctypes binding.

The kernel-level emulation (tests/test_emu_parity.py) hands hand-built parameter blocks to the kernels; this file runs
the API-level scenarios of the GPU suite (tests/test_gpu_parity.py, tests/test_spectral.py, tests/test_biased_table.py)
end to end on small grids, so that the calls the GPU suite will make have been made before: pointer offsets into the
work list, shared-memory sizes against the kernels' granted maximum (a launch asking for more fails as on the device),
launch counts, the three-band host pipeline, caller-owned spectral workspace, error statuses.  "Device" memory is
host memory with red zones; every cp.async source must lie inside an emulated cudaMalloc block.  Each scenario runs in
a subprocess (tests/emu/run_emu_api.py): a kernel-level failure ends that process with a message."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
RUNNER = os.path.join(ROOT, "tests", "emu", "run_emu_api.py")

SCENARIOS = ["config0", "delta_and_weights", "entry_points_bit_identical", "bad_pointers", "small_grids", "interleaved_plans",
             "spectral", "biased_table", "class_only_flags", "wide_tensor"]


@pytest.mark.parametrize("scenario", SCENARIOS)
def test_api_scenario_on_the_emulated_library(scenario):
    res = subprocess.run([sys.executable, RUNNER, scenario], capture_output=True, text=True, timeout=1800, cwd=ROOT)
    assert res.returncode == 0 and res.stdout.strip().startswith(f"ok {scenario}"), (res.stdout[-2000:], res.stderr[-4000:])
