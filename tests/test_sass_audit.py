"""Static audit of the compiled SASS of libarkcos.so (cuobjdump; no GPU needed).

The host emulation checks the kernels' SOURCE-level index logic; this file checks a few properties of what nvcc
actually emitted for sm_100a, the ones a fault on the device would come from:
  * the NARROW chain addresses shared memory with immediates only, and every immediate lies inside the lane-tile
    geometry the row slots are sized for (csrc/arkcos_internal.h: kNarrowSlotBytes);
  * no kernel spills to local memory (an LDL/STL in a hot loop would also invalidate the register-budget argument
    for two NARROW CTAs per SM);
  * the hot loops are plain FFMA, fully unrolled (1280 in the ten WIDE steps, 1024 in the 32 NARROW steps), and the
    rows are staged with cp.async (LDGSTS)."""
import os
import re
import shutil
import subprocess

import pytest

from paper_1211_3556_b200 import arkcos

pytestmark = pytest.mark.skipif(shutil.which("cuobjdump") is None, reason="cuobjdump not installed")


@pytest.fixture(scope="module")
def sass():
    arkcos.lib()
    out = subprocess.run(["cuobjdump", "-sass", arkcos.library_path()], capture_output=True, text=True, check=True).stdout
    funcs = {}
    for part in re.split(r"\n\s*Function : ", out)[1:]:
        name = part.split("\n")[0].strip()
        ins = [re.sub(r"\s*/\*[0-9a-f]{16}\*/\s*$", "", re.sub(r"^\s*/\*[0-9a-f]+\*/\s*", "", l)).strip()
               for l in part.split("\n") if re.search(r"/\*[0-9a-f]{4}\*/", l)]
        funcs[name] = ins
    return funcs


def find(funcs, key):
    names = [n for n in funcs if key in n]
    assert len(names) == 1, (key, list(funcs))
    return funcs[names[0]]


def opcode(line):
    return re.sub(r"^(@!?U?P\d+\s+)?", "", line).split()[0].rstrip(";")


def test_kernels_present_for_sm100_and_no_local_memory(sass):
    for key in ("k_generate_weights", "k_convolve_wideE", "k_convolve_wide_tc", "k_convolve_narrow", "k_rfft_rings", "k_spectral_apply", "k_spectral_weights"):
        ops = [opcode(l) for l in find(sass, key)]
        assert not any(o.startswith(("LDL", "STL")) for o in ops), f"{key} spills to local memory"
        if key.startswith("k_convolve"):       # every shared-memory access (stages, run tables, the partial sums of the
            # blocked summation) was resolved to the shared address space: no generic-address loads or stores
            assert not any(o.startswith(("LD.", "ST.")) for o in ops), f"{key} has generic-address memory accesses"


def test_hot_loops_are_unrolled_plain_ffma_with_cp_async_staging(sass):
    wide = [opcode(l) for l in find(sass, "k_convolve_wideE")]
    narrow = [opcode(l) for l in find(sass, "k_convolve_narrow")]
    assert wide.count("FFMA") == 10 * 128 and narrow.count("FFMA") == 32 * 32
    assert not any(o.startswith("FFMA2") or o.startswith("HMMA") or o.startswith("UTC") for o in wide + narrow)
    assert any(o.startswith("LDGSTS") for o in wide) and any(o.startswith("LDGSTS") for o in narrow)


def test_narrow_chain_shared_memory_immediates_stay_inside_the_row_slot(sass):
    ins = find(sass, "k_convolve_narrow")
    z_off, w_off = [], []
    for l in ins:
        m = re.search(r"LDS\.(128|64)\s+R\d+, \[R\d+(?:\+(-?0x[0-9a-f]+))?\]", l)
        if m:
            (z_off if m.group(1) == "128" else w_off).append(int(m.group(2), 16) if m.group(2) else 0)
    assert len(z_off) >= 100 and len(w_off) >= 33
    # chunk q of the tap axis (q = 0: d = -32) relative to the lane's own tile: ((q >> 2) - 2) * 80 + (q & 3) * 16
    chunk_offsets = {((q >> 2) - 2) * 80 + (q & 3) * 16 for q in range(0, 22)}
    assert all(o in chunk_offsets or o == 0 for o in z_off), sorted(set(z_off) - chunk_offsets)
    # the last lane's own tile is tile 33 of a 37-tile slot: reads may reach 3 tiles (240 bytes) + 16 bytes past its start
    assert min(z_off) >= -2 * 80 and max(z_off) <= 3 * 80 + 16 - 16
    # weights of step K at byte 8 K of the run, prefetched one step ahead: 0 .. 8 * 32
    assert all(o % 8 == 0 and 0 <= o <= 256 for o in w_off)
