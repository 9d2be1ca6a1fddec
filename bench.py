#!/usr/bin/env python
"""bench.py - throughput of the real-space spherical convolution hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]
    torchrun --nnodes=1 --nproc-per-node N ... bench.py --gpus N --steps K --warmup W

One "step" = one pass of the whole hot path (S2 weight generator + S3 convolution, all rows of
SURVEY.md §8(a); S1 is plan-time) over one synthetic map of the workload.  Default workload:
BASELINE.json configs[2], the Planck-resolution case north_star's target is quoted on.
Prints ONE JSON line (rank 0).  `--sweep` prints the five-config report and the cost-vs-theta_cut
curve instead (one JSON line per workload, then a fit line).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1211_3556_b200 import replicas  # noqa: E402
from paper_1211_3556_b200 import workloads as wl  # noqa: E402

METRIC = "kernel-pixel evaluations/s at theta_cut (output pixels/s alongside)"
UNIT = "kernel-pixel evals/s"
DEFAULT_WORKLOAD = "cfg2_planck_4096x8192_fwhm5"
# FP32 FMA roofline of one B200: SMs x 128 FP32 lanes x 2 flop x max SM clock (B200_PROFILING.md:
# 148 SMs, clocks.max.sm 1965 MHz; 128 FP32 lanes per SM, 4 SMSPs x 32).  DESIGN.md §Roofline.
FP32_LANES_PER_SM = 128


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d.get("hbm_gbs", 6650.0)), float(d.get("sm_max_mhz", 1965.0)), "measured"
    return 6650.0, 1965.0, "fallback"


def ncu_traffic(workload: str):
    """(dram bytes per launch of k_convolve, capture id) from the ncu `--set full` capture of THIS round's kernel
    committed as profiles/dram_traffic.csv (rows: workload, kernel, bytes, capture), or (None, None).  A row is
    only ever written from a capture named beside it in profiles/; it is never typed in from an older kernel."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if not os.path.exists(path):
        return None, None
    for line in open(path):
        parts = [p.strip() for p in line.split(",")]
        if len(parts) >= 4 and parts[0] == workload and parts[1] == "k_convolve":
            try:
                return float(parts[2]), parts[3]
            except ValueError:
                return None, None
    return None, None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="arkcos_clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        try:
            sm, mx, reasons, pw = [], [], set(), []
            for line in open(self.path):
                p = [x.strip() for x in line.split(",")]
                if len(p) < 9:
                    continue
                try:
                    sm.append(float(p[1])); mx.append(float(p[2])); pw.append(float(p[3]))
                except ValueError:
                    continue
                for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[5:9]):
                    if val.lower().startswith("active"):
                        reasons.add(name)
            if sm:
                out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                       "samples": len(sm), "power_w_max": float(max(pw))}
        except Exception:
            pass
        finally:
            try:
                os.unlink(self.path)
            except Exception:
                pass
        return out


def oracle_sample(w: wl.Workload, n_pixels: int, seed: int):
    """Time the CPU oracle, as it stands, on a seeded uniform sample of output pixels of `w`."""
    from oracle import oracle
    rng = np.random.default_rng(seed)
    pix = rng.integers(0, w.n_pix, size=n_pixels).astype(np.int64)
    x = w.map_f32()
    table = w.table()
    oracle.build()
    t0 = time.perf_counter()
    _, pairs = oracle.convolve(x, table, w.theta_cut, level=1, pixels=pix, return_pairs=True)
    dt = time.perf_counter() - t0
    return pairs, dt, oracle.max_threads()


def run_reference(args, w: wl.Workload):
    """--impl reference: the oracle on the host cores, bounded sample per step (tier contract ④)."""
    rank, _, world = replicas.env_world()
    if rank != 0:
        return
    n_pix = args.ref_pixels
    for _ in range(args.warmup):
        oracle_sample(w, max(1024, n_pix // 16), 777)
    pairs_total, t_total, cores = 0, 0.0, 1
    for s in range(args.steps):
        pairs, dt, cores = oracle_sample(w, n_pix, 1000 + s)
        pairs_total += pairs; t_total += dt
    value = pairs_total / t_total
    sample = f"{n_pix} seeded uniform random output pixels of {w.name} per step, oracle level 1 (windowed brute force)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w),
        "output_pixels_per_s": n_pix * args.steps / t_total,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(w: wl.Workload):
    return {"workload": w.name, "n_theta": w.n_theta, "n_phi": w.n_phi,
            "theta_cut_arcmin": w.theta_cut / wl.ARCMIN, "kernel": w.kernel,
            "fwhm_arcmin": w.sigma / wl.FWHM_TO_SIGMA / wl.ARCMIN, "n_table": w.n_table,
            "maps_per_step": len(w.map_seeds), "parallelism": "replicas (no sharding, SURVEY 8(e))",
            "l2": "maps in+out = %.0f MB per step vs 126 MB L2: %s" % (
                8e-6 * w.n_pix * len(w.map_seeds),
                "larger than L2, no flush needed" if 8 * w.n_pix * len(w.map_seeds) > 126e6 else "input buffers rotated")}


def measure(w: wl.Workload, steps: int, warmup: int, dist, local_rank: int, want_cpu: bool, want_e2e: bool = True,
            only: str = "all", path: str = "direct", wide_tensor: bool = False, all_wide: bool = False):
    """One step = S2 + S3 over ALL maps of the workload (configs[4]: the batch of 8 through arkcos_convolve_batch).
    path = "spectral": the N2 cross-check path (arkcos_convolve_spectral) instead; its step has no S2 (the weight
    spectra are plan-time) and is timed as a whole."""
    import torch
    from paper_1211_3556_b200 import arkcos

    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    hbm_gbs, sm_max_mhz, peak_src = load_peaks()
    table = w.table()
    n_maps = len(w.map_seeds)
    x32 = np.stack([w.map_f32(m) for m in range(n_maps)]) if n_maps > 1 else w.map_f32()
    # --only wide|narrow: the library's measurement hook launches one class of work items only (the
    # output is then incomplete; used for per-class timing and ncu captures, never for the bench line)
    flags = {"all": 0, "wide": arkcos.PLAN_ONLY_WIDE, "narrow": arkcos.PLAN_ONLY_NARROW}[only]
    spectral = path == "spectral"
    if spectral:
        flags |= arkcos.PLAN_SPECTRAL
    if wide_tensor:                                     # N1(a) experiment: WIDE items through k_convolve_wide_tc
        flags |= arkcos.PLAN_WIDE_TENSOR
    if all_wide:                                        # measurement hook: no NARROW class at all
        flags |= arkcos.PLAN_ALL_WIDE
    plan = arkcos.Plan(w.n_theta, w.n_phi, table, w.theta_cut, flags=flags)
    info = plan.info()
    stream = torch.cuda.Stream(device=dev)
    sh = stream.cuda_stream
    work = torch.empty(plan.spectral_workspace_bytes(n_maps), dtype=torch.uint8, device=dev) if spectral else None

    def step(src, dst):
        if spectral:
            plan.convolve_spectral(src, dst, work, n_maps, sh)
        else:
            plan.convolve_batch(src, dst, n_maps, sh)

    # rotate input buffers when the map would otherwise sit in L2 between steps
    n_rot = 1 if 8 * w.n_pix * n_maps > 126e6 else max(2, int(math.ceil(260e6 / (4 * w.n_pix))))
    d_in = [torch.from_numpy(x32).to(dev) for _ in range(n_rot)]
    d_out = torch.empty_like(d_in[0])
    with torch.cuda.stream(stream):
        for i in range(warmup):
            step(d_in[i % n_rot], d_out)
    stream.synchronize()

    # ---- timed region: K back-to-back steps, CUDA events on the launching stream --------------------
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    replicas.barrier(dist)
    torch.cuda.synchronize()
    with torch.cuda.stream(stream):
        e0.record(stream)
        for i in range(steps):
            step(d_in[i % n_rot], d_out)
        e1.record(stream)
    stream.synchronize()
    torch.cuda.synchronize()
    replicas.barrier(dist)
    elapsed_ms = e0.elapsed_time(e1)
    # ---- per-kernel device times (CUDA events inside the library, same stream), K more steps --------
    gen_ms, conv_ms = [], []
    for i in range(steps):
        if spectral:                                    # both spectral kernels together, events on the launching stream
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(stream):
                a.record(stream); step(d_in[i % n_rot], d_out); b.record(stream)
            stream.synchronize()
            g, c = 0.0, a.elapsed_time(b)
        else:
            g, c = plan.measure_convolve(d_in[i % n_rot], d_out, sh, n_maps)
        gen_ms.append(g); conv_ms.append(c)
    clocks = sampler.stop()

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    e2e = None
    if want_e2e and not spectral:
        plan.reserve_host_io()
        h_in = torch.from_numpy(x32[0] if n_maps > 1 else x32).pin_memory()
        h_out = torch.empty_like(h_in).pin_memory()
        hi, ho = h_in.numpy(), h_out.numpy()
        for _ in range(min(warmup, 2)):
            plan.convolve_host(hi, ho, sh)
        n_e2e = max(1, min(steps, 10))
        replicas.barrier(dist)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            plan.convolve_host(hi, ho, sh)      # returns after the result is in host memory
        e2e_ms = 1e3 * (time.perf_counter() - t0) / n_e2e
        checksum = float(np.abs(ho[:: max(1, w.n_theta // 64)]).sum())
        e2e = {"ms_per_step": e2e_ms, "steps": n_e2e, "checksum": checksum}

    result = {"elapsed_ms": elapsed_ms, "gen_ms": float(np.mean(gen_ms)), "conv_ms": float(np.mean(conv_ms)),
              "conv_ms_min": float(np.min(conv_ms)), "clocks": clocks, "info": info, "e2e": e2e,
              "hbm_gbs": hbm_gbs, "sm_max_mhz": sm_max_mhz, "peak_src": peak_src, "n_maps": n_maps, "path": path,
              "device_name": torch.cuda.get_device_name(dev), "sm_count": info.sm_count}
    plan.destroy()
    return result


def build_line(w, args, res, world, total_ms, total_units, cpu):
    info = res["info"]
    n_maps = res["n_maps"]
    pair_evals = int(info.pair_evals) * n_maps          # per step (= per launch of k_convolve)
    ms_per_step = total_ms / args.steps
    value = replicas.throughput(total_units, total_ms)
    peak_tflops = res["sm_count"] * FP32_LANES_PER_SM * 2 * res["sm_max_mhz"] * 1e6 / 1e12
    achieved_tflops = 2.0 * pair_evals / (res["conv_ms"] * 1e-3) / 1e12
    hbm_achieved = 8.0 * w.n_pix * n_maps / (res["conv_ms"] * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(w.name)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic", "config": workload_config(w),
        "output_pixels_per_s": world * w.n_pix * n_maps * args.steps / (total_ms * 1e-3),
        "pair_evals_per_map": int(info.pair_evals),
        "kernel_ms": {"generate_weights": res["gen_ms"], "convolve": res["conv_ms"], "convolve_min": res["conv_ms_min"]},
        "roofline": {
            "bound": "alu", "achieved": achieved_tflops, "peak": peak_tflops, "unit": "TFLOP/s",
            "frac": achieved_tflops / peak_tflops, "traffic": traffic, "traffic_source": traffic_src,
            "kernel": "k_convolve_wide + k_convolve_narrow (the two launches of step S3, timed together)", "flops_per_launch": 2.0 * pair_evals,
            "peak_source": "%d SMs x 128 FP32 lanes x 2 flop x %.0f MHz (sm_max_mhz, %s MEASURED_PEAKS.json)" % (
                res["sm_count"], res["sm_max_mhz"], res["peak_src"]),
            "issued_lane_frac": float(info.fma_slots) * n_maps / (res["conv_ms"] * 1e-3) / (peak_tflops * 1e12 / 2.0),
            "hbm": {"achieved": hbm_achieved, "peak": res["hbm_gbs"], "unit": "GB/s", "frac": hbm_achieved / res["hbm_gbs"],
                    "algorithmic_bytes_per_launch": 8.0 * w.n_pix * n_maps},
        },
        "clocks": res["clocks"],
        "gpu_launches": args.steps * int(info.kernels_per_convolve),
        "device": res["device_name"],
    }
    if res["e2e"] is not None:
        e = res["e2e"]
        line["e2e"] = {"value": world * int(info.pair_evals) / (e["ms_per_step"] * 1e-3), "unit": UNIT, "maps_per_step": 1,
                       "h2d_bytes_per_step": 4 * w.n_pix, "d2h_bytes_per_step": 4 * w.n_pix,
                       "ms_per_step": e["ms_per_step"], "steps": e["steps"], "host_memory": "pinned",
                       "api": "arkcos_convolve_host"}
    if cpu is not None:
        line["cpu_baseline"] = cpu
    return line


def spectral_line(line, w, res):
    """The N2 path is bound by memory traffic, not by the FP32 ALUs: per map it reads the map, writes and re-reads
    the ring spectra X_j (2R+1 times, mostly from L2), reads the weight spectra once and writes the result.  The
    roofline entry is therefore recomputed against HBM with the traffic that MUST cross HBM: map in + out (8 B per
    pixel), the spectra written once and read at least once (2 x 8 B per mode), and the weight spectra (4 B per
    ring pair and mode, read once per call and shared by the maps of a batch)."""
    info = res["info"]
    n_maps = res["n_maps"]
    h1 = w.n_phi // 2 + 1
    w_rows = ((w.n_theta + 1) // 2) * (2 * int(info.ring_halfband) + 1)
    bytes_alg = n_maps * (8.0 * w.n_pix + 16.0 * w.n_theta * h1) + 4.0 * w_rows * h1
    ach = bytes_alg / (res["conv_ms"] * 1e-3) / 1e9
    line["config"]["path"] = "spectral (N2 cross-check path, include/arkcos_spectral.h)"
    line["kernel_ms"] = {"rfft_rings+spectral_apply": res["conv_ms"]}
    line["roofline"] = {"bound": "hbm", "achieved": ach, "peak": res["hbm_gbs"], "unit": "GB/s", "frac": ach / res["hbm_gbs"],
                        "traffic": None, "kernel": "k_rfft_rings + k_spectral_apply", "algorithmic_bytes_per_launch": bytes_alg,
                        "peak_source": "hbm_gbs, %s MEASURED_PEAKS.json" % res["peak_src"]}
    line["gpu_launches"] = line["steps"] * 2


def cpu_baseline(w: wl.Workload, n_pixels: int):
    pairs, dt, cores = oracle_sample(w, n_pixels, 4242)
    return {"value": pairs / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "tuned": False,
            "sample": f"{n_pixels} seeded uniform random output pixels of {w.name} ({pairs} pair evals in {dt:.1f} s), "
                      "oracle level 1, OpenMP dynamic",
            "output_pixels_per_s": n_pixels / dt}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--cpu-pixels", type=int, default=1 << 20, help="oracle sample size of the cpu_baseline leg")
    ap.add_argument("--ref-pixels", type=int, default=1 << 17, help="oracle sample per step of --impl reference")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="five-config report + cost-vs-theta_cut curve")
    ap.add_argument("--path", default="direct", choices=["direct", "spectral"],
                    help="direct = the product's hot path (S2 + S3); spectral = the N2 cross-check path (arkcos_convolve_spectral)")
    ap.add_argument("--wide-tensor", action="store_true",
                    help="N1(a) experiment: the WIDE work items on the tensor cores (mma.m16n8k8 TF32, 3-term split; "
                         "ARKCOS_PLAN_WIDE_TENSOR) instead of the default FFMA kernel; the line says so in config.wide_path")
    ap.add_argument("--all-wide", action="store_true",
                    help="measurement hook: every ring in the WIDE class (ARKCOS_PLAN_ALL_WIDE), to compare the NARROW kernel "
                         "with the WIDE kernel (FFMA, or tensor cores with --wide-tensor) on the same rings")
    ap.add_argument("--only", default="all", choices=["all", "wide", "narrow"],
                    help="measurement hook: launch only the WIDE or only the NARROW work items (partial output; "
                         "prints a per-class line, not the bench line)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = wl.by_name(args.workload)

    if args.impl == "reference":
        run_reference(args, w)
        return 0

    rank, local_rank, world = replicas.env_world()
    dist = replicas.init("nccl")
    import torch
    dev = torch.device("cuda", local_rank)

    if args.sweep:
        if rank == 0:
            sweep(args)
        return 0

    if args.only != "all":
        if rank == 0:
            res = measure(w, args.steps, args.warmup, None, local_rank, want_cpu=False, want_e2e=False, only=args.only,
                          wide_tensor=args.wide_tensor, all_wide=args.all_wide)
            info = res["info"]
            slots = int(info.fma_slots_wide) if args.only == "wide" else int(info.fma_slots) - int(info.fma_slots_wide)
            slots *= res["n_maps"]
            peak = res["sm_count"] * FP32_LANES_PER_SM * res["sm_max_mhz"] * 1e6
            print(json.dumps({"report": "class_only", "only": args.only, "workload": w.name, "items": int(info.n_items),
                              "wide_path": "tensor (k_convolve_wide_tc)" if args.wide_tensor else "ffma (k_convolve_wide)",
                              "convolve_ms": res["conv_ms"], "fma_slots": slots,
                              "issued_lane_frac": slots / (res["conv_ms"] * 1e-3) / peak, "clocks": res["clocks"]}), flush=True)
        if dist is not None:
            dist.destroy_process_group()
        return 0

    res = measure(w, args.steps, args.warmup, dist, local_rank, want_cpu=False, path=args.path, wide_tensor=args.wide_tensor,
                  all_wide=args.all_wide)
    units = float(res["info"].pair_evals) * res["n_maps"] * args.steps
    total_ms, total_units = replicas.aggregate(dist, res["elapsed_ms"], units, device=dev)
    if rank == 0:
        cpu = None if (args.no_cpu or world > 1) else cpu_baseline(w, args.cpu_pixels)
        line = build_line(w, args, res, world, total_ms, total_units, cpu)
        if args.path == "spectral":
            spectral_line(line, w, res)
        if args.all_wide:
            line["config"]["ring_classes"] = "all rings WIDE (measurement hook ARKCOS_PLAN_ALL_WIDE, not the default schedule)"
        if args.wide_tensor:
            line["config"]["wide_path"] = "tensor cores: k_convolve_wide_tc, mma.m16n8k8 TF32 x 3-term split (N1(a) experiment, not the default)"
            line["roofline"]["kernel"] = "k_convolve_wide_tc + k_convolve_narrow"
            line["roofline"]["note"] = "useful FP32-equivalent FMAs against the FP32 FFMA peak; the WIDE items run on the tensor pipe"
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def sweep(args):
    """All five configs: throughput, roofline fractions, and GPU time vs theta_cut with both fits
    (a*cut^2 + c, and the paper's linear form of Eq. 2.3)."""
    curve = {}
    for w in wl.all_workloads():
        for path in ("direct", "spectral"):
            if path == "spectral" and (w.n_phi & (w.n_phi - 1) or w.n_phi < 16):
                continue
            res = measure(w, max(3, args.steps // 2), 3, None, 0, want_cpu=False, want_e2e=False, path=path)
            a = argparse.Namespace(**vars(args)); a.steps = max(3, args.steps // 2)
            line = build_line(w, a, res, 1, res["elapsed_ms"], float(res["info"].pair_evals) * res["n_maps"] * a.steps, None)
            if path == "spectral":
                spectral_line(line, w, res)
            line["report"] = "sweep"
            print(json.dumps(line), flush=True)
            key = w.name.split("_cut")[0] + ("" if path == "direct" else " [spectral path]")
            curve.setdefault(key, []).append((w.theta_cut / wl.ARCMIN, line["ms_per_step"] / res["n_maps"]))
    for key, pts in curve.items():
        if len(pts) >= 3:
            print(json.dumps(cost_curve_line(key, pts)), flush=True)


def cost_curve_line(key, pts):
    """Least-squares fits of GPU time per map against theta_cut [arcmin]: a*cut^2 + c (a direct sum) and the paper's
    linear form a*cut + c (Eq. 2.3); the coefficients are what arkcos_split_search consumes
    (include/arkcos_split.h: gpu_a2 / gpu_a1 / gpu_c, there in seconds)."""
    t = np.array([p[0] for p in pts], dtype=np.float64); ms = np.array([p[1] for p in pts], dtype=np.float64)
    quad = np.linalg.lstsq(np.stack([t ** 2, np.ones_like(t)], 1), ms, rcond=None)[0]
    lin = np.linalg.lstsq(np.stack([t, np.ones_like(t)], 1), ms, rcond=None)[0]
    return {"report": "cost_curve", "family": key, "theta_cut_arcmin": t.tolist(), "gpu_ms_per_map": ms.tolist(),
            "fit_quadratic_ms": {"a_per_arcmin2": float(quad[0]), "c": float(quad[1]),
                                 "rms_resid": float(np.sqrt(np.mean((quad[0] * t ** 2 + quad[1] - ms) ** 2)))},
            "fit_linear_ms": {"a_per_arcmin": float(lin[0]), "c": float(lin[1]),
                              "rms_resid": float(np.sqrt(np.mean((lin[0] * t + lin[1] - ms) ** 2)))},
            "split_cost_model_s": {"gpu_a2": float(quad[0]) * 1e-3, "gpu_a1": 0.0, "gpu_c": float(max(quad[1], 0.0)) * 1e-3},
            "paper_eq_2_3": "t = 0.0232 s * theta_cut[arcmin] + 2.428 s (GTX 480, HEALPix nside 2048; context only)"}


if __name__ == "__main__":
    sys.exit(main())
