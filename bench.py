#!/usr/bin/env python
"""bench.py — throughput of the Wilson-clover operator (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

A "step" is one pass of the whole hot path over one batch of synthetic input: one application
out = D in of the fused Wilson-clover kernel to a device-resident spinor
of the configured lattice (default: BASELINE.json configs[3], 64^4, m0=-0.4, csw=1.0, 1 RHS, Haar
links, S built on the device).  Inputs rotate over three fields and outputs over two, 25.8 GB are
touched per step (>> L2), so no L2 flush is needed between timed iterations.

The path does not shard (BASELINE.json: "Everything runs on one GPU"): with --gpus N > 1 every rank
runs an independent replica on its own GPU ("replicas only"), no data-path collective;
value = units of all ranks / max-over-ranks device time.

Prints ONE JSON line on rank 0.  `--impl reference` times the CPU oracle (oracle/, as it stands)
on the host cores on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Wilson-clover D applications: GFLOP/s, sites/s and HBM GB/s (% B200 peak), 64^4 FP64"
FLOP_WILSON, FLOP_CLOVER = 1320, 504          # per site (BASELINE.json north_star, R15)
BYTES_WILSON, BYTES_CLOVER = 960, 1536        # algorithmic B/site, each datum once
FALLBACK_HBM_GBS = 6650.0                     # /opt/skills/guides/B200_PROFILING.md fallback


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config number 1..5")
    ap.add_argument("--dims", type=str, default="", help="override lattice, e.g. 32,32,32,32")
    ap.add_argument("--nrhs", type=int, default=0, help="override the number of right-hand sides")
    ap.add_argument("--kernel", type=str, default="", help="kernel geometry name (default automatic)")
    ap.add_argument("--variant", type=int, default=0, help="0 fused, 1 unfused")
    ap.add_argument("--tchunk", type=int, default=0)
    ap.add_argument("--zgroup", type=int, default=0)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    return ap.parse_args()


def workload(args):
    import wdinputs

    cfg = dict(wdinputs.CONFIGS[args.config])
    if args.dims:
        cfg["dims"] = tuple(int(v) for v in args.dims.split(","))
    if args.nrhs:
        cfg["nrhs"] = args.nrhs
    return cfg


def peak_hbm():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(name):
    """dram bytes per launch of the dominant kernel from the committed ncu capture, or None."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)).get(name)
        except Exception:
            return None
    return None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        self.ok = False
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            pass

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.01)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def cpu_baseline_sample(cfg, max_seconds=25.0):
    """The oracle, as it stands, on the host cores, on a bounded sample of the workload: the same
    recipe on a lattice of at most 32^3 x 64 sites (a 1/8 .. 1/16 sub-volume of the 64^4 job), S
    prebuilt by the oracle (untimed), whole-lattice applies timed for <= ~25 s."""
    import oracle
    import wdinputs

    dims = tuple(min(n, 32) for n in cfg["dims"])
    V = wdinputs.volume(dims)
    U = wdinputs.config_gauge(cfg, dims)
    psi = wdinputs.spinor(dims, cfg["spinor_seed"])
    C = oracle.build_clover(dims, cfg["m0"], cfg["csw"], U) if cfg["csw"] else None
    oracle.apply(dims, cfg["m0"], U, C, psi)  # warm
    n, t0 = 0, time.perf_counter()
    while True:
        oracle.apply(dims, cfg["m0"], U, C, psi)
        n += 1
        el = time.perf_counter() - t0
        if el > 10.0 or n >= 20 or el > max_seconds:
            break
    flop = FLOP_WILSON + (FLOP_CLOVER if cfg["csw"] else 0)
    sites_per_s = n * V / el
    return {
        "value": sites_per_s * flop / 1e9, "unit": "GFLOP/s", "sites_per_s": sites_per_s,
        "cores": oracle.num_threads(), "kind": "oracle",
        "sample": f"{n} whole-lattice oracle applies of a {'x'.join(map(str, dims))} lattice "
                  f"({V} sites, same recipe: m0={cfg['m0']} csw={cfg['csw']}, S prebuilt untimed), {el:.1f} s",
    }, el / n


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = workload(args)
    import oracle
    import wdinputs

    dims = tuple(min(n, 32) for n in cfg["dims"])
    V = wdinputs.volume(dims)
    U = wdinputs.config_gauge(cfg, dims)
    psi = wdinputs.spinor(dims, cfg["spinor_seed"])
    C = oracle.build_clover(dims, cfg["m0"], cfg["csw"], U) if cfg["csw"] else None
    steps = max(1, min(args.steps, 20))
    warm = max(1, min(args.warmup, 3))
    for _ in range(warm):
        oracle.apply(dims, cfg["m0"], U, C, psi)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.apply(dims, cfg["m0"], U, C, psi)
    el = time.perf_counter() - t0
    flop = FLOP_WILSON + (FLOP_CLOVER if cfg["csw"] else 0)
    val = steps * V / el * flop / 1e9
    sample = (f"each step = one whole-lattice oracle apply of a {'x'.join(map(str, dims))} lattice "
              f"({V} sites; bounded sample of {cfg['name']}), S prebuilt untimed")
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": "GFLOP/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": el / steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "sites_per_s": steps * V / el,
        "config": {"workload": cfg["name"], "lattice": list(cfg["dims"]), "sample_lattice": list(dims),
                   "m0": cfg["m0"], "csw": cfg["csw"], "nrhs": 1},
        "cpu_baseline": {"value": val, "unit": "GFLOP/s", "cores": oracle.num_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def reduce_over_ranks(total_ms, units, dist=None, device="cpu"):
    """Replicas only: every rank ran the same independent job.  Whole-job time =
    MAX over ranks of the device time, whole-job work = SUM over ranks of the units (site x RHS
    applications) each processed.  No data-path collective: these two scalars are all that is exchanged."""
    if dist is None:
        return float(total_ms), int(units)
    import torch

    t = torch.tensor([float(total_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([int(units)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.barrier()
    return float(t.item()), int(u.item())


def run_ours(args):
    import numpy as np
    import torch

    import paper_2407_00041_b200 as wd
    import wdinputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = workload(args)
    dims, nrhs = cfg["dims"], cfg["nrhs"]
    V = wdinputs.volume(dims)
    clover = cfg["csw"] != 0.0
    flop = FLOP_WILSON + (FLOP_CLOVER if clover else 0)
    gauge_b, self_b = 576, (576 if clover else 0)
    alg_bytes_site_rhs = (gauge_b + self_b) / nrhs + 384  # per site and RHS: links and S once for all RHS (a8)
    alg_bytes_step = V * (gauge_b + self_b + 384 * nrhs)  # one step = all nrhs right-hand sides

    # ---- setup (untimed): fields become device resident in device layout
    h = wd.wd_create(*dims, cfg["m0"], cfg["csw"])
    stream = torch.cuda.current_stream()
    wd.wd_set_stream(h, stream.cuda_stream)
    wd.wd_set_option(h, wd.WD_OPT_DEVICE_PACK, 1)
    wd.wd_set_option(h, wd.WD_OPT_VARIANT, args.variant)
    if args.kernel:
        wd.wd_set_option(h, wd.WD_OPT_KERNEL, wd.kernel_id(args.kernel))
    if args.tchunk:
        wd.wd_set_option(h, wd.WD_OPT_TCHUNK, args.tchunk)
    if args.zgroup:
        wd.wd_set_option(h, wd.WD_OPT_ZGROUP, args.zgroup)
    U = wdinputs.config_gauge(cfg)
    wd.wd_load_gauge(h, U)
    del U
    if clover:
        wd.wd_build_clover(h)
    n64 = wd.wd_spinor_bytes(h, nrhs) // 8
    ins = [torch.empty(n64, dtype=torch.float64, device="cuda") for _ in range(3)]
    outs = [torch.empty(n64, dtype=torch.float64, device="cuda") for _ in range(2)]
    psi_host = wdinputs.spinor(dims, cfg["spinor_seed"], nrhs=nrhs)
    wd.wd_pack_spinor(h, ins[0], psi_host, nrhs)
    # two more distinct, device-resident inputs (GMRES-like: D applied to the previous vector)
    wd.wd_apply(h, ins[1], ins[0], nrhs)
    wd.wd_apply(h, ins[2], ins[1], nrhs)
    ins[1].mul_(1.0 / 8.0)
    ins[2].mul_(1.0 / 64.0)
    torch.cuda.synchronize()
    kname = wd.wd_kernel_name(wd.wd_kernel_for(h, nrhs))

    def step(k):
        wd.wd_apply(h, outs[k % 2], ins[k % 3], nrhs)

    for k in range(args.warmup):
        step(k)
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    launches0 = wd.wd_launch_count(h)
    torch.cuda.synchronize()
    evs[0].record(stream)
    for k in range(args.steps):
        step(k)
        evs[k + 1].record(stream)
    torch.cuda.synchronize()
    launches = wd.wd_launch_count(h) - launches0
    sampler.stop_flag = True
    sampler.join()
    per_step = [evs[k].elapsed_time(evs[k + 1]) for k in range(args.steps)]
    total_ms = evs[0].elapsed_time(evs[-1])
    total_ms, units = reduce_over_ranks(total_ms, V * nrhs * args.steps, dist, "cuda")
    torch.cuda.synchronize()
    ms_per_step = total_ms / args.steps
    site_rhs_per_s = units / (total_ms * 1e-3)
    value = site_rhs_per_s * flop / 1e9

    # ---- roofline of the dominant kernel (the fused kernel is the whole step)
    peak, peak_src = peak_hbm()
    launches_per_step = launches / args.steps
    avg_launch_ms = (sum(per_step) / len(per_step)) / launches_per_step
    alg_bytes_launch = alg_bytes_step / launches_per_step  # tma_*: one launch per step, all RHS
    achieved = alg_bytes_launch / (avg_launch_ms * 1e-3) / 1e9
    roofline = {
        "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "traffic": (ncu_traffic(kname + ("/clover" if clover else "/wilson"))
                    if tuple(dims) == (64, 64, 64, 64) and nrhs == 1 else None),  # captured for that workload only
        "peak_source": peak_src,
        "kernel": kname + ("/fused" if args.variant == 0 else "/unfused"),
        "algorithmic_bytes_per_launch": alg_bytes_launch, "avg_launch_ms": avg_launch_ms,
        "best_launch_ms": min(per_step) / launches_per_step,
        "frac_of_8000_spec": achieved / 8000.0,
    }

    # second roof: FP64 FMA peak measured on this GPU with a register-only microbenchmark
    fp64_peak, _ = wd.wd_measure_fp64(1024, 8, False)
    roofline["fp64_peak_tflops_measured"] = fp64_peak
    roofline["frac_of_fp64_peak"] = (value / 1e3) / fp64_peak

    line = {
        "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "sites_per_s": site_rhs_per_s, "hbm_gbs_algorithmic": site_rhs_per_s * alg_bytes_site_rhs / 1e9,
        "config": {"workload": cfg["name"], "lattice": list(dims), "m0": cfg["m0"], "csw": cfg["csw"],
                   "nrhs": nrhs, "kernel": kname, "variant": "fused" if args.variant == 0 else "unfused",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "inputs larger than L2 (25.8 GB touched per step at 64^4); 3 inputs / 2 outputs rotate"},
        "roofline": roofline, "gpu_launches": launches, "clocks": sampler.summary(),
    }

    # ---- end to end through the C-ABI with HOST buffers (pinned), copies inside the timed region
    if not args.no_e2e and rank == 0:
        hin = torch.from_numpy(psi_host).pin_memory()
        hout = torch.empty_like(hin).pin_memory()
        del psi_host
        wd.wd_apply_host(h, hout, hin, nrhs)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(args.e2e_steps):
            wd.wd_apply_host(h, hout, hin, nrhs)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.e2e_steps
        line["e2e"] = {"value": V * nrhs * flop / (ms * 1e-3) / 1e9, "unit": "GFLOP/s",
                       "h2d_bytes_per_step": V * nrhs * 192, "d2h_bytes_per_step": V * nrhs * 192,
                       "ms_per_step": ms, "steps": args.e2e_steps,
                       "api": "wd_apply_host (pinned host buffers, canonical layout)"}
        del hin, hout
    wd.wd_destroy(h)
    del ins, outs
    torch.cuda.empty_cache()

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"], _ = cpu_baseline_sample(cfg)
    if dist:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
