#!/usr/bin/env python
"""bench.py — throughput of the Wilson-clover operator (BASELINE.json metric) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

A "step" is one pass of the whole hot path over one batch of synthetic input: one application
out = D in of the fused Wilson-clover kernel to a device-resident spinor
of the configured lattice (default: BASELINE.json configs[3], 64^4, m0=-0.4, csw=1.0, 1 RHS, Haar
links, S built on the device).  Inputs rotate over three fields and outputs over two, 25.8 GB are
touched per step (>> L2), so no L2 flush is needed between timed iterations.

BASELINE.json's headline path is single-GPU.  With --gpus N > 1 the default (--parallel dd) is STRONG scaling of the
domain-decomposed operator of SURVEY.md section 8(f)1 (the same global lattice cut over N ranks, half-spinor faces
exchanged over NCCL; run_dd below); --parallel replicas runs N independent copies with no data-path collective.
value = units of all ranks / max-over-ranks device time.

The default line also carries two sub-records measured in the same process: "sustained" (8 s of back-to-back
applications after the timed region, the figure of the LAST second with its clocks: the steady state of the power cap)
and "cfg5" (BASELINE.json configs[4], 48^3 x 96 with 12 right-hand sides, blocked layout, run after cfg 4's buffers are freed).

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
    ap.add_argument("--rhs-block", type=int, default=0, choices=[0, 1, 4],
                    help="device layout of multi-RHS spinors (WD_OPT_RHS_BLOCK): 1 plain [nrhs][12][Vs], 4 blocked [unit][12][Vs][4]; "
                         "0 (default) = blocked when the workload has at least four right-hand sides and the 2x4x8 tile divides the lattice")
    ap.add_argument("--tchunk", type=int, default=0)
    ap.add_argument("--zgroup", type=int, default=0)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-ceilings", action="store_true", help="skip the streaming / FP64 ceiling microbenchmarks")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--gauge-rows", type=int, default=3, choices=[2, 3],
                    help="2 = opt-in two-row link storage (SU(3) links only): 1344 instead of 1536 algorithmic B/site")
    ap.add_argument("--f32", action="store_true", help="also time the FP32 variant (wd_apply_f32) on the same workload")
    ap.add_argument("--parallel", default="dd", choices=["dd", "replicas"],
                    help="N > 1: dd = ONE lattice cut over the ranks, half-spinor faces exchanged with NCCL send/recv "
                         "(strong scaling, default); replicas = N independent copies (weak)")
    ap.add_argument("--gmres", type=int, default=0, metavar="M",
                    help="also run restarted GMRES(M) on the device (wd_gmres) and report its timing")
    ap.add_argument("--sustain-seconds", type=float, default=8.0,
                    help="back-to-back applications after the timed region; the last second is reported as 'sustained' (0 = skip)")
    ap.add_argument("--no-cfg5", action="store_true", help="skip the cfg 5 (12 right-hand sides) sub-record of the default line")
    ap.add_argument("--print-source-hash", type=str, default="", metavar="KERNEL",
                    help="print the hash of the sources kernel KERNEL is built from (goes into profiles/roofline_traffic.json) and exit")
    ap.add_argument("--graph", action="store_true",
                    help="also time the K steps captured as ONE CUDA graph (cfg 3: 100 back-to-back applies)")
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


KERNEL_SOURCES = {  # the files a kernel family is compiled from (paper_2407_00041_b200/csrc/)
    "tmw": ["wd_tmw.cu"], "tma": ["wd_tma.cu"], "tmb": ["wd_tmb.cu"], "tmq": ["wd_tmq.cu"], "tmqb": ["wd_tmq.cu"],
    "_tma_shared": ["wd_tma_common.cuh", "wd_tma_plan.cuh", "wd_tma.cuh", "wd_smem_ops.cuh", "wd_math.cuh", "wd_internal.h"],
    "_ldg": ["wd_kernels.cu", "wd_ldg_kernels.cuh", "wd_math.cuh", "wd_internal.h"],
}


def kernel_source_hash(kernel_name):
    """sha256 (16 hex digits) of the sources the named kernel geometry is built from: a capture in
    profiles/roofline_traffic.json is only quoted for the build it was taken from."""
    import hashlib

    fam = kernel_name.split("_")[0].split("/")[0]
    files = KERNEL_SOURCES[fam] + KERNEL_SOURCES["_tma_shared"] if fam in KERNEL_SOURCES else KERNEL_SOURCES["_ldg"]
    hsh = hashlib.sha256()
    for f in files:
        hsh.update(open(os.path.join(ROOT, "paper_2407_00041_b200", "csrc", f), "rb").read())
    return hsh.hexdigest()[:16]


def ncu_traffic(name):
    """(dram bytes per launch of the dominant kernel, where that number comes from): a CONSTANT read from the
    committed ncu capture table profiles/roofline_traffic.json (ncu cannot run inside a timed bench) — quoted only if the
    kernel's sources still hash to what the entry recorded at capture time; otherwise (None, why)."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if os.path.exists(p):
        try:
            ent = json.load(open(p)).get(name)
            if isinstance(ent, dict):
                now = kernel_source_hash(name)
                if ent.get("source_hash") != now:
                    return None, (f"profiles/roofline_traffic.json has a capture for {name}, but of another build "
                                  f"(source hash {ent.get('source_hash')}, now {now}): not quoted")
                return ent.get("bytes"), "profiles/roofline_traffic.json: " + ent.get("source", "?")
        except Exception:
            pass
    return None, None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        self.power = []
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
                    self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1e3)
                except Exception:
                    pass
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
        pw = sorted(self.power)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s), "sm_mhz_min": s[0], "power_w": pw[len(pw) // 2] if pw else None,
                "power_w_max": pw[-1] if pw else None}


def oracle_inputs(cfg):
    """Host inputs of the oracle timing legs on the bench lattice ITSELF (same dims, same links and spinor recipe).
    S: the 42-entry field is filled with seeded random Hermitian blocks instead of being built from the links —
    building it with the oracle costs minutes at 64^4 and the values do not change the cost of an apply.
    Only if the host has less free memory than the fields need (1.65 KB per site) is the lattice halved in T until
    it fits; the `sample` text names the lattice that was timed."""
    import wdinputs

    dims = list(cfg["dims"])
    try:
        import psutil

        free = psutil.virtual_memory().available
        while wdinputs.volume(dims) * 1650 > 0.8 * free and dims[0] % 2 == 0 and dims[0] > 4:
            dims[0] //= 2
    except Exception:
        pass
    dims = tuple(dims)
    U = wdinputs.config_gauge(cfg, dims)
    psi = wdinputs.spinor(dims, cfg["spinor_seed"])
    C = wdinputs.selfcoupling_random(dims, 7) if cfg["csw"] else None
    return dims, U, C, psi


def time_oracle(dims, m0, U, C, psi, reps, threads=None):
    """Seconds per whole-lattice oracle apply (best of reps), with `threads` OpenMP threads (None: all)."""
    import oracle

    nall = oracle.num_threads()
    if threads:
        oracle.set_num_threads(threads)
    try:
        best = 1e30
        for _ in range(reps):
            t0 = time.perf_counter()
            oracle.apply(dims, m0, U, C, psi)
            best = min(best, time.perf_counter() - t0)
    finally:
        oracle.set_num_threads(nall)
    return best


def cpu_baseline_sample(cfg):
    """The oracle, as it stands, on the host cores, on the bench lattice itself (one right-hand side): best of 2
    whole-lattice applies on all cores after one warm-up, and one apply on a single thread (skipped above 2^25 sites
    x RHS to keep the default run within minutes)."""
    import oracle
    import wdinputs

    dims, U, C, psi = oracle_inputs(cfg)
    V = wdinputs.volume(dims)
    flop = FLOP_WILSON + (FLOP_CLOVER if cfg["csw"] else 0)
    time_oracle(dims, cfg["m0"], U, C, psi, 1)  # warm
    t_all = time_oracle(dims, cfg["m0"], U, C, psi, 2)
    t_one = time_oracle(dims, cfg["m0"], U, C, psi, 1, threads=1) if V <= (1 << 25) else None
    lat = "x".join(map(str, dims))
    base = {
        "value": V / t_all * flop / 1e9, "unit": "GFLOP/s", "sites_per_s": V / t_all,
        "cores": oracle.num_threads(), "kind": "oracle", "seconds_per_apply": t_all,
        "sample": f"whole-lattice oracle applies of the bench lattice itself, {lat} ({V} sites, one right-hand side, "
                  f"m0={cfg['m0']} csw={cfg['csw']}; S = seeded random Hermitian blocks, untimed set-up): best of 2 on "
                  f"all cores, 1 on one thread",
    }
    if t_one:
        base["single_thread"] = {"value": V / t_one * flop / 1e9, "unit": "GFLOP/s", "sites_per_s": V / t_one,
                                 "cores": 1, "seconds_per_apply": t_one}
    return base


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = workload(args)
    import oracle
    import wdinputs

    dims, U, C, psi = oracle_inputs(cfg)
    V = wdinputs.volume(dims)
    # bounded: every step is one whole-lattice apply of ONE right-hand side of the bench lattice; at most 20 steps
    per = time_oracle(dims, cfg["m0"], U, C, psi, 1)  # warm-up 1
    steps = max(1, min(args.steps, 20, int(120.0 / max(per, 1e-3)) or 1))
    warm = max(1, min(args.warmup, 3))
    for _ in range(warm - 1):
        oracle.apply(dims, cfg["m0"], U, C, psi)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.apply(dims, cfg["m0"], U, C, psi)
    el = time.perf_counter() - t0
    flop = FLOP_WILSON + (FLOP_CLOVER if cfg["csw"] else 0)
    val = steps * V / el * flop / 1e9
    sample = (f"each step = one whole-lattice oracle apply of ONE right-hand side of the bench lattice itself "
              f"({'x'.join(map(str, dims))}, {V} sites); S = seeded random Hermitian blocks (values do not change the "
              f"cost), untimed set-up; steps capped at 20")
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


def run_dd(args, torch, dist, world, rank, local):
    """N > 1, --parallel dd: ONE lattice of the configured size cut into `world` sub-lattices (T first, then Z:
    decomp.default_grid), one per rank.  A step = one application of D to the global field: pack the half-spinor
    faces, exchange them with NCCL point-to-point on a communication stream while the fused kernel computes the
    interior, add the exterior terms.  value = global sites x steps / max-over-ranks device time (strong scaling)."""
    import numpy as np

    import paper_2407_00041_b200 as wd
    import wdinputs
    from paper_2407_00041_b200 import dd as wdd
    from paper_2407_00041_b200.decomp import Decomposition, default_grid

    cfg = workload(args)
    dims, nrhs = tuple(cfg["dims"]), cfg["nrhs"]
    V = wdinputs.volume(dims)
    clover = cfg["csw"] != 0.0
    flop = FLOP_WILSON + (FLOP_CLOVER if clover else 0)
    d = Decomposition(dims, default_grid(world, dims))
    # ---- setup (untimed).  The generators are counter-based: every rank draws only ITS sites of the global fields (and the
    # one-site halo of links its clover term needs), never the global field (9.7 GB per rank at 64^4 otherwise).
    Ul = wdinputs.config_gauge_sites(cfg, d.global_sites(rank))
    Cl = wdd.local_clover(d, rank, cfg["m0"], cfg["csw"], wdinputs.config_gauge_sites(cfg, d.global_sites(rank, halo=1))) if clover else None
    lo = wdd.LocalOperator(torch, d, rank, cfg["m0"], cfg["csw"], Ul, Cl)
    del Ul, Cl
    op = wdd.DistributedOperator(torch, dist, lo)
    ins = [lo.spinor(nrhs) for _ in range(3)]
    outs = [lo.spinor(nrhs) for _ in range(2)]
    for k in range(3):
        psi = wdinputs.spinor_sites(cfg["spinor_seed"] + 100 * k, d.global_sites(rank), nrhs)
        wd.wd_pack_spinor(lo.h, ins[k], psi, nrhs)
    del psi
    torch.cuda.synchronize()
    kname = wd.wd_kernel_name(wd.wd_kernel_for(lo.h, nrhs))

    def step(k):
        op.apply(outs[k % 2], ins[k % 3], nrhs)

    for k in range(args.warmup):
        step(k)
    torch.cuda.synchronize()
    dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = wd.wd_launch_count(lo.h)
    torch.cuda.synchronize()
    e0.record(lo.stream)
    for k in range(args.steps):
        step(k)
    e1.record(lo.stream)
    torch.cuda.synchronize()
    launches = wd.wd_launch_count(lo.h) - launches0
    sampler.stop_flag = True
    sampler.join()
    total_ms, _ = reduce_over_ranks(e0.elapsed_time(e1), 0, dist, "cuda")
    units = V * nrhs * args.steps  # the GLOBAL lattice, once per step
    site_rhs_per_s = units / (total_ms * 1e-3)
    peak, peak_src = peak_hbm()
    alg_bytes_step = V * (576 + (576 if clover else 0) + 384 * nrhs)
    face_bytes = sum(2 * wd.wd_dd_face_bytes(lo.h, mu, nrhs) for mu in d.decomposed)
    achieved = alg_bytes_step / world / (total_ms / args.steps * 1e-3) / 1e9  # per GPU
    line = {
        "metric": METRIC, "value": site_rhs_per_s * flop / 1e9, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "strong",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic", "sites_per_s": site_rhs_per_s,
        "config": {"workload": cfg["name"], "lattice": list(dims), "m0": cfg["m0"], "csw": cfg["csw"], "nrhs": nrhs,
                   "kernel": kname, "variant": "fused", "parallelism": f"dd grid {d.grid} local {d.local_dims}",
                   "exchange": "half-spinor faces (96 B per face site and direction), NCCL send/recv on a side stream",
                   "l2": f"inputs larger than L2 ({alg_bytes_step / world / 1e9:.2f} GB touched per GPU and step)"},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": None, "peak_source": peak_src, "kernel": kname + "/fused+dd",
                     "algorithmic_bytes_per_launch": alg_bytes_step / world,
                     "nvlink_bytes_sent_per_gpu_and_step": face_bytes,
                     "note": "per GPU: its share of the algorithmic bytes / time of the whole step (pack, interior, exterior)"},
        "gpu_launches": launches, "clocks": sampler.summary(),
    }
    lo.close()
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


def sustained_record(torch, step, stream, local, seconds, ms_guess, alg_bytes_step, flop_step, peak):
    """Back-to-back applications for >= `seconds` (two batches of ~0.1 s always in flight, so the GPU never idles); the
    figure reported is that of the LAST second, with the SM clock, power and throttle reasons sampled during that second:
    the steady state under the board's power cap, which a 20-step burst at full clock does not show."""
    batch = max(5, int(0.1 / (ms_guess * 1e-3)))
    counter = [0]

    def enqueue():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(batch):
            step(counter[0])
            counter[0] += 1
        e1.record(stream)
        return e0, e1

    def run_for(sec):
        times, t0 = [], time.time()
        pending = enqueue()
        while True:
            nxt = enqueue() if time.time() - t0 < sec else None
            pending[1].synchronize()
            times.append(pending[0].elapsed_time(pending[1]))
            if nxt is None:
                return times
            pending = nxt

    by_second = []  # ms per step of every whole second before the last one: shows the drift towards the steady state
    soak = []
    for _ in range(max(int(round(seconds)) - 1, 1)):
        sec = run_for(1.0)
        by_second.append(round(sum(sec) / (len(sec) * batch), 4))
        soak += sec
    smp = ClockSampler(local)
    smp.start()
    last = run_for(1.0)
    smp.stop_flag = True
    smp.join()
    ms = sum(last) / (len(last) * batch)
    by_second.append(round(ms, 4))
    gbs = alg_bytes_step / (ms * 1e-3) / 1e9
    return {"seconds": seconds, "ms_per_step": ms, "steps_total": (len(soak) + len(last)) * batch,
            "steps_in_last_second": len(last) * batch, "first_batch_ms_per_step": soak[0] / batch, "ms_per_step_by_second": by_second,
            "value": flop_step / (ms * 1e-3) / 1e9, "unit": "GFLOP/s", "achieved_gbs": gbs, "frac": gbs / peak,
            "frac_of_8000_spec": gbs / 8000.0, "clocks": smp.summary(),
            "what": "ms per step, algorithmic GB/s and clocks of the last second of the run"}


def cfg5_record(torch, wd, wdinputs, local, steps, warmup, peak):
    """BASELINE.json configs[4] (48^3 x 96, Wilson-clover, 12 right-hand sides, blocked multi-RHS layout) as a sub-record of
    the default line: same timing rules as the main record (device events on the launching stream, inputs resident and
    far larger than L2, clocks sampled during the timed region)."""
    cfg = dict(wdinputs.CONFIGS[5])
    dims, nrhs = cfg["dims"], cfg["nrhs"]
    V = wdinputs.volume(dims)
    h = wd.wd_create(*dims, cfg["m0"], cfg["csw"])
    try:
        stream = torch.cuda.current_stream()
        wd.wd_set_stream(h, stream.cuda_stream)
        wd.wd_set_option(h, wd.WD_OPT_DEVICE_PACK, 1)
        wd.wd_set_option(h, wd.WD_OPT_RHS_BLOCK, 4)
        U = wdinputs.config_gauge(cfg)
        wd.wd_load_gauge(h, U)
        del U
        wd.wd_build_clover(h)
        n64 = wd.wd_spinor_bytes(h, nrhs) // 8
        unit64 = wd.wd_spinor_bytes(h, 4) // 8
        ins = [torch.empty(n64, dtype=torch.float64, device="cuda") for _ in range(2)]
        outs = [torch.empty(n64, dtype=torch.float64, device="cuda") for _ in range(2)]
        for u in range(nrhs // 4):  # a unit of four right-hand sides at a time (8 GB of host memory, not 24)
            part = wdinputs.spinor(dims, cfg["spinor_seed"] + u, nrhs=4)
            wd.wd_pack_spinor(h, ins[0][u * unit64:], part, 4)
            del part
        wd.wd_apply(h, ins[1], ins[0], nrhs)
        ins[1].mul_(1.0 / 8.0)
        torch.cuda.synchronize()
        kname = wd.wd_kernel_name(wd.wd_kernel_for(h, nrhs))
        for k in range(warmup):
            wd.wd_apply(h, outs[k % 2], ins[k % 2], nrhs)
        torch.cuda.synchronize()
        smp = ClockSampler(local)
        smp.start()
        l0 = wd.wd_launch_count(h)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for k in range(steps):
            wd.wd_apply(h, outs[k % 2], ins[k % 2], nrhs)
        e1.record(stream)
        torch.cuda.synchronize()
        launches = wd.wd_launch_count(h) - l0
        smp.stop_flag = True
        smp.join()
        ms = e0.elapsed_time(e1) / steps
        alg = V * (576 + 576 + 384 * nrhs)
        gbs = alg / (ms * 1e-3) / 1e9
        traffic, traffic_src = ncu_traffic(kname + f"/clover/x{nrhs}@" + "x".join(map(str, dims)))
        return {"workload": cfg["name"], "lattice": list(dims), "nrhs": nrhs, "kernel": kname, "rhs_layout": "blocked [unit][12][Vs][4]",
                "steps": steps, "warmup": warmup, "ms_per_step": ms, "value": V * nrhs * (FLOP_WILSON + FLOP_CLOVER) / (ms * 1e-3) / 1e9,
                "unit": "GFLOP/s", "site_rhs_per_s": V * nrhs / (ms * 1e-3), "algorithmic_bytes_per_launch": alg, "achieved_gbs": gbs,
                "frac": gbs / peak, "hbm_roof_ms": alg / (peak * 1e9) * 1e3, "traffic": traffic, "traffic_source": traffic_src,
                "gpu_launches": launches, "clocks": smp.summary()}
    finally:
        wd.wd_destroy(h)


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

        # NCCL logging stays on (stderr; the JSON line is the only thing on stdout): which transport each pair got
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT,P2P")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        if args.parallel == "dd":
            return run_dd(args, torch, dist, world, rank, local)

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
    if args.rhs_block == 0:  # cfg 5 ("multi-tuple layout"): the blocked layout where it exists
        fits = dims[1] % 2 == 0 and dims[2] % 4 == 0 and dims[3] % 8 == 0
        args.rhs_block = 4 if (nrhs >= 4 and fits and args.variant == 0 and not args.kernel) else 1
    if args.rhs_block != 1:
        wd.wd_set_option(h, wd.WD_OPT_RHS_BLOCK, args.rhs_block)
    if args.kernel:
        wd.wd_set_option(h, wd.WD_OPT_KERNEL, wd.kernel_id(args.kernel))
    if args.tchunk:
        wd.wd_set_option(h, wd.WD_OPT_TCHUNK, args.tchunk)
    if args.zgroup:
        wd.wd_set_option(h, wd.WD_OPT_ZGROUP, args.zgroup)
    if args.gauge_rows == 2:
        wd.wd_set_option(h, wd.WD_OPT_GAUGE_ROWS, 2)
        gauge_b = 384  # rows 0 and 1 only: the roofline is reported against the reduced byte count
        alg_bytes_site_rhs = (gauge_b + self_b) / nrhs + 384
        alg_bytes_step = V * (gauge_b + self_b + 384 * nrhs)
    U = wdinputs.config_gauge(cfg)
    t_setup = time.time()
    wd.wd_load_gauge(h, U)  # synchronous: H2D copy of the canonical array + transpose on the device (WD_OPT_DEVICE_PACK)
    setup = {"load_gauge_ms": (time.time() - t_setup) * 1e3, "gauge_bytes": V * 576}
    del U
    if clover:
        c0, c1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        c0.record(stream)
        wd.wd_build_clover(h)  # the first launch of a kernel also pays for loading its code
        c1.record(stream)
        torch.cuda.synchronize()
        first_ms = c0.elapsed_time(c1)
        c0.record(stream)
        wd.wd_build_clover(h)
        c1.record(stream)
        torch.cuda.synchronize()
        cms = c0.elapsed_time(c1)
        setup.update({"build_clover_ms": cms, "build_clover_first_call_ms": first_ms, "build_clover_tflops": V * 60 * 198 / (cms * 1e-3) / 1e12,
                      "build_clover_gbs": V * 1152 / (cms * 1e-3) / 1e9,
                      "build_clover_what": "k_build_clover, second call: 60 3x3 complex products per site (FP64-bound), reads U, writes S"})
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
    traffic, traffic_src = (ncu_traffic(kname + ("/clover" if clover else "/wilson") + ("" if nrhs == 1 else f"/x{nrhs}")
                                        + ("/rows2" if args.gauge_rows == 2 else "")
                                        + "@" + "x".join(map(str, dims))))
    roofline = {
        "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "traffic": traffic, "traffic_source": traffic_src,  # a constant from the committed ncu capture of this
        "peak_source": peak_src,                            # kernel on this workload — not measured in this run
        "kernel": kname + ("/fused" if args.variant == 0 else "/unfused"),
        "algorithmic_bytes_per_launch": alg_bytes_launch, "avg_launch_ms": avg_launch_ms,
        "best_launch_ms": min(per_step) / launches_per_step,
        "frac_of_8000_spec": achieved / 8000.0,
    }
    if traffic:  # the two ways SURVEY.md section 8(d) asks for: algorithmic GB/s and the DRAM bytes ncu counted / time
        roofline["traffic_gbs"] = traffic / (avg_launch_ms * 1e-3) / 1e9
        roofline["reuse_efficiency"] = alg_bytes_launch / traffic  # 1.0 = every byte fetched once

    line = {
        "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
        # --parallel dd (the default): the N > 1 lines cut this same lattice over N ranks, so the N = 1 point of that curve is
        # a strong-scaling point; replicas: per-GPU work fixed
        "scaling": "strong" if args.parallel == "dd" else "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "sites_per_s": site_rhs_per_s, "hbm_gbs_algorithmic": site_rhs_per_s * alg_bytes_site_rhs / 1e9,
        "config": {"workload": cfg["name"], "lattice": list(dims), "m0": cfg["m0"], "csw": cfg["csw"],
                   "nrhs": nrhs, "kernel": kname, "variant": "fused" if args.variant == 0 else "unfused", "gauge_rows": args.gauge_rows,
                   "rhs_layout": "plain [nrhs][12][Vs]" if args.rhs_block == 1 else f"blocked [unit][12][Vs][{args.rhs_block}]",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"inputs larger than L2 ({alg_bytes_step / 1e9:.2f} GB touched per step); "
                         "3 inputs / 2 outputs rotate"},
        "roofline": roofline, "gpu_launches": launches, "clocks": sampler.summary(), "setup": setup,
    }

    # ---- the steady state of the power cap: seconds of back-to-back applications, the last second reported
    if args.sustain_seconds > 0 and rank == 0 and world == 1:
        line["sustained"] = sustained_record(torch, step, stream, local, args.sustain_seconds, ms_per_step, alg_bytes_step,
                                             V * nrhs * flop, peak)
    # ---- end to end through the C-ABI with HOST buffers (pinned), copies inside the timed region
    if args.rhs_block != 1:  # the host-to-host path, the FP32 variant and GMRES below use the plain device layout
        wd.wd_set_option(h, wd.WD_OPT_RHS_BLOCK, 1)
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
        # the bound of that path: one right-hand side up and one down AT THE SAME TIME, plain copies on two streams
        one = hin.numel() // nrhs
        dbuf = [torch.empty(one, dtype=torch.float64, device="cuda") for _ in range(2)]
        s_up, s_dn = torch.cuda.Stream(), torch.cuda.Stream()
        best = 1e30
        for _ in range(3):
            torch.cuda.synchronize()
            e0.record(stream)
            s_up.wait_stream(stream)
            s_dn.wait_stream(stream)
            with torch.cuda.stream(s_up):
                dbuf[0].copy_(hin.view(-1)[:one], non_blocking=True)
            with torch.cuda.stream(s_dn):
                hout.view(-1)[:one].copy_(dbuf[1], non_blocking=True)
            stream.wait_stream(s_up)
            stream.wait_stream(s_dn)
            e1.record(stream)
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        line["e2e"]["pcie_bidirectional_ms_per_rhs"] = best
        line["e2e"]["frac_of_pcie_bound"] = best * nrhs / ms
        del dbuf
        del hin, hout
    # ---- the FP32 variant on the same workload: 768 instead of 1536 algorithmic B/site
    if args.f32 and rank == 0:
        wd.wd_enable_f32(h)
        n32 = wd.wd_spinor_bytes_f32(h, nrhs) // 4
        fin = [torch.empty(n32, dtype=torch.float32, device="cuda") for _ in range(3)]
        fout = [torch.empty(n32, dtype=torch.float32, device="cuda") for _ in range(2)]
        for k in range(3):
            wd.wd_convert_spinor(h, fin[k], ins[k], nrhs, True)
        for k in range(5):
            wd.wd_apply_f32(h, fout[k % 2], fin[k % 3], nrhs)
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        nst = max(10, args.steps // 4)
        f0.record(stream)
        for k in range(nst):
            wd.wd_apply_f32(h, fout[k % 2], fin[k % 3], nrhs)
        f1.record(stream)
        torch.cuda.synchronize()
        fms = f0.elapsed_time(f1) / nst
        line["f32"] = {"ms_per_step": fms, "steps": nst, "value": V * nrhs * flop / (fms * 1e-3) / 1e9, "unit": "GFLOP/s",
                       "dtype": "f32", "algorithmic_gbs": alg_bytes_step / 2 / (fms * 1e-3) / 1e9,
                       "frac_of_measured_peak": alg_bytes_step / 2 / (fms * 1e-3) / 1e9 / peak,
                       "kernel": "tma_2x4x16<float2>: the TMA kernel on 8-byte elements, two persistent CTAs per SM"}
        del fin, fout
    # ---- restarted GMRES(M) on the device around the operator: the consumer of the applies
    if args.gmres and rank == 0 and nrhs == 1:
        gs = torch.cuda.Stream()
        wd.wd_set_stream(h, gs.cuda_stream)
        M, cycles_max = args.gmres, 10
        res = {}
        with torch.cuda.stream(gs):
            for label, graph in (("graph", 1), ("eager", 0)):
                wd.wd_set_option(h, wd.WD_OPT_GMRES_GRAPH, graph)
                hist = np.zeros(cycles_max + 1)
                for rep in range(2):  # first repetition: work-space allocation, graph capture
                    outs[0].zero_()
                    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    l0 = wd.wd_launch_count(h)
                    g0.record(gs)
                    cyc = wd.wd_gmres(h, outs[0], ins[0], M, cycles_max, 1e-30, hist)  # tol unreachable: all cycles run
                    g1.record(gs)
                    gs.synchronize()
                ms = g0.elapsed_time(g1)
                res[label] = {"ms_per_cycle": ms / max(cyc, 1), "cycles": cyc, "launches": wd.wd_launch_count(h) - l0,
                              "applies": cyc * (M + 1) + 1, "resid_drop": float(hist[cyc] / hist[0]) if hist[0] else None}
            # the same cycles with single-precision Krylov vectors and operator applications (wd_gmres_mixed)
            wd.wd_enable_f32(h)
            hist = np.zeros(cycles_max + 1)
            for rep in range(2):
                outs[0].zero_()
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                l0 = wd.wd_launch_count(h)
                g0.record(gs)
                cyc = wd.wd_gmres_mixed(h, outs[0], ins[0], M, cycles_max, 1e-30, hist)
                g1.record(gs)
                gs.synchronize()
            ms = g0.elapsed_time(g1)
            res["mixed"] = {"ms_per_cycle": ms / max(cyc, 1), "cycles": cyc, "launches": wd.wd_launch_count(h) - l0,
                            "resid_drop": float(hist[cyc] / hist[0]) if hist[0] else None,
                            "what": "Krylov vectors and M applications per cycle in FP32, residual and solution in FP64"}
        apply_ms = ms_per_step * (M + 1)
        line["gmres"] = {"m": M, **res, "apply_ms_per_cycle": apply_ms,
                         "operator_share_of_cycle": apply_ms / res["graph"]["ms_per_cycle"],
                         "note": "one cycle = M + 1 operator applications + modified Gram-Schmidt (fused axpy+dot kernels), "
                                 "least squares and update on the device; graph = cycles 2.. replayed as one CUDA graph"}
        wd.wd_set_stream(h, stream.cuda_stream)
    # ---- the K steps as ONE CUDA graph (cfg 3: "100 back-to-back applies ... also as one CUDA graph")
    if args.graph and rank == 0:
        gs = torch.cuda.Stream()
        wd.wd_set_stream(h, gs.cuda_stream)
        with torch.cuda.stream(gs):
            for k in range(3):
                step(k)
            gs.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=gs):
                for k in range(args.steps):
                    step(k)
            graph.replay()
            gs.synchronize()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(gs)
            graph.replay()
            g1.record(gs)
            gs.synchronize()
        gms = g0.elapsed_time(g1) / args.steps
        line["graph"] = {"ms_per_step": gms, "steps_in_graph": args.steps,
                         "value": V * nrhs * flop / (gms * 1e-3) / 1e9, "unit": "GFLOP/s"}
        wd.wd_set_stream(h, stream.cuda_stream)
        del graph
    wd.wd_destroy(h)
    del ins, outs
    torch.cuda.empty_cache()
    # ---- cfg 5 (12 right-hand sides) in the same line, now that cfg 4's buffers are gone
    if rank == 0 and world == 1 and args.config == 4 and not args.dims and not args.nrhs and not args.no_cfg5:
        try:
            line["cfg5"] = cfg5_record(torch, wd, wdinputs, local, max(5, min(args.steps, 20)), max(3, min(args.warmup, 5)), peak)
        except Exception as exc:  # a sub-record never costs the main line
            line["cfg5"] = {"error": repr(exc)}
        torch.cuda.empty_cache()

    # ---- ceilings measured on this GPU in this run (bench-only library, include/wd_bench.h): streaming read-only /
    # copy / 7 reads per write (the operator's mix), and the FP64 FMA roof that co-limits a multi-RHS application
    if rank == 0 and not args.no_ceilings:
        from paper_2407_00041_b200 import benchlib

        try:
            nb = 8 << 30
            roofline["stream_read_only_gbs"] = benchlib.wdb_measure_stream(0, nb, 5)
            roofline["stream_copy_gbs"] = benchlib.wdb_measure_stream(1, nb // 2, 5)
            roofline["stream_7r1w_gbs"] = benchlib.wdb_measure_stream(2, nb, 5)
            roofline["frac_of_stream_7r1w"] = achieved / roofline["stream_7r1w_gbs"]
            fs = ClockSampler(local)
            fs.start()
            fp64 = max(benchlib.wdb_measure_fp64(1024, 8, False)[0] for _ in range(5))
            fs.stop_flag = True
            fs.join()
            roofline["fp64_peak_tflops_measured"] = fp64
            roofline["fp64_peak_clocks"] = fs.summary()
            roofline["fp64_peak_how"] = "best of 5, 1024 threads x 8 chains per SM, register-only DFMA"
            roofline["frac_of_fp64_peak"] = (value / 1e3) / fp64
            if nrhs > 1:  # the measurement behind the lane mapping of the quad kernels
                roofline["lds128_cycles_per_warp_instruction"] = {
                    name: round(benchlib.wdb_measure_lds(k), 3) for k, name in enumerate(benchlib.LDS_PATTERNS)}
        except Exception as exc:  # the ceilings are context, never the reason a bench line is lost
            roofline["ceilings_error"] = repr(exc)

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        try:
            line["cpu_baseline"] = cpu_baseline_sample(cfg)
        except Exception as exc:  # never lose the GPU line to the host-side baseline
            line["cpu_baseline"] = {"value": None, "unit": "GFLOP/s", "cores": None, "kind": "oracle", "sample": "failed: " + repr(exc)}
    if dist:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    a = parse_args()
    if a.print_source_hash:
        print(kernel_source_hash(a.print_source_hash))
    elif a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
