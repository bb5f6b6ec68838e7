#!/usr/bin/env python
"""bench.py -- proton histories/s of the whole pbs4d hot path on B200 (BASELINE.json metric).

A step = one pass of the whole path over one synthetic plan: HU->density for every phase, DVF
upload, delivery simulation, Monte Carlo transport + scoring + finalize for every phase that receives protons,
subvoxel accumulation onto the reference phase.  `value` times it with inputs resident in HBM; `e2e` times the
C-ABI call pbs4d_run_plan_host with HOST buffers (H2D/D2H inside).  One JSON line on stdout (rank 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config5|config3|config2] [--impl reference]
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# algorithmic work of one condensed-history step, in fp32/int32 lane-operations
OPS_PER_STEP = 262
# dram__bytes_read.sum + dram__bytes_write.sum of one transport_kernel launch (ncu --set full, profiles/)
# histories of the bounded oracle sample (10-30 s of host work on 16 cores); the reference arm uses half per step
ORACLE_SAMPLE = {"config5": 200_000, "config3": 400_000, "config2": 200_000}
TRANSPORT_DRAM_BYTES_PER_LAUNCH = {"config3": 7.6e6, "config5": 74.8e6}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config5", choices=["config5", "config3", "config2"])
    ap.add_argument("--histories", type=int, default=0, help="override the config's history count (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def make_workload(name, rank, histories=0):
    from paper_1809_03927_b200 import synth
    if name == "config5":
        cfg = synth.config5(seed=5 + 1000 * rank)
    elif name == "config3":
        cfg = synth.config3(seed=3 + 1000 * rank)
    else:
        cfg = synth.config2(seed=2 + 1000 * rank)
        cfg.update(dvf=[None], dvf_grid=None, ref_phase=0, subvox=(2, 2, 2))
    if histories:
        cfg["histories"] = histories
    return cfg


class ClockSampler(threading.Thread):
    """samples SM clock and throttle reasons through NVML during the timed region (the recipe's clocks line; NVML
    in-process instead of spawning nvidia-smi, which perturbs the host thread that issues the launches)"""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.sm, self.mx, self.reasons, self.stop_flag = index, [], [], set(), False

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown",
                     nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                     nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown",
                     nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap"}
            while not self.stop_flag:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                self.mx.append(float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)))
                mask = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
                time.sleep(0.1)
        except Exception as e:                                  # no NVML: report nothing rather than guess
            self.error = repr(e)

    def summary(self):
        self.stop_flag = True
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None,
                "sm_max_mhz": max(self.mx) if self.mx else None, "reasons": sorted(self.reasons),
                "samples": len(self.sm), **({"error": self.error} if hasattr(self, "error") else {})}


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def oracle_sample(cfg, budget_hist):
    """CPU oracle (as it stands) on a bounded sample of the same workload: the plan with `budget_hist` histories
    allocated over its segments, transported on every phase that receives protons.  Returns (hist/s, cores, text)."""
    import oracle as orc
    t0 = time.time()
    segs, _, _ = orc.simulate_delivery(cfg["fields"], cfg["spots"], cfg["deliv"], budget_hist)
    k = orc.fixed_shift(segs, cfg["spots"])
    g = cfg["ct_grid"] if cfg["dose_grid"] is None else cfg["dose_grid"]
    n = 0
    t_tr = 0.0
    for p in sorted(set(int(x) for x in segs["phase"])):
        rho = orc.hu_to_density(cfg["ct_grid"], cfg["hu"][p], cfg["dose_grid"])
        t1 = time.time()
        _, st, _, _ = orc.transport(g, rho, cfg["fields"], cfg["spots"], segs[segs["phase"] == p], cfg["seed"], k)
        t_tr += time.time() - t1
        n += int(st["histories"])
    wall = time.time() - t0
    cores = len(os.sched_getaffinity(0))
    return n / wall, cores, (f"{n} histories of the {cfg['name']} plan over its delivered phases "
                             f"(delivery + HU->density + transport; {wall:.1f} s wall, transport {t_tr:.1f} s)")


def reduce_over_ranks(ms, e2e_s, hist, hist_e2e, world, device):
    """Replicas: every rank ran an independent plan.  Times -> MAX over ranks, histories -> SUM over ranks
    (whole-job throughput = all histories / slowest rank's time).  The only collectives of the whole program."""
    if world <= 1:
        return ms, e2e_s, hist, hist_e2e
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms, e2e_s], dtype=torch.float64, device=device)
    n = torch.tensor([float(hist), float(hist_e2e)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), float(n[0]), float(n[1])


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores (rank 0 only)."""
    if rank != 0:
        return
    cfg = make_workload(args.workload, 0, args.histories)
    budget = ORACLE_SAMPLE[args.workload] // 2
    rates, text, cores = [], "", 0
    for i in range(args.warmup + args.steps):
        r, cores, text = oracle_sample(cfg, budget)
        if i >= args.warmup:
            rates.append((budget / r, r))
    tot_t = sum(t for t, _ in rates)
    value = budget * len(rates) / tot_t
    line = {"impl": "reference", "metric": "proton histories/s", "value": value, "unit": "histories/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / len(rates),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "histories_per_step": budget, "note": "bounded sample of the workload"},
            "cpu_baseline": {"value": value, "unit": "histories/s", "cores": cores, "kind": "oracle", "sample": text},
            "e2e": {"value": value, "unit": "histories/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1809_03927_b200 import binding, build
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the pbs4d path has no CPU fallback")
    build.build()
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- inputs: every rank runs an independent plan (replicas / weak scaling) ----
    cfg = make_workload(args.workload, rank, args.histories)
    P = cfg["hu"].shape[0]
    ctx = binding.Context(local_rank)
    hu_dev = torch.from_numpy(cfg["hu"]).cuda()
    dvf_dev = [None if d is None else torch.from_numpy(d).cuda() for d in cfg["dvf"]]
    hu_host = [cfg["hu"][p] for p in range(P)]
    h2d = cfg["hu"].nbytes + sum(d.nbytes for d in cfg["dvf"] if d is not None) + cfg["spots"].nbytes + cfg["fields"].nbytes
    for a in hu_host + [d for d in cfg["dvf"] if d is not None]:
        torch.cuda.cudart().cudaHostRegister(a.ctypes.data, a.nbytes, 0)          # pinned host inputs

    stats = {}

    def step_device():
        ctx.set_ct_phases(cfg["ct_grid"], [hu_dev[p] for p in range(P)], cfg["dose_grid"])
        for p in range(P):
            if dvf_dev[p] is not None:
                ctx.set_dvf(p, cfg["ref_phase"], cfg["dvf_grid"], dvf_dev[p])
        ctx.set_plan_spots(cfg["fields"], cfg["spots"])
        deliv = ctx.simulate_delivery(cfg["deliv"], cfg["histories"])
        phases = sorted(set(int(x) for x in deliv["segments"]["phase"]) | {cfg["ref_phase"]})
        sts, t_ms = ctx.mc_dose_phases(phases, cfg["seed"])          # all phases, concurrent launches; t_ms = fork..join
        n_hist = sum(st["histories"] for st in sts); n_steps = sum(st["steps"] for st in sts)
        n_red = sum(st["scoring_atomics"] for st in sts)
        out, ast = ctx.accumulate_subvoxel(cfg["ref_phase"], cfg["subvox"])
        n_dvf = sum(1 for p in range(P) if dvf_dev[p] is not None and p != cfg["ref_phase"])      # fields re-laid out
        g_ = ctx_shape(cfg)
        n_src = int(ast["subvoxels"]) // (g_[0] * g_[1] * g_[2] * int(np.prod(cfg["subvox"])))   # phases really pushed
        # kernels launched: HU->density per phase, DVF interleave per source phase, transport + dose finalize per
        # phase run, push per source phase, coverage flags + accumulation finalize
        stats.update(histories=n_hist, mc_steps=n_steps, reds=n_red, transport_ms=t_ms, push_ms=ast["push_ms"],
                     finalize_ms=ast["finalize_ms"], phases=len(phases), n_src=n_src, subvoxels=ast["subvoxels"],
                     launches=P + n_dvf + 2 * len(phases) + n_src + 2, checksum=float(out.sum()))
        return n_hist

    out_host = np.zeros(ctx_shape(cfg), np.float32)
    torch.cuda.cudart().cudaHostRegister(out_host.ctypes.data, out_host.nbytes, 0)

    def step_e2e():
        run, secs = ctx.run_plan_host(cfg["ct_grid"], hu_host, cfg["dose_grid"], cfg["dvf_grid"],
                                      cfg["dvf"] if cfg["dvf_grid"] is not None else None, cfg["ref_phase"],
                                      cfg["fields"], cfg["spots"], cfg["deliv"], cfg["histories"], cfg["seed"],
                                      cfg["subvox"], out_host)
        stats["e2e_seconds"] = secs
        return run

    # ---- in-run roofline probes (small kernels of the library itself, before the timed region) ----
    probes = {k: ctx.roofline_probe(k) for k in ("fp32_issue", "red_random", "red_hot", "hbm_copy")}

    # ---- device-resident timing ----
    for _ in range(max(args.warmup, 3)):
        step_device()
    sampler = ClockSampler(local_rank); sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    hist = 0; tr_ms = 0.0; mc_steps = 0; reds = 0
    for _ in range(args.steps):
        hist += step_device(); tr_ms += stats["transport_ms"]; mc_steps += stats["mc_steps"]; reds += stats["reds"]
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.summary()

    # ---- end-to-end timing (host buffers through the C-ABI) ----
    step_e2e()
    barrier()
    t0 = time.perf_counter()
    hist_e2e = 0
    for _ in range(args.steps):
        hist_e2e += step_e2e()
    barrier()
    e2e_s = time.perf_counter() - t0

    ms, e2e_s, hist, hist_e2e = reduce_over_ranks(ms, e2e_s, hist, hist_e2e, world, torch.device("cuda", local_rank))
    if rank != 0:
        return

    peaks, peak_kind = measured_peaks()
    sm_mhz = clocks["sm_mhz"] or peaks.get("sm_max_mhz", 1965.0)
    steps_per_s = mc_steps / (tr_ms * 1e-3)
    achieved = steps_per_s * OPS_PER_STEP / 1e12
    props = torch.cuda.get_device_properties(local_rank)
    nvox = int(np.prod(ctx_shape(cfg)))
    acc_bytes = stats["n_src"] * nvox * (20 + 16)
    fin_bytes = nvox * (16 * stats["n_src"] + 8)
    peak = props.multi_processor_count * 128 * sm_mhz * 1e6 / 1e12
    line = {
        "metric": "proton histories/s", "value": hist / (ms * 1e-3), "unit": "histories/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": args.workload, "histories_per_step": stats["histories"], "phases_run": stats["phases"],
                   "source_phases": stats["n_src"], "subvoxels": list(cfg["subvox"]),
                   "l2": "per-step working set (CT int16 + DVFs + int64 grids) exceeds the 126 MB L2"
                         if args.workload != "config2" else "inputs smaller than L2 (parity config)",
                   "parallelism": "replicas" if world > 1 else "single"},
        "e2e": {"value": hist_e2e / e2e_s, "unit": "histories/s", "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(out_host.nbytes), "seconds_per_plan": e2e_s / args.steps,
                "split_s": stats.get("e2e_seconds")},
        "seconds_per_plan_device": ms * 1e-3 / args.steps,
        "gpu_launches": stats["launches"] * args.steps,
        "kernel_ms_per_step": {"transport": tr_ms / args.steps, "push": stats["push_ms"], "acc_finalize": stats["finalize_ms"]},
        "transport_histories_per_s": hist / world / (tr_ms * 1e-3) if world == 1 else None,
        "clocks": clocks,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tlane-op/s", "frac": achieved / peak,
                     "traffic": TRANSPORT_DRAM_BYTES_PER_LAUNCH.get(args.workload), "kernel": "transport_kernel",
                     "how": f"{OPS_PER_STEP} algorithmic lane-ops/step x {steps_per_s:.3e} steps/s over the CUDA-event time of the "
                            f"transport launches of a pass (fork to join of the per-phase kernels, which overlap at their tails); peak = SMs x 128 lanes x median SM clock under load ({sm_mhz:.0f} MHz, {peak_kind} peaks file); "
                            "traffic = dram bytes read+written per launch from the ncu --set full capture under profiles/",
                     "measured_fp32_issue": probes["fp32_issue"] / 1e12,
                     "frac_of_measured_fp32_issue": achieved / (probes["fp32_issue"] / 1e12),
                     "scoring_atomics_per_s": reds / (tr_ms * 1e-3), "measured_red_random_per_s": probes["red_random"],
                     "measured_red_hot_per_s": probes["red_hot"],
                     "atomic_frac": reds / (tr_ms * 1e-3) / probes["red_random"]},
        "roofline_accumulate": {"bound": "hbm" if max(cfg["subvox"]) <= 2 else "alu", "kernel": "emtm_push_kernel",
                                "achieved": acc_bytes / (stats["push_ms"] * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                                "unit": "GB/s", "frac": acc_bytes / (stats["push_ms"] * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                "measured_hbm_copy": probes["hbm_copy"] / 1e9,
                                "subvoxels_per_s": stats["subvoxels"] / (stats["push_ms"] * 1e-3),
                                "finalize_GBps": fin_bytes / (stats["finalize_ms"] * 1e-3) / 1e9,
                                "how": "algorithmic bytes = 20 B per source voxel (dose, density, 3 DVF components) + 16 B "
                                       "read-modify-write per reference voxel, per source phase, over the push kernels' "
                                       "CUDA-event time; finalize = (16 n_src + 8) B per voxel"},
    }
    if not args.no_cpu_baseline and world == 1:
        r, cores, text = oracle_sample(cfg, ORACLE_SAMPLE[args.workload])
        line["cpu_baseline"] = {"value": r, "unit": "histories/s", "cores": cores, "kind": "oracle", "sample": text}
    print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def ctx_shape(cfg):
    g = cfg["ct_grid"] if cfg["dose_grid"] is None else cfg["dose_grid"]
    return int(g["nz"][0]), int(g["ny"][0]), int(g["nx"][0])


if __name__ == "__main__":
    main()
