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

# hand-count MODEL of the lane-operations of one condensed-history step; used only when the ncu
# summary under profiles/ is missing -- the reported figure is the measured one (profile_metrics)
OPS_PER_STEP_MODEL = 262
# lane-instructions per step that ARE the algorithm (DESIGN.md section 5 census of the transport kernel's SASS: 199.1 for
# the model of every lane + the voxel-change work of the lanes that change voxel); the rest of the executed count is
# loop control, refill and source sampling.  Reported beside the issue utilisation as `frac_algorithmic`.
ALGORITHM_OPS_PER_STEP = 210.0
# histories of the bounded oracle sample (10-30 s of host work on 16 cores); the reference arm uses half per step
ORACLE_SAMPLE = {"config5": 2_000_000, "config3": 4_000_000, "config2": 2_000_000}
# per-kernel numbers taken from the committed ncu captures (kernel, workload, metric, value); written by hand from the
# reports named in profiles/r2_summary.md
PROFILE_CSV = os.path.join(ROOT, "profiles", "r3_kernel_metrics.csv")


def profile_metrics():
    """{(kernel, workload, metric): value} from profiles/r3_kernel_metrics.csv; {} if the file is absent"""
    out = {}
    try:
        with open(PROFILE_CSV) as f:
            for line in f:
                c = [x.strip() for x in line.split(",")]
                if len(c) >= 4 and not line.startswith("#") and c[0] != "kernel":
                    out[(c[0], c[1], c[2])] = float(c[3])
    except OSError:
        pass
    return out


def profile_source_state():
    """{kernel: "current" | "STALE: ..."} -- the `#source,kernel,path,hash` stamps of the metrics file (git blob hash
    of the kernel's source when it was captured) against the same hash of the file in the working tree"""
    import hashlib
    out = {}
    try:
        with open(PROFILE_CSV) as f:
            stamps = [line.strip().split(",") for line in f if line.startswith("#source,")]
    except OSError:
        return out
    for c in stamps:
        if len(c) < 4:
            continue
        kernel, path, want = c[1], c[2], c[3]
        try:
            data = open(os.path.join(ROOT, path), "rb").read()
            have = hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()
        except OSError:
            have = "missing"
        out[kernel] = "current" if have == want else \
            f"STALE: {path} is {have[:10]}, the capture was taken of {want[:10]} -- re-capture and re-stamp"
    return out


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config5", choices=["config5", "config3", "config2", "config4"],
                    help="config5 (default, the metric's config), config3, config2: the whole path; config4: the "
                         "accumulation stress of BASELINE.json config 4 alone (push / DIM at n = 2, 4, 8 and (2,2,5))")
    ap.add_argument("--histories", type=int, default=0, help="override the config's history count (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--dry-ranks", action="store_true",
                    help="launch check without a GPU: start the ranks, count them over gloo, print {'dry': true, ...}")
    return ap.parse_args()


def free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_ranks(args):
    """`python bench.py --gpus N` (N > 1) outside a launcher: start N ranks of this same command, one per GPU, through
    torch.distributed.run on 127.0.0.1 (the line the driver uses) and hand back its exit code.  Rank 0 prints the one
    JSON line.  Fails loudly when fewer than N devices are visible; NCCL's own logging is left as the caller set it."""
    if not args.dry_ranks:
        import torch
        have = torch.cuda.device_count()
        if have < args.gpus:
            raise SystemExit(f"bench.py --gpus {args.gpus}: only {have} CUDA device(s) visible")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def dry_ranks(args, rank, world):
    """the launch path alone (CPU, gloo): every rank joins, the ranks are counted with an all-reduce, rank 0 prints"""
    import torch
    import torch.distributed as dist
    seen = 1
    if world > 1:
        dist.init_process_group("gloo")
        t = torch.ones(1, dtype=torch.int64)
        dist.all_reduce(t)
        seen = int(t[0])
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"dry": True, "n_gpus": world, "ranks_seen": seen, "requested": args.gpus}), flush=True)


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
    cores = orc.threads()                                       # the threads the oracle's history loop ran on
    return n / wall, cores, (f"{n} histories of the {cfg['name']} plan over its delivered phases "
                             f"(delivery + HU->density + transport; {wall:.1f} s wall, transport {t_tr:.1f} s)")


def source_owners(src_phases, world):
    """accumulation shards by source phase: the i-th source phase (ascending) is pushed by rank i % world"""
    return {p: i % world for i, p in enumerate(sorted(src_phases))}


def owner_mask(owners, rank):
    m = 0
    for p, r in owners.items():
        if r == rank:
            m |= 1 << p
    return m


def sum_energy_grids(grids, world):
    """integer all-reduce (SUM) of the int64 energy grids of the phases, in place: exact and order-independent, so
    every rank ends up with the grid of the unsharded run bit for bit"""
    if world <= 1:
        return
    import torch.distributed as dist
    for q in grids:
        assert q.dtype.is_floating_point is False and q.element_size() == 8
        dist.all_reduce(q, op=dist.ReduceOp.SUM)


def share_accumulators(pairs, owners, world):
    """pairs: {source phase: (E, M)} int64 sums; broadcast each from the rank that pushed it"""
    if world <= 1:
        return
    import torch.distributed as dist
    for p in sorted(pairs):
        for t in pairs[p]:
            dist.broadcast(t, src=owners[p])


def run_accumulation_stress(args):
    """--workload config4 (BASELINE.json:10): 10 phase doses of 128^3 at 2 mm, random smooth DVFs |u| <= 20 mm,
    accumulated onto phase 0 at subvoxel edges 1.0 / 0.5 / 0.25 mm (n = 2, 4, 8) and at (2,2,5); EMTM push + finalize and
    the DIM pull, each against BOTH rooflines (algorithmic HBM bytes, executed lane-instructions from profiles/).
    One JSON line; launch order is fixed (per subdivision: warm-up + timed calls of 9 source phases each), which is what
    the ncu captures under profiles/ index with -s."""
    import torch
    from paper_1809_03927_b200 import binding, build, synth
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the pbs4d path has no CPU fallback")
    build.build()
    c = synth.config4()
    ctx = binding.Context(0)
    P = len(c["doses"])
    rho = torch.from_numpy(c["rhos"]).cuda(); dose = torch.from_numpy(c["doses"]).cuda()
    ctx.set_density_phases(c["grid"], [rho[p] for p in range(P)])
    disp = [None if d is None else torch.from_numpy(d).cuda() for d in c["disps"]]
    for p in range(P):
        if disp[p] is not None:
            ctx.set_dvf(p, c["ref_phase"], c["dvf_grid"], disp[p])
            ctx.set_dvf_pull(p, c["ref_phase"], c["dvf_grid"], disp[p])
    doses = [dose[p] for p in range(P)]
    n_src = sum(1 for d in disp if d is not None)
    nvox = int(np.prod(c["doses"].shape[1:]))
    peaks, peak_kind = measured_peaks()
    prof = profile_metrics()
    props = torch.cuda.get_device_properties(0)
    # defaults long enough for the NVML sampler (one sample per 0.1 s) to see the clocks under load
    warm, steps = max(args.warmup, 1) if args.warmup != 3 else 2, args.steps if args.steps != 3 else 20
    src_state = profile_source_state()
    for _ in range(warm):                                            # clocks up before the sampler starts
        ctx.accumulate_subvoxel(c["ref_phase"], (4, 4, 4), doses)
    sampler = ClockSampler(0); sampler.start()

    def timed(fn, ns):
        ms = fin = 0.0
        for i in range(warm + steps):
            _, st = fn(c["ref_phase"], ns, doses)
            if i >= warm:
                ms += st["push_ms"]; fin += st["finalize_ms"]
        return ms / steps, fin / steps, st

    out = {"metric": "subvoxels/s (accumulation stress)", "unit": "subvoxels/s", "n_gpus": 1, "steps": steps,
           "warmup": warm, "higher_is_better": True, "dtype": "f32+i64", "data": "synthetic",
           "config": {"workload": "config4", "grid": list(c["doses"].shape[1:]), "source_phases": n_src},
           "push": {}, "dim": {}}
    raw = {"push": {}, "dim": {}}
    for ns in [(2, 2, 2), (4, 4, 4), (8, 8, 8), (2, 2, 5)]:
        raw["push"][ns] = timed(ctx.accumulate_subvoxel, ns)
    for ns in [(1, 1, 1), (2, 2, 2), (4, 4, 4), (8, 8, 8)]:
        raw["dim"][ns] = timed(ctx.accumulate_dim, ns)
    torch.cuda.synchronize()
    clocks = sampler.summary()
    sm_mhz = clocks["sm_mhz"] or peaks.get("sm_max_mhz", 1965.0)
    issue_peak = props.multi_processor_count * 128 * sm_mhz * 1e6 / 1e12
    out["clocks"] = clocks
    out["peaks"] = {"hbm_GBps": peaks["hbm_gbs"], "issue_Tlaneops": issue_peak, "kind": peak_kind,
                    "issue_how": f"SMs x 128 lanes x median SM clock under load ({sm_mhz:.0f} MHz)"}
    out["lane_ops_source"] = {k: src_state.get(k, "unstamped") for k in ("emtm_push_kernel", "dim_pull_kernel")}
    for ns in [(2, 2, 2), (4, 4, 4), (8, 8, 8), (2, 2, 5)]:
        ms, fin, st = raw["push"][ns]
        key = "x".join(map(str, ns))
        ops = prof.get(("emtm_push_kernel", f"config4_{key}", "thread_inst_per_subvoxel"))
        rate = st["subvoxels"] / (ms * 1e-3)
        gbs = n_src * nvox * 36 / (ms * 1e-3) / 1e9
        out["push"][key] = {"ms": ms, "subvoxels_per_s": rate, "hbm_GBps": gbs, "hbm_frac": gbs / peaks["hbm_gbs"],
                            "lane_ops_per_subvoxel": ops, "issue_frac": None if not ops else rate * ops / 1e12 / issue_peak,
                            "finalize_ms": fin, "finalize_GBps": nvox * (16 * n_src + 8) / (fin * 1e-3) / 1e9}
    for ns in [(1, 1, 1), (2, 2, 2), (4, 4, 4), (8, 8, 8)]:
        ms, fin, st = raw["dim"][ns]
        key = "x".join(map(str, ns))
        ops = prof.get(("dim_pull_kernel", f"config4_{key}", "thread_inst_per_subvoxel"))
        rate = st["subvoxels"] / (ms * 1e-3)
        gbs = n_src * nvox * 36 / (ms * 1e-3) / 1e9                 # DVF float4 + dose + double accumulator RMW per voxel
        out["dim"][key] = {"ms": ms, "subvoxels_per_s": rate, "hbm_GBps": gbs, "hbm_frac": gbs / peaks["hbm_gbs"],
                           "lane_ops_per_subvoxel": ops, "issue_frac": None if not ops else rate * ops / 1e12 / issue_peak}
    out["value"] = out["push"]["2x2x2"]["subvoxels_per_s"]
    print(json.dumps(out), flush=True)
    ctx.close()


def run_pass(ctx, cfg, hu_dev, dvf_dev, rank, world, sum_grids=sum_energy_grids, share=share_accumulators):
    """One pass of the whole path with inputs resident in HBM.  world > 1: this rank's shard --
    its slice of every phase's history range, then the integer all-reduce of the energy grids (`sum_grids`), a7 again,
    the push of the source phases this rank owns, the exchange of the int64 sums (`share`) and a9.
    Returns (histories transported here, 4D dose tensor, stats dict)."""
    P = cfg["hu"].shape[0]
    shape = ctx_shape(cfg)
    nvox = int(np.prod(shape)); n_sub = int(np.prod(cfg["subvox"]))
    ctx.set_ct_phases(cfg["ct_grid"], [hu_dev[p] for p in range(P)], cfg["dose_grid"])
    for p in range(P):
        if dvf_dev[p] is not None:
            ctx.set_dvf(p, cfg["ref_phase"], cfg["dvf_grid"], dvf_dev[p])
    ctx.set_plan_spots(cfg["fields"], cfg["spots"])
    deliv = ctx.simulate_delivery(cfg["deliv"], cfg["histories"])
    phases = sorted(set(int(x) for x in deliv["segments"]["phase"]) | {cfg["ref_phase"]})
    ctx.set_shard(rank, world)
    sts, t_ms = ctx.mc_dose_phases(phases, cfg["seed"])              # all phases, concurrent launches; t_ms = fork..join
    n_hist = sum(st["histories"] for st in sts)
    n_dvf = sum(1 for p in range(P) if dvf_dev[p] is not None and p != cfg["ref_phase"])          # fields re-laid out
    src = [p for p in phases if p != cfg["ref_phase"] and dvf_dev[p] is not None]
    extra = 0
    if world == 1:
        out, ast = ctx.accumulate_subvoxel(cfg["ref_phase"], cfg["subvox"])
    else:
        sum_grids([ctx.phase_energy_view(p) for p in phases], world)                               # the exchange step
        for p in phases:
            ctx.finalize_phase_dose(p)
        owners = source_owners(src, world)
        ast = ctx.accumulate_push(cfg["ref_phase"], cfg["subvox"], owner_mask(owners, rank))
        share({p: ctx.accumulator_views(p) for p in src}, owners, world)
        out, fst = ctx.accumulate_finalize(cfg["ref_phase"])
        ast["finalize_ms"] = fst["finalize_ms"]
        extra = len(phases)                                                                        # second a7 launches
    ctx.set_shard(0, 1)
    n_src = int(ast["subvoxels"]) // (nvox * n_sub)                                               # phases pushed here
    # kernels launched: density table + HU->density per phase, DVF interleave per source phase, transport per phase with histories
    # here, dose finalize per phase run (twice when sharded), push per source phase pushed here, coverage flags +
    # accumulation finalize
    n_tr = sum(1 for st in sts if st["histories"] > 0)
    stats = dict(histories=n_hist, mc_steps=sum(st["steps"] for st in sts), reds=sum(st["scoring_atomics"] for st in sts),
                 transport_ms=t_ms, push_ms=ast["push_ms"], finalize_ms=ast["finalize_ms"], phases=len(phases),
                 n_src=n_src, subvoxels=ast["subvoxels"], launches=2 * P + n_dvf + n_tr + len(phases) + extra + n_src + 2,
                 active=phases, src=src)
    return n_hist, out, stats


def reduce_over_ranks(ms, e2e_s, hist, hist_e2e, world, device):
    """Times -> MAX over ranks, histories -> SUM over ranks (whole-job throughput = all histories / slowest rank's
    time)."""
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
    if args.workload == "config4":
        raise SystemExit("--impl reference times the transport oracle; use --workload config5 | config3 | config2")
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
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if args.impl == "reference":
        run_reference(args, int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))
        return
    if args.gpus > 1 and args.workload != "config4" and "WORLD_SIZE" not in os.environ:
        sys.exit(launch_ranks(args))                             # plain `python bench.py --gpus N`: become N ranks
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus and args.workload != "config4":
        raise SystemExit(f"bench.py: --gpus {args.gpus} but the launcher started {world} rank(s)")
    if args.dry_ranks:
        dry_ranks(args, rank, world)
        return
    if args.workload == "config4":
        if rank == 0:
            run_accumulation_stress(args)
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

    # ---- inputs.  N = 1: the plan of the workload.  N > 1: STRONG scaling -- every rank holds the same plan and
    # transports its slice of every phase's history range; the int64 energy grids are summed over the ranks with one
    # integer all-reduce per phase (NCCL), the accumulation is sharded by source phase and its int64 sums are
    # broadcast from their owners ----
    cfg = make_workload(args.workload, 0, args.histories)
    P = cfg["hu"].shape[0]
    ctx = binding.Context(local_rank)
    hu_dev = torch.from_numpy(cfg["hu"]).cuda()
    dvf_dev = [None if d is None else torch.from_numpy(d).cuda() for d in cfg["dvf"]]
    hu_host = [cfg["hu"][p] for p in range(P)]
    for a in hu_host + [d for d in cfg["dvf"] if d is not None]:
        torch.cuda.cudart().cudaHostRegister(a.ctypes.data, a.nbytes, 0)          # pinned host inputs
    nvox = int(np.prod(ctx_shape(cfg)))
    n_sub = int(np.prod(cfg["subvox"]))

    stats = {}

    def step_device():
        n, out, st = run_pass(ctx, cfg, hu_dev, dvf_dev, rank, world)
        stats.update(st)
        return n, out

    out_host = np.zeros(ctx_shape(cfg), np.float32)
    torch.cuda.cudart().cudaHostRegister(out_host.ctypes.data, out_host.nbytes, 0)
    out_pinned = torch.from_numpy(out_host)

    def step_e2e():
        """the same pass from HOST buffers, copies inside.  N = 1: the C-ABI entry pbs4d_run_plan_host.  N > 1: every
        rank uploads the plan's inputs from pinned host memory, runs its shard, rank 0 reads the 4D dose back."""
        if world == 1:
            run, secs, h2d = ctx.run_plan_host(cfg["ct_grid"], hu_host, cfg["dose_grid"], cfg["dvf_grid"],
                                               cfg["dvf"] if cfg["dvf_grid"] is not None else None, cfg["ref_phase"],
                                               cfg["fields"], cfg["spots"], cfg["deliv"], cfg["histories"],
                                               cfg["seed"], cfg["subvox"], out_host)
            stats.update(e2e_seconds=secs, h2d=h2d)
            return run
        h2d = cfg["spots"].nbytes + cfg["fields"].nbytes
        for p in range(P):
            hu_dev[p].copy_(torch.from_numpy(hu_host[p]), non_blocking=True); h2d += hu_host[p].nbytes
            if dvf_dev[p] is not None:
                dvf_dev[p].copy_(torch.from_numpy(cfg["dvf"][p]), non_blocking=True); h2d += cfg["dvf"][p].nbytes
        n, out = step_device()
        if rank == 0:
            out_pinned.copy_(out, non_blocking=True)
        torch.cuda.synchronize()
        stats.update(h2d=h2d)
        return n

    # ---- in-run roofline probes (small kernels of the library itself, before the timed region) ----
    probes = {k: ctx.roofline_probe(k) for k in ("fp32_issue", "red_random", "red_hot", "hbm_copy")}

    # ---- device-resident timing ----
    for _ in range(max(args.warmup, 3)):
        step_device()
    sampler = ClockSampler(local_rank); sampler.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    hist = 0; tr_ms = 0.0; mc_steps = 0; reds = 0; launches = 0
    for _ in range(args.steps):
        hist += step_device()[0]; tr_ms += stats["transport_ms"]; mc_steps += stats["mc_steps"]; reds += stats["reds"]
        launches += stats["launches"]
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.summary()

    # ---- end-to-end timing (host buffers) ----
    step_e2e()
    barrier()
    t0 = time.perf_counter()
    hist_e2e = 0
    for _ in range(args.steps):
        hist_e2e += step_e2e()
    barrier()
    e2e_s = time.perf_counter() - t0

    ms, e2e_s, hist, hist_e2e = reduce_over_ranks(ms, e2e_s, hist, hist_e2e, world, torch.device("cuda", local_rank))
    if world > 1:                                         # per-rank launch counts and transport steps -> whole job
        tot = torch.tensor([float(launches), float(mc_steps), float(reds)], dtype=torch.float64, device="cuda")
        tmax = torch.tensor([tr_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(tot, op=dist.ReduceOp.SUM); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        launches, mc_steps, reds, tr_ms = int(tot[0]), float(tot[1]), float(tot[2]), float(tmax[0])
    if rank != 0:
        ctx.close()
        dist.destroy_process_group()
        return

    peaks, peak_kind = measured_peaks()
    prof = profile_metrics()
    wl = args.workload
    sm_mhz = clocks["sm_mhz"] or peaks.get("sm_max_mhz", 1965.0)
    steps_per_s = mc_steps / (tr_ms * 1e-3)
    props = torch.cuda.get_device_properties(local_rank)
    peak = world * props.multi_processor_count * 128 * sm_mhz * 1e6 / 1e12
    # lane-instructions per condensed-history step: executed thread instructions of the transport kernel / steps, from
    # the committed ncu capture of the kernel (profiles/); the hand-count model only when that file is missing
    # (a count captured on another workload is not borrowed: the voxel-change share of a step depends on the geometry)
    src_state = profile_source_state()
    ops_step = prof.get(("transport_kernel", wl, "thread_inst_per_step"))
    ops_kind = "ncu smsp__thread_inst_executed / steps (profiles/r3_kernel_metrics.csv), source " + \
        src_state.get("transport_kernel", "unstamped")
    if src_state.get("transport_kernel", "").startswith("STALE"):
        ops_kind = src_state["transport_kernel"]
    if not ops_step:
        ops_step, ops_kind = OPS_PER_STEP_MODEL, f"hand-count model (no ncu capture of the transport kernel on {wl})"
    achieved = steps_per_s * ops_step / 1e12
    acc_bytes = stats["n_src"] * nvox * (20 + 16)
    fin_bytes = nvox * (16 * len(stats["src"]) + 8)
    push_s = stats["push_ms"] * 1e-3
    sub_key = "x".join(str(v) for v in cfg["subvox"])
    push_ops = prof.get(("emtm_push_kernel", f"{wl}_{sub_key}", "thread_inst_per_subvoxel"))
    push_peak = props.multi_processor_count * 128 * sm_mhz * 1e6 / 1e12
    line = {
        "metric": "proton histories/s", "value": hist / (ms * 1e-3), "unit": "histories/s", "n_gpus": world,
        "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "strong" if world > 1 else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": wl, "histories_per_step": int(hist / args.steps), "phases_run": stats["phases"],
                   "source_phases": len(stats["src"]), "subvoxels": list(cfg["subvox"]),
                   "l2": "per-step working set (CT int16 + DVFs + int64 grids) exceeds the 126 MB L2"
                         if wl != "config2" else "inputs smaller than L2 (parity config)",
                   "parallelism": (f"one plan sharded over {world} ranks: history slices + int64 all-reduce of the "
                                   "energy grids, accumulation by source phase") if world > 1 else "single"},
        "e2e": {"value": hist_e2e / e2e_s, "unit": "histories/s", "h2d_bytes_per_step": int(stats["h2d"]),
                "d2h_bytes_per_step": int(out_host.nbytes), "seconds_per_plan": e2e_s / args.steps,
                "split_s": stats.get("e2e_seconds"),
                "note": "h2d bytes are those actually copied: CT and DVF of the phases that receive beam"},
        "seconds_per_plan_device": ms * 1e-3 / args.steps,
        "gpu_launches": launches,
        "kernel_ms_per_step": {"transport": tr_ms / args.steps, "push": stats["push_ms"], "acc_finalize": stats["finalize_ms"]},
        "transport_histories_per_s": hist / (tr_ms * 1e-3),
        "mc_steps_per_plan": mc_steps / args.steps,
        "clocks": clocks,
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tlane-op/s", "frac": achieved / peak,
                     "frac_kind": "issue utilisation: EXECUTED lane-instructions (algorithm + loop/refill overhead) over the "
                                  "lane-issue peak",
                     "frac_algorithmic": steps_per_s * ALGORITHM_OPS_PER_STEP / 1e12 / peak,
                     "algorithmic_lane_ops_per_step": ALGORITHM_OPS_PER_STEP,
                     "traffic": prof.get(("transport_kernel", wl, "dram_bytes_per_launch")), "kernel": "transport_kernel",
                     "lane_ops_per_step": ops_step, "lane_ops_source": ops_kind,
                     "how": f"{ops_step:.1f} executed lane-instructions per step x {steps_per_s:.3e} steps/s over the CUDA-event time of the "
                            f"transport launches of a pass (fork to join of the per-phase kernels, which overlap at their tails); peak = SMs x 128 lanes x median SM clock under load ({sm_mhz:.0f} MHz, {peak_kind} peaks file); "
                            "traffic = dram bytes read+written per launch from the ncu --set full capture under profiles/",
                     "measured_fp32_issue": probes["fp32_issue"] / 1e12,
                     "frac_of_measured_fp32_issue": achieved / (world * probes["fp32_issue"] / 1e12),
                     "scoring_atomics_per_s": reds / (tr_ms * 1e-3), "measured_red_random_per_s": probes["red_random"],
                     "measured_red_hot_per_s": probes["red_hot"],
                     "atomic_frac": reds / (tr_ms * 1e-3) / (world * probes["red_random"])},
        # the push kernel against BOTH rooflines: algorithmic HBM bytes and executed lane-instructions
        "roofline_accumulate": {"kernel": "emtm_push_kernel", "subvoxels": list(cfg["subvox"]),
                                "hbm": {"bound": "hbm", "achieved": acc_bytes / push_s / 1e9, "peak": peaks["hbm_gbs"],
                                        "unit": "GB/s", "frac": acc_bytes / push_s / 1e9 / peaks["hbm_gbs"],
                                        "traffic": prof.get(("emtm_push_kernel", f"{wl}_{sub_key}", "dram_bytes_per_launch"))},
                                "issue": None if not push_ops else
                                {"bound": "alu", "achieved": stats["subvoxels"] / push_s * push_ops / 1e12, "peak": push_peak,
                                 "unit": "Tlane-op/s", "frac": stats["subvoxels"] / push_s * push_ops / 1e12 / push_peak,
                                 "lane_ops_per_subvoxel": push_ops},
                                "binding": "alu" if push_ops else "unknown (no ncu capture for this subdivision)",
                                "lane_ops_source": src_state.get("emtm_push_kernel", "unstamped"),
                                "measured_hbm_copy": probes["hbm_copy"] / 1e9,
                                "subvoxels_per_s": stats["subvoxels"] / push_s,
                                "finalize_GBps": fin_bytes / (stats["finalize_ms"] * 1e-3) / 1e9,
                                "how": "hbm: algorithmic bytes = 20 B per source voxel (dose, density, 3 DVF components) + 16 B "
                                       "read-modify-write per reference voxel, per source phase, over the push kernels' "
                                       "CUDA-event time; issue: executed lane-instructions per subvoxel from the ncu capture "
                                       "under profiles/ x subvoxels/s; finalize = (16 n_src + 8) B per voxel"},
    }
    if not args.no_cpu_baseline and world == 1:
        r, cores, text = oracle_sample(cfg, ORACLE_SAMPLE[wl])
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
