#!/usr/bin/env python
"""bench.py -- spin updates/s of the Viana-Bray hot path on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--T 1.0]

Workload (N=1): BASELINE.json configs[2], the bandwidth-bound roofline config: VB N=2^24, c=4, 64 samples
(1 word) per site, T=1.0, seed 1.  One STEP = one pass of the whole hot path on the resident instance:
  sg_sweep(SWEEPS_PER_STEP) + sg_snapshot + sg_correlation + sg_energy
value = spin updates (Metropolis trials, Q23) of all ranks / device time (max over ranks).
N>1: the path shards by sample: every rank runs its own 64-sample replica of the same
recipe with seed+rank, no data-path collective ("weak" scaling).
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SWEEPS_PER_STEP = 64
BYTES_PER_SITE_WORD = 80.0          # own word 8 + 4 neighbour words 32 + 4 coupling words 32 + write-back 8
CPU_SAMPLE_LOG2N = 22               # oracle sample: same recipe at N = 2^22
METRIC = "spin updates/sec on 1 B200 (VB N=2^24, c=4) and % of HBM roofline"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=8)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--T", type=float, default=1.0)
    ap.add_argument("--model", default="vb", choices=["vb", "sk", "rrbg", "rrg"],
                    help="sk: BASELINE.json configs[3] with --log2n 12 (absolute rate only); rrbg / rrg: the paper's own ensembles "
                         "(SURVEY.md 8(f) rank 1), use --T 1.2149")
    ap.add_argument("--windowed", type=int, default=0, metavar="S",
                    help="also time the windowed protocol: sg_sweep(1) + one sg_corr_accumulate against S stored configurations per sweep")
    ap.add_argument("--clones", type=int, default=1, help="SK: replicas that share the couplings (PAPER.md:233)")
    ap.add_argument("--shard", default="sample", choices=["sample", "site"],
                    help="N > 1: 'sample' = independent replicas per rank (default, no collective); 'site' = ONE instance, every "
                         "colour class split over the ranks with an exchange of the updated slices after each class (PAPER.md:322-324)")
    ap.add_argument("--log2n", type=int, default=24)
    ap.add_argument("--n-words", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--sweeps-per-step", type=int, default=SWEEPS_PER_STEP)
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        sm = sorted(int(float(r[0])) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit())
        mx = [int(float(r[1])) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for q, n in enumerate(names) if any(len(r) >= 7 and r[3 + q].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def dist_setup(n):
    """One process per GPU; RANK/LOCAL_RANK/WORLD_SIZE/MASTER_* come from torchrun."""
    rank, world, local = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))
    return rank, world, local


def cpu_sample(args, sweeps):
    """Time the oracle, as it stands, on one host core: same recipe at N = 2^CPU_SAMPLE_LOG2N."""
    import oracle

    n = 1 << min(CPU_SAMPLE_LOG2N, args.log2n)
    o = oracle.Oracle(oracle.VB, n, 4.0, args.T, 1, args.n_words)
    t0 = time.perf_counter()
    o.sweep(sweeps)
    dt = time.perf_counter() - t0
    return n * 64 * args.n_words * sweeps / dt, dt, n


def cpu_sample_other(model, n, c, T, sweeps, clones=1):
    """The other two samples of BASELINE.md section 3: config 1 in full, the SK instance of config 4 for a few sweeps."""
    import oracle

    o = oracle.Oracle(model, n, c, T, 1, 1, n_clones=clones) if clones > 1 else oracle.Oracle(model, n, c, T, 1, 1)
    t0 = time.perf_counter()
    o.sweep(sweeps)
    dt = time.perf_counter() - t0
    return n * 64 * clones * sweeps / dt, dt


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step = 1 sweep of the N=2^22 sample."""
    rank, world, _ = dist_setup(args.gpus)
    if rank != 0:
        return
    import oracle

    n = 1 << min(CPU_SAMPLE_LOG2N, args.log2n)
    o = oracle.Oracle(oracle.VB, n, 4.0, args.T, 1, args.n_words)
    for _ in range(args.warmup):
        o.sweep(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.sweep(1)
    dt = time.perf_counter() - t0
    val = n * 64 * args.n_words * args.steps / dt
    sample = f"VB c=4 T={args.T} seed 1, same recipe at N=2^{n.bit_length() - 1} (bounded sample), 1 oracle sweep per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "spin updates/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": f"VB N=2^{args.log2n} c=4 W={args.n_words} T={args.T} seed=1 (BASELINE.json configs[2])", "sample": sample},
        "cpu_baseline": {"value": val, "unit": "spin updates/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "spin updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank, world, local = dist_setup(args.gpus)
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_1906_11195_b200 import build as b

    if rank == 0:
        b.build()
    if world > 1:
        dist.barrier()
    import paper_1906_11195_b200 as sg

    N, W = 1 << args.log2n, args.n_words
    t0 = time.perf_counter()
    from paper_1906_11195_b200.workloads import Workload, shard

    model = {"vb": sg.SG_MODEL_VB, "sk": sg.SG_MODEL_SK, "rrbg": sg.SG_MODEL_RRBG, "rrg": sg.SG_MODEL_RRG}[args.model]
    site = args.shard == "site" and world > 1
    wl = Workload("bench", model, N, 4.0, args.T, 1, W, 0) if site else shard(Workload("bench", model, N, 4.0, args.T, 1, W, 0), rank, world)
    sim = sg.Sim(wl.model, wl.N, wl.c, wl.T, wl.seed, wl.n_words, n_clones=args.clones)
    if site:
        from paper_1906_11195_b200.workloads import exchange_on_device, sweep_site_sharded

        exch = exchange_on_device(sim, dist, rank)
    create_s = time.perf_counter() - t0
    counts = np.zeros(sim.lanes, dtype=np.uint64)
    energy = np.zeros(sim.lanes, dtype=np.int64)
    sweep_ev = []

    def step(timed):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        if site:
            sweep_site_sharded(sim, SWEEPS_PER_STEP, rank, world, exch)
        else:
            sim.sweep(SWEEPS_PER_STEP)
        e1.record()
        sim.snapshot(0)
        sim.correlation(0, counts)
        sim.energy(energy)
        if timed:
            sweep_ev.append((e0, e1))

    def sync_all():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(False)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = sg.kernel_launches()
    sync_all()
    s_ev, f_ev = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s_ev.record()
    for _ in range(args.steps):
        step(True)
    f_ev.record()
    sync_all()
    launches = sg.kernel_launches() - l0
    clocks = sampler.stop() if rank == 0 else None
    ms = s_ev.elapsed_time(f_ev)
    sweep_ms = sum(a.elapsed_time(b_) for a, b_ in sweep_ev)
    if world > 1:
        t = torch.tensor([ms, sweep_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, sweep_ms = float(t[0]), float(t[1])
    updates_per_rank = N * sim.lanes * SWEEPS_PER_STEP * args.steps
    value = updates_per_rank * (1 if site else world) / (ms * 1e-3)      # site-sharded: one instance, strong scaling

    # ---- e2e: the same step through the C-ABI with HOST buffers: the configuration goes in from pinned host
    # memory (sg_set_spins) and comes back (sg_get_spins) every step, as in the paper's flow
    e2e = None
    if not args.no_e2e:
        host = torch.empty((N, sim.groups), dtype=torch.int64, pin_memory=True).numpy().view(np.uint64)
        sim.spins(out=host)
        for _ in range(2):
            sim.set_spins(host); step(False); sim.spins(out=host)
        sync_all()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            sim.set_spins(host)
            step(False)
            sim.spins(out=host)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], device="cuda", dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t[0])
        e2e = {"value": updates_per_rank * (1 if site else world) / dt, "unit": "spin updates/s",
               "h2d_bytes_per_step": N * sim.groups * 8, "d2h_bytes_per_step": N * sim.groups * 8 + 2 * sim.lanes * 8,
               "note": "sg_set_spins(pinned host) + step + sg_get_spins(pinned host) per step, wall clock"}
    windowed = None
    if args.windowed > 0:
        # the paper's measurement protocol: after EVERY sweep count against every stored tw;
        # here S stored configurations, the sums kept on the device (sg_corr_accumulate), fetched once at the end
        S = args.windowed
        for k in range(S):
            sim.snapshot(k)
            sim.sweep(1)
        sim.corr_configure(S)
        slots, bins = list(range(S)), list(range(S))
        nsw = 64

        def timed(with_acc):
            sync_all()
            a, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(nsw):
                sim.sweep(1)
                if with_acc:
                    sim.corr_accumulate(slots, bins)
            b_.record()
            sync_all()
            return a.elapsed_time(b_) / nsw

        timed(True)
        t_with, t_without = timed(True), timed(False)
        acc, hits = sim.corr_fetch(0, S)
        assert int(hits[0]) == 3 * nsw - nsw and np.all(acc[0] > 0)
        bytes_per_sweep = (8 + 8 * S) * N * W
        windowed = {"slots": S, "ms_per_sweep_with_accumulate": t_with, "ms_per_sweep_without": t_without,
                    "accumulate_ms_per_sweep": t_with - t_without, "algorithmic_bytes_per_sweep": bytes_per_sweep,
                    "accumulate_gb_per_s": bytes_per_sweep / ((t_with - t_without) * 1e-3) / 1e9,
                    "note": "one asynchronous sg_corr_accumulate per sweep: (8 + 8 S) bytes per site-word in passes of up to 3 slots"}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_src = peaks()
    site_words = N * W * SWEEPS_PER_STEP * args.steps
    achieved = BYTES_PER_SITE_WORD * site_words / (sweep_ms * 1e-3) / 1e9
    out = {
        "metric": METRIC, "value": value, "unit": "spin updates/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if site else "weak",
        "vs_baseline": None, "dtype": "u64", "data": "synthetic",
        "config": {"workload": (f"VB N=2^{args.log2n} c=4 W={W} T={args.T} seed=1+rank (BASELINE.json configs[2])" if args.model == "vb"
                                else f"{args.model.upper()} degree 4 N=2^{args.log2n} W={W} T={args.T} seed=1+rank (the paper's ensemble, PAPER.md:75, :260; not the headline workload)" if args.model in ("rrbg", "rrg")
                                else f"SK N=2^{args.log2n} W={W} T={args.T} seed=1+rank (BASELINE.json configs[3]; dependency-latency bound, roofline fields not meaningful)"),
                   "step": f"sg_sweep({SWEEPS_PER_STEP}) + sg_snapshot + sg_correlation + sg_energy",
                   "l2": "inputs larger than L2: every sweep streams 660 MiB of couplings+indices+labels+headers and reads/writes the 128 MiB spin array (L2 126 MiB); no flush needed",
                   "parallelism": ("one instance sharded by site: per-class NCCL exchange of the updated slices" if site else
                                   "replicas sharded by sample word, no data-path collective") if world > 1 else "single GPU",
                   "create_s": round(create_s, 2)},
        "roofline": {"bound": "hbm", "kernel": "k_vb_sweep (the 6-7 colour-class launches of a sweep)", "achieved": achieved, "peak": peak,
                     "unit": "GB/s", "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                     "bytes_per_site_word": BYTES_PER_SITE_WORD, "sweep_ms": sweep_ms / (SWEEPS_PER_STEP * args.steps),
                     "sweep_share_of_step": sweep_ms / ms},
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
    }
    if windowed:
        out["windowed"] = windowed
    tr = os.path.join(ROOT, "profiles", "traffic.json")
    headline = args.model == "vb" and args.log2n == 24 and W == 1 and args.T == 1.0
    if os.path.exists(tr) and headline:
        # ncu counters of one sweep of exactly this workload, captured once per kernel change and stored under profiles/
        # (a run under ncu is never a bench run): quoted here, not measured in this run
        t = json.load(open(tr))
        out["roofline"]["traffic"] = t.get("dram_bytes_per_sweep")
        out["roofline"]["traffic_source"] = "profiles/traffic.json (ncu --set full capture of this workload, quoted)"
        out["roofline"]["per"] = "sweep (the K colour-class launches): achieved, traffic and sweep_ms are per sweep"
        out["roofline"]["dram_bytes_per_site_word"] = out["roofline"]["traffic"] / (N * W)       # ncu, BASELINE.md section 2
        if t.get("warp_instructions_per_sweep") and clocks and clocks.get("sm_max_mhz"):
            # the ALU ceiling of BASELINE.json: the kernel's whole instruction stream (Philox + bit-sliced arithmetic +
            # addressing) at 4 warp instructions per SM and clock
            issue = 148 * 4 * clocks["sm_max_mhz"] * 1e6
            out["roofline"]["alu_ceiling"] = {"value": N * 64 * W / (t["warp_instructions_per_sweep"] / issue), "unit": "spin updates/s",
                                              "warp_instructions_per_sweep": t["warp_instructions_per_sweep"],
                                              "source": "profiles/traffic.json smsp__inst_executed.sum (quoted); 148 SMs x 4 issue slots x sm_max_mhz"}
    if not headline:
        out["config"]["l2"] = "not the headline workload: see DESIGN.md section 10"
    if args.model == "sk":
        out["roofline"] = {"bound": "latency", "kernel": "k_sk_sweep", "achieved": None, "peak": None, "unit": None, "frac": None, "traffic": None,
                           "note": "sequential sweep of one instance per CTA (PAPER.md:233): dependency-latency bound, absolute rate only",
                           "sweep_ms": sweep_ms / (SWEEPS_PER_STEP * args.steps)}
    if not args.no_cpu_baseline and args.model == "vb":   # the headline ensemble
        v, dt, n = cpu_sample(args, 2)
        out["cpu_baseline"] = {"value": v, "unit": "spin updates/s", "cores": 1, "kind": "oracle", "host_cores": os.cpu_count(),
                               "sample": f"same recipe at N=2^{n.bit_length() - 1}, 2 oracle sweeps, {dt:.1f} s (N=2^24 itself would take "
                                         "about 35 s per sweep plus 40 s of setup on one core: the rate per site does not depend on N)"}
        if headline:                                      # the other two samples of BASELINE.md section 3
            import oracle

            v1, d1 = cpu_sample_other(oracle.VB, 1024, 4.0, 1.0, 1024)
            v4, d4 = cpu_sample_other(oracle.SK, 4096, 0.0, 0.6, 2)
            out["cpu_baseline"]["also"] = [
                {"value": v1, "unit": "spin updates/s", "sample": f"BASELINE.json configs[0] in full: VB N=1024, 1024 sweeps, {d1:.1f} s"},
                {"value": v4, "unit": "spin updates/s", "sample": f"BASELINE.json configs[3]: SK N=4096 T=0.6, 2 sweeps, {d4:.1f} s"}]
    if not args.no_cpu_baseline and args.model == "sk":
        import oracle

        n = 1 << min(12, args.log2n)
        v4, d4 = cpu_sample_other(oracle.SK, n, 0.0, args.T, 2, args.clones)
        out["cpu_baseline"] = {"value": v4, "unit": "spin updates/s", "cores": 1, "kind": "oracle", "host_cores": os.cpu_count(),
                               "sample": f"SK N={n} T={args.T}, {args.clones} clone(s), 2 oracle sweeps, {d4:.1f} s"}
    out["context"] = {"paper": "~15 ps per spin update on one P100 = 6.7e10 spin updates/s (PAPER.md:320); "
                               "total work of the order of 2^64 spin updates (PAPER.md:165)"}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    global SWEEPS_PER_STEP
    args = parse()
    SWEEPS_PER_STEP = args.sweeps_per_step
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
