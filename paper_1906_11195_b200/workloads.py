"""BASELINE.json's configurations as parameter tuples, and the tw,t = 2^k measurement schedule.

Shared by tests/ and bench.py (and by the oracle-side harness): it holds NO arithmetic of the
method -- only which (model, N, c, T, seed, n_words, sweeps) to run and at which sweep counts to
snapshot / correlate (O10).  Every instance is synthetic and follows from these
parameters through the seeded generator each side implements for itself.
"""
from __future__ import annotations

from dataclasses import dataclass

VB, SK, RRBG, RRG = 0, 1, 2, 3


@dataclass(frozen=True)
class Workload:
    name: str
    model: int
    N: int
    c: float
    T: float
    seed: int
    n_words: int
    sweeps: int


# BASELINE.json configs[0..3]
CFG1 = Workload("cfg1_vb_n1024", VB, 1 << 10, 4.0, 1.0, 1, 1, 1 << 10)
CFG2 = Workload("cfg2_vb_n2^20_w4", VB, 1 << 20, 4.0, 1.0, 1, 4, 1 << 14)
CFG3 = [Workload(f"cfg3_vb_n2^24_T{T}", VB, 1 << 24, 4.0, T, 1, 1, 1 << 12) for T in (0.6, 1.0, 1.4)]
CFG4 = Workload("cfg4_sk_n4096", SK, 1 << 12, 0.0, 0.6, 1, 1, 1 << 12)


# The paper's own workload: RRBG degree 4, T = 0.8 Tc = 0.8 / atanh(1/sqrt(3))
T_PAPER = 0.8 / 0.6584789484624083      # atanh(1/sqrt(3)) = 0.658478948...
PAPER_RRBG = Workload("paper_rrbg_n2^24", RRBG, 1 << 24, 0.0, T_PAPER, 1, 1, 1 << 12)


def cfg5():
    """BASELINE.json configs[4]: the aging protocol sweep (Q17/Q18)."""
    out = []
    for log2n, w, sweeps in ((12, 16, 1 << 16), (16, 16, 1 << 16), (20, 4, 1 << 16), (24, 1, 1 << 12), (26, 1, 1 << 12)):
        for ti, T in enumerate((0.6, 1.0, 1.4)):
            out.append(Workload(f"cfg5_vb_n2^{log2n}_T{T}", VB, 1 << log2n, 4.0, T, 1000 * log2n + ti, w, sweeps))
    return out


def schedule(total_sweeps: int):
    """Events of the tw,t = 2^k protocol in time order (O10).

    Yields (time, kind, slot) with kind 'snap' (slot a <- s(2^a)) or 'corr' (count against slot a at
    time 2^a + 2^b).  Snapshots sort before correlations at equal times.
    """
    ev = []
    a = 0
    while (1 << a) <= total_sweeps:
        ev.append((1 << a, 0, a))
        b = 0
        while (1 << a) + (1 << b) <= total_sweeps:
            ev.append(((1 << a) + (1 << b), 1, a))
            b += 1
        a += 1
    ev.sort()
    return [(t, "snap" if k == 0 else "corr", s) for (t, k, s) in ev]


def run_schedule(sim, total_sweeps: int):
    """Drive any object with sweep/snapshot/correlation (the binding's Sim or the oracle's handle).

    Returns {(tw, t): counts array}."""
    out = {}
    now = 0
    for time, kind, slot in schedule(total_sweeps):
        if time > now:
            sim.sweep(time - now)
            now = time
        if kind == "snap":
            sim.snapshot(slot)
        else:
            out[(1 << slot, time - (1 << slot))] = sim.correlation(slot).copy()
    if now < total_sweeps:
        sim.sweep(total_sweeps - now)
    return out


def shard(w: Workload, rank: int, world: int) -> Workload:
    """The replica rank `rank` of `world` runs: the path shards by sample, so every rank gets its
    own n_words*64 samples of the same recipe (seed + rank); there is no data-path collective."""
    if not 0 <= rank < world:
        raise ValueError("rank out of range")
    return Workload(f"{w.name}_r{rank}of{world}", w.model, w.N, w.c, w.T, w.seed + rank, w.n_words, w.sweeps)


def global_lane(w: Workload, rank: int, lane: int) -> int:
    """Index of a rank's lane in the job-wide, rank-major list of samples."""
    return rank * 64 * w.n_words + lane


# ---- windowed protocol ---------------------------------------------------------
def window_index(time: int) -> int:
    """Index m of the minor-third logarithmic interval (t_m, t_{m+1}], t_m = 2^(m/4), that contains the integer time
    ("minor thirds logarithmic intervals tw + t in [t_m, t_{m+1}], with t_{m+1}/t_m = 2^{1/4}").
    Integer-exact: m = ceil(4 log2 time) - 1 for time >= 2, found by comparing time^4 with 2^m; time 1 -> m = -1."""
    if time < 1:
        raise ValueError("time must be >= 1")
    t4 = time ** 4
    m = t4.bit_length() - 1                  # 2^m <= time^4 < 2^(m+1)
    return m - 1 if t4 == 1 << m else m      # time^4 in (2^m, 2^(m+1)]  <=>  time in (t_m, t_{m+1}]


def tritone_index(time: int) -> int:
    """Index of the tritone lump of the total time tw + t (data with the same value of
    floor(ln((t + tw)/4) / (0.5 ln 2)) are lumped together, e.g. tw + t = {4, 5}).  Integer-exact:
    floor(2 log2(time/4)) = floor(log2(time^2)) - 4."""
    if time < 1:
        raise ValueError("time must be >= 1")
    return (time * time).bit_length() - 1 - 4


def run_windowed_device(sim, total_sweeps: int, tws=(4, 16, 64, 256, 1024, 4096), binning=window_index):
    """The windowed protocol with the bookkeeping on the device (sg_corr_configure / _accumulate / _fetch): after every
    sweep ONE asynchronous call adds D against every stored tw to that tw's current bin; the host fetches once at the
    end.  Same result as run_windowed (the reference harness, which works on any object with sweep/snapshot/correlation):
    {(tw, m): (sum of D per lane, number of times)}."""
    tws = [tw for tw in tws if tw <= total_sweeps]
    slot_of = {tw: k for k, tw in enumerate(tws)}
    m0 = binning(1)
    nb = binning(total_sweeps) - m0 + 1                     # bins per tw
    sim.corr_configure(max(1, nb * len(tws)))
    for time in range(1, total_sweeps + 1):
        sim.sweep(1)
        active = [tw for tw in tws if time > tw]
        if active:
            sim.corr_accumulate([slot_of[tw] for tw in active], [slot_of[tw] * nb + binning(time) - m0 for tw in active])
        if time in slot_of:
            sim.snapshot(slot_of[time])
    acc, hits = sim.corr_fetch(0, max(1, nb * len(tws)))
    out = {}
    for tw in tws:
        for b in range(nb):
            q = slot_of[tw] * nb + b
            if hits[q]:
                out[(tw, b + m0)] = (acc[q].copy(), int(hits[q]))
    return out


def run_windowed(sim, total_sweeps: int, tws=(4, 16, 64, 256, 1024, 4096), binning=window_index):
    """The paper's measurement protocol on any object with sweep/snapshot/correlation (the binding's Sim or the oracle's
    handle): snapshot at every waiting time tw (tw = 2^2, 2^4, ..., 2^12), then after EVERY sweep count D
    against every stored tw and add it to the bin of the total time tw + t (window_index).  Returns
    {(tw, m): (sum of D over the bin as uint64 per lane, number of times in the bin)}: the caller's window average is
    C = 1 - 2 * sumD / (n * N).  Exact integers; no arithmetic of the method is done here."""
    import numpy as np

    tws = [tw for tw in tws if tw <= total_sweeps]
    slot_of = {tw: k for k, tw in enumerate(tws)}
    out = {}
    for time in range(1, total_sweeps + 1):
        sim.sweep(1)
        for tw in tws:
            if time > tw:
                key = (tw, binning(time))
                d = np.asarray(sim.correlation(slot_of[tw]), dtype=np.uint64)
                if key in out:
                    out[key] = (out[key][0] + d, out[key][1] + 1)
                else:
                    out[key] = (d.copy(), 1)
        if time in slot_of:
            sim.snapshot(slot_of[time])
    return out


# ---- site-sharded sweeps over several ranks -------------------------------------
def split_units(n_units: int, rank: int, world: int):
    """Units [a, b) of a class that rank `rank` of `world` updates: contiguous, balanced to within one unit."""
    if not 0 <= rank < world:
        raise ValueError("rank out of range")
    return n_units * rank // world, n_units * (rank + 1) // world


def sweep_site_sharded(backend, n_sweeps: int, rank: int, world: int, exchange):
    """The paper's multi-GPU scheme on any backend with n_colours, class_units(k), sweep_part(k, unit0, n),
    end_sweep() (the binding's Sim on a GPU, or tests' oracle backend): every rank holds the full configuration; for
    each colour class in order a rank updates its own units, then `exchange(k, parts)` -- parts[r] = (unit0, n) of every
    rank -- makes every rank's copy of the class current before the next class starts.  No arithmetic of the method
    here.  The result on every rank equals backend.sweep(n_sweeps) on one rank, bit for bit."""
    for _ in range(n_sweeps):
        for k in range(backend.n_colours):
            units = backend.class_units(k)
            parts = []
            for r in range(world):
                a, b = split_units(units, r, world)
                parts.append((a, b - a))
            backend.sweep_part(k, *parts[rank])
            if world > 1:
                exchange(k, parts)
        backend.end_sweep()


def exchange_through_host(backend, dist, rank: int):
    """exchange() for sweep_site_sharded with host buffers and torch.distributed broadcasts (any backend, gloo or nccl)."""
    import numpy as np
    import torch

    def exchange(k, parts):
        for r, (u0, n) in enumerate(parts):
            if n == 0:
                continue
            if r == rank:
                buf = torch.from_numpy(backend.export_part(k, u0, n).view(np.int64).copy())
            else:
                buf = torch.empty(backend.part_range(k, u0, n)[1], dtype=torch.int64)
            dist.broadcast(buf, src=r)
            if r != rank:
                backend.import_part(k, u0, n, buf.numpy().view(np.uint64))

    return exchange


def exchange_on_device(sim, dist, rank: int):
    """exchange() for the binding's Sim on GPUs: NCCL broadcasts of each rank's contiguous range of the device spin array,
    in place (NVLink / NVSwitch), on torch's current stream -- the stream the library launches on, so the next class's
    kernels are ordered after the exchange."""
    spins = sim.spin_tensor()

    def exchange(k, parts):
        works = []
        for r, (u0, n) in enumerate(parts):
            if n == 0:
                continue
            first, count = sim.part_range(k, u0, n)
            works.append(dist.broadcast(spins[first:first + count], src=r, async_op=True))
        for w in works:
            w.wait()

    return exchange
