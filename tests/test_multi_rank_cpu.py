"""N > 1 path on CPU (gloo, world size 2): the job shards by sample -- every rank runs its own replica (seed + rank)
with no data-path collective; only the timing (MAX over ranks) and, for the caller's convenience, the per-lane results
are exchanged.  The replicas here are driven with the oracle (tests may use it); the GPU runs the same host logic."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist

    import oracle
    from paper_1906_11195_b200.workloads import CFG1, global_lane, run_schedule, shard

    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = shard(CFG1, rank, world)
    assert w.seed == CFG1.seed + rank
    o = oracle.Oracle(w.model, w.N, w.c, w.T, w.seed, w.n_words)
    counts = run_schedule(o, 64)
    mine = np.stack([counts[k] for k in sorted(counts)]).astype(np.int64)            # (pairs, lanes)
    # per-lane results, rank-major: gathered for the caller, never reduced (samples are independent)
    gathered = [torch.zeros(mine.shape, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(mine))
    # timing: max over ranks
    t = torch.tensor([10.0 + rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    assert float(t) == 10.0 + world - 1
    dist.barrier()
    if rank == 0:
        alll = np.concatenate([g.numpy() for g in gathered], axis=1)
        assert alll.shape[1] == world * 64 * w.n_words
        assert global_lane(w, 1, 3) == 64 * w.n_words + 3
        np.save(os.path.join(out_dir, "all.npy"), alll)
    dist.destroy_process_group()


def test_two_ranks_shard_by_sample(tmp_path, oracle_mod):
    import torch.multiprocessing as mp

    from paper_1906_11195_b200.workloads import CFG1, run_schedule, shard

    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    got = np.load(os.path.join(str(tmp_path), "all.npy"))
    # the job's result equals the independent single-process runs of each replica, side by side
    for rank in range(world):
        w = shard(CFG1, rank, world)
        o = oracle_mod.Oracle(w.model, w.N, w.c, w.T, w.seed, w.n_words)
        counts = run_schedule(o, 64)
        ref = np.stack([counts[k] for k in sorted(counts)]).astype(np.int64)
        assert np.array_equal(got[:, rank * 64:(rank + 1) * 64], ref)
    # different seeds give different samples
    assert not np.array_equal(got[:, :64], got[:, 64:])


def test_shard_rejects_bad_rank():
    from paper_1906_11195_b200.workloads import CFG1, shard

    with pytest.raises(ValueError):
        shard(CFG1, 2, 2)


# ---- site-sharded sweeps ---------------------------------------------------------
class OracleSiteBackend:
    """The backend interface of workloads.sweep_site_sharded on top of the oracle: a unit is a run of UNIT consecutive
    members (label order) of a colour class; a part is exchanged as the spin words of its sites."""

    UNIT = 7

    def __init__(self, o):
        self.o = o
        _, _, colour = o.graph()
        self.n_colours = o.n_colours
        self.members = [np.nonzero(colour == k)[0].astype(np.uint32) for k in range(o.n_colours)]

    def class_units(self, k):
        return (len(self.members[k]) + self.UNIT - 1) // self.UNIT

    def _sites(self, k, unit0, n):
        return self.members[k][unit0 * self.UNIT:(unit0 + n) * self.UNIT]

    def sweep_part(self, k, unit0, n):
        self.o.vb_update_sites(self._sites(k, unit0, n))

    def end_sweep(self):
        self.o.set_sweep_count(self.o.sweep_count + 1)

    def part_range(self, k, unit0, n):
        return 0, len(self._sites(k, unit0, n)) * self.o.W

    def export_part(self, k, unit0, n):
        return np.ascontiguousarray(self.o.spins()[self._sites(k, unit0, n)]).ravel()

    def import_part(self, k, unit0, n, words):
        s = self.o.spins()
        s[self._sites(k, unit0, n)] = np.asarray(words, dtype=np.uint64).reshape(-1, self.o.W)
        self.o.set_spins(s)


def _site_worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist

    import oracle
    from paper_1906_11195_b200.workloads import exchange_through_host, sweep_site_sharded

    dist.init_process_group("gloo", rank=rank, world_size=world)
    o = oracle.Oracle(oracle.VB, 900, 4.0, 1.0, 5, 2)          # every rank builds the same instance
    be = OracleSiteBackend(o)
    sweep_site_sharded(be, 3, rank, world, exchange_through_host(be, dist, rank))
    assert o.sweep_count == 3
    np.save(os.path.join(out_dir, f"site_{rank}.npy"), o.spins())
    dist.barrier()
    dist.destroy_process_group()


def test_site_sharded_sweep_equals_the_single_rank_run(tmp_path, oracle_mod):
    """Two ranks (gloo), each with a full copy of the spins, update their own units of every colour class and exchange
    them before the next class: both end with exactly the configuration of the single-rank run."""
    import torch.multiprocessing as mp

    world, port = 2, _free_port()
    mp.spawn(_site_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    ref = oracle_mod.Oracle(oracle_mod.VB, 900, 4.0, 1.0, 5, 2)
    ref.sweep(3)
    for rank in range(world):
        assert np.array_equal(np.load(os.path.join(str(tmp_path), f"site_{rank}.npy")), ref.spins()), rank


def test_site_sharded_harness_single_rank_and_partition(oracle_mod):
    from paper_1906_11195_b200.workloads import split_units, sweep_site_sharded

    for n in (0, 1, 5, 64, 1001):
        for world in (1, 2, 3, 8):
            parts = [split_units(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            assert max(b - a for a, b in parts) - min(b - a for a, b in parts) <= 1
    o = oracle_mod.Oracle(oracle_mod.VB, 500, 4.0, 0.6, 6, 1)
    ref = oracle_mod.Oracle(oracle_mod.VB, 500, 4.0, 0.6, 6, 1)
    sweep_site_sharded(OracleSiteBackend(o), 4, 0, 1, None)
    ref.sweep(4)
    assert np.array_equal(o.spins(), ref.spins()) and o.sweep_count == 4
    # emulated ranks in one process: each "rank" updates its units on the shared state = the same composition
    o2 = oracle_mod.Oracle(oracle_mod.VB, 500, 4.0, 0.6, 6, 1)
    be = OracleSiteBackend(o2)
    for _ in range(4):
        for k in range(be.n_colours):
            for r in (2, 0, 1):                                   # any rank order: the units of a class are independent
                a, b = split_units(be.class_units(k), r, 3)
                be.sweep_part(k, a, b - a)
        be.end_sweep()
    assert np.array_equal(o2.spins(), ref.spins())
