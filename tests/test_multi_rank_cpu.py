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
