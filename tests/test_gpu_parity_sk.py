"""GPU parity (Sherrington-Kirkpatrick): CUDA path through the C-ABI vs the oracle, bit for bit."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sg():
    import torch

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1906_11195_b200 import build as b

    b.build()
    import paper_1906_11195_b200 as sg

    return sg


def _same(g, o):
    gs, os_ = g.spins(), o.spins()
    if not np.array_equal(gs, os_):
        bad = np.argwhere(gs != os_)
        raise AssertionError(f"spins differ at {len(bad)} places, first {bad[:5].tolist()}")
    assert g.sweep_count == o.sweep_count


@pytest.mark.parametrize("N,T,seed,W,sweeps", [
    (256, 0.6, 1, 1, 12),
    (100, 0.6, 2, 1, 12),       # N not a multiple of 32
    (33, 1.0, 3, 2, 10),        # two words per site, ragged
    (2, 0.5, 4, 1, 6),
    (512, 0.4, 5, 1, 6),
    (96, 0.0, 6, 1, 10),        # T = 0
    (96, float("inf"), 7, 1, 5),  # T = inf: everything flips
    (320, 50.0, 8, 1, 4),       # hot: thresholds non-zero for every m
    (200, 0.6, 9, 5, 4),        # five words (c1 = w>>2 changes at w = 4)
])
def test_sk_matches_oracle(sg, oracle_mod, N, T, seed, W, sweeps):
    g = sg.Sim(sg.SG_MODEL_SK, N, 0.0, T, seed, W)
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, seed, W)
    assert g.M == o.M == N * (N - 1) // 2
    assert np.array_equal(g.couplings(), o.couplings())
    assert np.array_equal(g.thresholds(N), o.thresholds(N))
    _same(g, o)
    assert np.array_equal(g.energy(), o.energy())
    g.snapshot(0); o.snapshot(0)
    E0 = g.energy()
    Eprev = E0
    for t in range(1, sweeps + 1):
        g.sweep(1); o.sweep(1)
        _same(g, o)
        E = g.energy()
        assert np.array_equal(E, o.energy())
        assert np.array_equal(g.correlation(0), o.correlation(0))
        if T == 0.0:
            assert np.all(E <= Eprev)
        if math.isinf(T):
            assert np.all(g.correlation(0) == (N if t % 2 else 0))
        Eprev = E
    # several sweeps inside one kernel launch == one at a time
    g.sweep(7); o.sweep(7)
    _same(g, o)
    assert np.array_equal(g.energy(), o.energy())


def test_sk_config4_instance_first_sweeps(sg, oracle_mod):
    """BASELINE.json configs[3] instance (N=4096, T=0.6, seed 1): the oracle's from-scratch fields cost
    ~N^2*64 per sweep, so compare the first sweeps in full and then properties."""
    from paper_1906_11195_b200.workloads import CFG4 as w

    g = sg.Sim(w.model, w.N, w.c, w.T, w.seed, w.n_words)
    o = oracle_mod.Oracle(w.model, w.N, w.c, w.T, w.seed, w.n_words)
    _same(g, o)
    g.snapshot(0); o.snapshot(0)
    for _ in range(3):
        g.sweep(1); o.sweep(1)
        _same(g, o)
        assert np.array_equal(g.energy(), o.energy())
        assert np.array_equal(g.correlation(0), o.correlation(0))


def test_sk_pure_function_and_set_spins(sg, oracle_mod):
    N, W = 192, 1
    g = sg.Sim(sg.SG_MODEL_SK, N, 0.0, 0.6, 3, W)
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, 0.6, 3, W)
    rng = np.random.default_rng(1)
    state = rng.integers(0, 1 << 64, size=(N, W), dtype=np.uint64)
    for t in (1000, (1 << 32) + 3):
        for h in (g, o):
            h.set_spins(state)
            h.set_sweep_count(t)
            h.sweep(2)
        _same(g, o)
        assert np.array_equal(g.energy(), o.energy())


def test_sk_long_run_energy_consistency(sg):
    """Incremental int16 fields stay equal to from-scratch fields: energy from the fields equals the
    energy recomputed from couplings and spins on the host after many sweeps."""
    from tests import exact

    N = 256
    g = sg.Sim(sg.SG_MODEL_SK, N, 0.0, 0.6, 11, 1)
    g.sweep(300)
    S = exact.unpack(g.spins())
    K = exact.unpack(g.couplings())
    pr = np.array([[i, j] for i in range(N) for j in range(i + 1, N)])
    E = -(K * S[pr[:, 0]] * S[pr[:, 1]]).sum(axis=0)
    assert np.array_equal(g.energy(), E)


@pytest.mark.parametrize("N,T,seed,W,aligned", [(256, 0.4, 21, 1, True), (100, 0.5, 22, 2, True), (512, 0.6, 23, 1, False)])
def test_sk_protocol_of_the_si(sg, oracle_mod, N, T, seed, W, aligned):
    """two clones per coupling set, all-aligned start, T in {0.4, 0.5, 0.6}, waiting time tw = 3;
    every sweep compared with the oracle, energies and the counts against the tw = 3 snapshot as well."""
    g = sg.Sim(sg.SG_MODEL_SK, N, 0.0, T, seed, W, n_clones=2, aligned_start=aligned)
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, seed, W, n_clones=2, aligned_start=aligned)
    assert g.lanes == o.lanes == 128 * W
    _same(g, o)
    if aligned:
        assert np.all(g.spins() == 0)
    assert np.array_equal(g.couplings(), o.couplings())
    assert np.array_equal(g.energy(), o.energy())
    g.sweep(3); o.sweep(3)
    g.snapshot(0); o.snapshot(0)
    for _ in range(5):
        g.sweep(1); o.sweep(1)
        _same(g, o)
        assert np.array_equal(g.energy(), o.energy())
        assert np.array_equal(g.correlation(0), o.correlation(0))
    # clone 0 is the plain run of the same instance
    p = sg.Sim(sg.SG_MODEL_SK, N, 0.0, T, seed, W, aligned_start=aligned)
    p.sweep(8)
    assert np.array_equal(p.spins(), g.spins()[:, :W])


def test_sk_word_offset(sg, oracle_mod):
    """sg_options.word0: words 4..7 of an 8-word instance from their own handle."""
    N, T = 160, 0.6
    full = sg.Sim(sg.SG_MODEL_SK, N, 0.0, T, 31, 8)
    part = sg.Sim(sg.SG_MODEL_SK, N, 0.0, T, 31, 4, word0=4)
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 31, 4, word0=4)
    full.sweep(4); part.sweep(4); o.sweep(4)
    assert np.array_equal(part.spins(), full.spins()[:, 4:])
    assert np.array_equal(part.spins(), o.spins())
    assert np.array_equal(part.energy(), full.energy()[256:])


def test_two_sk_handles_of_different_size(sg, oracle_mod):
    """The dynamic shared-memory limit of the sweep kernel belongs to the function, not to a handle: creating and
    sweeping a small instance must not break a larger one that needs more than 48 KiB."""
    big = sg.Sim(sg.SG_MODEL_SK, 12000, 0.0, 0.6, 41, 1)
    small = sg.Sim(sg.SG_MODEL_SK, 64, 0.0, 0.6, 42, 1)
    small.sweep(2)
    big.sweep(1)
    small.sweep(1)
    big.sweep(1)
    E = big.energy()
    assert E.shape == (64,) and np.all(E < 0)
    o = oracle_mod.Oracle(oracle_mod.SK, 64, 0.0, 0.6, 42, 1)
    o.sweep(3)
    assert np.array_equal(small.spins(), o.spins())


def test_sk_largest_size(sg, oracle_mod):
    """N = 2^15, the largest size of the paper's SK runs and the limit of int16 local fields (Q22).  The
    GPU runs two sweeps from the aligned start; the oracle (from-scratch fields) replays three windows of the second
    sweep -- its first, a middle and its last 512 site updates -- from the mixed state in which the sites below the
    window carry the GPU's new values and the others its old ones.  Plus: the incremental int16 fields after the sweeps
    equal fields recomputed from scratch (energy before and after re-importing the configuration)."""
    N, T, K = 1 << 15, 0.4, 512
    from concurrent.futures import ThreadPoolExecutor

    with ThreadPoolExecutor(max_workers=2) as ex:
        fo = ex.submit(lambda: oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 51, 1, aligned_start=True))
        fg = ex.submit(lambda: sg.Sim(sg.SG_MODEL_SK, N, 0.0, T, 51, 1, aligned_start=True))
        o, g = fo.result(), fg.result()
    g.sweep(1)
    old = g.spins()
    g.sweep(1)
    new = g.spins()
    assert 0 < int((old != new).sum()) < N
    o.set_sweep_count(1)
    for i0 in (0, N // 2 - 100, N - K):
        mixed = old.copy()
        mixed[:i0] = new[:i0]
        o.set_spins(mixed)
        o.sk_update_range(i0, i0 + K)
        assert np.array_equal(o.spins()[i0:i0 + K], new[i0:i0 + K]), i0
    E = g.energy()
    g.set_spins(new)                       # recomputes every local field from scratch
    assert np.array_equal(g.energy(), E)
    g.sweep(1)                             # and the dynamics goes on from there
    assert g.sweep_count == 3


def test_sk_windowed_tritone_protocol(sg, oracle_mod):
    """SK as the SI measures it: two clones, aligned start, tw = 3, every sweep counted against the tw = 3 snapshot and
    lumped in tritone intervals of tw + t, accumulated on the device."""
    from paper_1906_11195_b200 import workloads as wl

    N, S = 128, 60
    g = sg.Sim(sg.SG_MODEL_SK, N, 0.0, 0.5, 61, 1, n_clones=2, aligned_start=True)
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, 0.5, 61, 1, n_clones=2, aligned_start=True)
    rd = wl.run_windowed_device(g, S, tws=(3,), binning=wl.tritone_index)
    ro = wl.run_windowed(o, S, tws=(3,), binning=wl.tritone_index)
    assert rd.keys() == ro.keys() and len(rd) >= 6
    for k in rd:
        assert rd[k][1] == ro[k][1] and np.array_equal(rd[k][0], ro[k][0]), k
