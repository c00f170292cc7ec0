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
