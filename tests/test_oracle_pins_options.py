"""Pins of the oracle's options (oracle/sg_oracle.c header: word0, clones, aligned; Q24-Q26).

P15a  word offset: words share only the graph, so a W-word run IS W one-word runs started at
      word0 = 0 .. W-1 -- spins, energies and correlation counts, for VB, RRBG and SK.
P15b  clones ("replicas with the same couplings"): clone 0 is the plain run; clone 1 has the same
      couplings (equal energies on equal configurations) but its own initial spins and its own uniforms.
P15c  aligned start: every spin +1 at t = 0, E'(0) = -sum_{i<j} J'_ij; "gauge-equivalent to a random
      start": the energy after a few sweeps has the same distribution over samples for both starts.
"""
import numpy as np
import pytest

from tests import exact


@pytest.mark.parametrize("model,N,c,T", [(0, 700, 4.0, 1.0), (2, 512, 0.0, 1.2149), (1, 48, 0.0, 0.6)])
def test_word_offset_splits_a_run_exactly(oracle_mod, model, N, c, T):
    W = 5
    full = oracle_mod.Oracle(model, N, c, T, 7, W)
    parts = [oracle_mod.Oracle(model, N, c, T, 7, 1, word0=w) for w in range(W)]
    full.snapshot(0)
    for p in parts:
        p.snapshot(0)
    for _ in range(3):
        full.sweep(2)
        S, E, D = full.spins(), full.energy(), full.correlation(0)
        for w, p in enumerate(parts):
            p.sweep(2)
            assert np.array_equal(p.spins()[:, 0], S[:, w])
            assert np.array_equal(p.energy(), E[64 * w:64 * w + 64])
            assert np.array_equal(p.correlation(0), D[64 * w:64 * w + 64])
    # a two-word handle in the middle
    mid = oracle_mod.Oracle(model, N, c, T, 7, 2, word0=2)
    mid.sweep(6)
    assert np.array_equal(mid.spins(), full.spins()[:, 2:4])
    assert np.array_equal(full.couplings()[:, 2:4], mid.couplings())


def test_clones_share_couplings_only(oracle_mod):
    N, T, W = 40, 0.6, 2
    one = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 11, W)
    two = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 11, W, n_clones=2)
    assert two.lanes == 2 * one.lanes and two.spins().shape == (N, 2 * W)
    assert np.array_equal(two.couplings(), one.couplings())
    s0 = two.spins()
    assert np.array_equal(s0[:, :W], one.spins())                  # clone 0 = the plain run
    assert not np.array_equal(s0[:, W:], s0[:, :W])                # clone 1 starts elsewhere
    frac = exact.unpack(s0[:, W:]).mean()
    assert abs(frac) < 5 / np.sqrt(N * 64 * W)                     # ... from fair bits
    one.sweep(3); two.sweep(3)
    assert np.array_equal(two.spins()[:, :W], one.spins())
    assert np.array_equal(two.energy()[:64 * W], one.energy())
    # same couplings: equal configurations have equal energies in both clones
    rng = np.random.default_rng(3)
    cfg = rng.integers(0, 1 << 64, size=(N, W), dtype=np.uint64)
    two.set_spins(np.concatenate([cfg, cfg], axis=1))
    E = two.energy()
    assert np.array_equal(E[:64 * W], E[64 * W:])
    # own uniforms: from equal configurations the two clones part ways
    two.sweep(1)
    s1 = two.spins()
    assert not np.array_equal(s1[:, :W], s1[:, W:])
    with pytest.raises(ValueError):
        oracle_mod.Oracle(oracle_mod.VB, 100, 4.0, 1.0, 1, 1, n_clones=2)


def test_aligned_start(oracle_mod):
    N, T = 32, 0.5
    a = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 5, 4, n_clones=2, aligned_start=True)
    assert np.all(a.spins() == 0)                                  # every spin +1
    J = exact.unpack(a.couplings())                                # (pairs, lanes) +-1
    E0 = a.energy()
    assert np.array_equal(E0[:256], -J.sum(axis=0)) and np.array_equal(E0[256:], E0[:256])
    v = oracle_mod.Oracle(oracle_mod.VB, 300, 4.0, 1.0, 5, 1, aligned_start=True)
    assert np.all(v.spins() == 0)
    assert np.array_equal(v.energy(), -exact.unpack(v.couplings()).sum(axis=0))
    # gauge equivalence: same energy distribution a few sweeps after either start
    r = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 5, 4, n_clones=2)
    a.sweep(6); r.sweep(6)
    Ea, Er = a.energy().astype(float), r.energy().astype(float)
    z = (Ea.mean() - Er.mean()) / np.sqrt(Ea.var() / Ea.size + Er.var() / Er.size)
    assert abs(z) < 4.5, z
    # the two clones of the aligned run differ only through their uniforms, and they do differ
    s = a.spins()
    assert not np.array_equal(s[:, :4], s[:, 4:])
