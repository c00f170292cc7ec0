"""Pins for the oracle's RRBG instance generator (model 2): the paper's own ensemble, a random regular bipartite graph
of degree 4 ("each spin interact with a fixed number (4) of other spins and ... all of them are
in the same half of the lattice").  The dynamics on it is the VB code already pinned by test_oracle_pins_dynamics.py;
what is new is the graph, pinned here by what the definition fixes and by a statistic of the ensemble."""
import math

import numpy as np
import pytest


@pytest.mark.parametrize("N,seed", [(8, 1), (64, 2), (1000, 3), (4096, 4), (1 << 16, 5)])
def test_rrbg_graph_is_4_regular_bipartite_simple(oracle_mod, N, seed):
    o = oracle_mod.Oracle(oracle_mod.RRBG, N, 0.0, 1.2, seed, 1)
    H = N // 2
    e = o.edges().astype(np.int64)
    assert o.M == 2 * N == len(e)
    # every edge joins half A (labels < N/2) to half B; edge a*H + i leaves vertex i
    assert np.all(e[:, 0] < H) and np.all(e[:, 1] >= H)
    assert np.array_equal(e[:, 0], np.tile(np.arange(H), 4))
    # each of the four blocks is a permutation of half B; no pair is repeated
    for a in range(4):
        assert np.array_equal(np.sort(e[a * H:(a + 1) * H, 1]), np.arange(H, N))
    assert len({(int(a), int(b)) for a, b in e}) == len(e)
    deg = np.bincount(e.ravel(), minlength=N)
    assert np.all(deg == 4) and o.max_degree == 4
    # first-fit colouring in label order = the bipartition: two classes, "two halves"
    _, _, colour = o.graph()
    assert o.n_colours == 2
    assert np.all(colour[:H] == 0) and np.all(colour[H:] == 1)


def test_rrbg_rejects_bad_sizes(oracle_mod):
    for N in (2, 6, 7, 1001):
        with pytest.raises(ValueError):
            oracle_mod.Oracle(oracle_mod.RRBG, N, 0.0, 1.0, 1, 1)


def test_rrbg_seeds_differ_and_are_reproducible(oracle_mod):
    a = oracle_mod.Oracle(oracle_mod.RRBG, 512, 0.0, 1.0, 7, 1)
    b = oracle_mod.Oracle(oracle_mod.RRBG, 512, 0.0, 1.0, 7, 1)
    c = oracle_mod.Oracle(oracle_mod.RRBG, 512, 0.0, 1.0, 8, 1)
    assert np.array_equal(a.edges(), b.edges()) and not np.array_equal(a.edges(), c.edges())
    assert np.array_equal(a.spins(), b.spins()) and np.array_equal(a.couplings(), b.couplings())


def test_rrbg_four_cycle_count_matches_the_ensemble(oracle_mod):
    """In a random (d1, d2)-biregular bipartite graph the number of cycles of length 2k tends to a Poisson variable of
    mean ((d1-1)(d2-1))^k / (2k) (Bollobas; Wormald's survey of random regular graphs): for degree 4 and k = 2,
    9^2 / 4 = 20.25, independent of N.  Counted by brute force over pairs of A-vertices with two common neighbours; a
    generator that kept repeated pairs, or was not uniform over matchings, misses this."""
    counts = []
    for seed in range(40):
        o = oracle_mod.Oracle(oracle_mod.RRBG, 2048, 0.0, 1.0, 100 + seed, 1)
        e = o.edges().astype(np.int64)
        H = 1024
        nbrs = [[] for _ in range(H)]
        for a, b in e:
            nbrs[a].append(b)
        byb = {}
        for a in range(H):
            for b in nbrs[a]:
                byb.setdefault(b, []).append(a)
        pair_common = {}
        for b, lst in byb.items():
            for x in range(len(lst)):
                for y in range(x + 1, len(lst)):
                    k = (lst[x], lst[y])
                    pair_common[k] = pair_common.get(k, 0) + 1
        counts.append(sum(c * (c - 1) // 2 for c in pair_common.values()))
    mean = float(np.mean(counts))
    # Poisson(20.25): standard error of the mean of 40 draws = sqrt(20.25/40) = 0.71; O(1/N) corrections are below that
    assert abs(mean - 20.25) < 4 * math.sqrt(20.25 / 40), (mean, counts)


def test_rrbg_paramagnetic_energy_density(oracle_mod):
    """Locally tree-like with degree 4: above Tc = 1/atanh(1/sqrt 3) = 1.5187 the equilibrium energy per site is
    -(z/2) tanh(1/T) (Bethe lattice), reached within a few tens of sweeps.  T = 3: -0.6430."""
    N, T = 1 << 14, 3.0
    o = oracle_mod.Oracle(oracle_mod.RRBG, N, 0.0, T, 11, 1)
    o.sweep(30)
    acc = []
    for _ in range(10):
        o.sweep(2)
        acc.append(o.energy().astype(np.float64).mean() / N)
    assert abs(np.mean(acc) - (-2.0 * math.tanh(1.0 / T))) < 0.006
