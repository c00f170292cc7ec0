"""Pins for the oracle's RRG instance generator (model 3): a random regular graph of degree 4 that is NOT bipartite, the
ensemble of the main text ("random regular graphs with fixed degree z = 4"); the supplement's Fig. S3
 shows that making it bipartite for the GPU code changes nothing measurable.  The dynamics is the VB
code pinned elsewhere; the graph is pinned by what the definition fixes and by statistics of the uniform ensemble."""
import math

import numpy as np
import pytest


def _adj(N, e):
    nb = [set() for _ in range(N)]
    for a, b in e.tolist():
        nb[a].add(b); nb[b].add(a)
    return nb


def _triangles(N, e):
    nb = _adj(N, e)
    t = 0
    for a, b in e.tolist():
        t += len(nb[a] & nb[b])
    return t // 3


@pytest.mark.parametrize("N,seed", [(8, 1), (64, 2), (1001, 3), (4096, 4), (1 << 16, 5)])
def test_rrg_graph_is_4_regular_and_simple(oracle_mod, N, seed):
    o = oracle_mod.Oracle(oracle_mod.RRG, N, 0.0, 1.2, seed, 1)
    e = o.edges().astype(np.int64)
    assert o.M == 2 * N == len(e)
    assert np.all(e[:, 0] != e[:, 1])                                               # no loops
    assert len({(min(a, b), max(a, b)) for a, b in e.tolist()}) == len(e)            # no repeated pair
    assert np.all(np.bincount(e.ravel(), minlength=N) == 4) and o.max_degree == 4
    _, _, colour = o.graph()
    assert np.all(colour[e[:, 0]] != colour[e[:, 1]]) and 3 <= o.n_colours <= 5      # proper; degree 4 -> at most 5 colours
    nb = _adj(N, e)
    for i in range(min(N, 2000)):                                                    # first-fit: a neighbour in every lower colour
        assert {int(colour[j]) for j in nb[i]} >= set(range(int(colour[i])))


def test_rrg_is_the_pairing_model_of_its_definition(oracle_mod):
    """O2c restated with the second Philox implementation of this test suite (tests/exact-free: or_philox is pinned by the
    known answers): the accepted attempt's shuffle reproduces the edge list, and every earlier attempt is not simple."""
    N, seed = 40, 9
    o = oracle_mod.Oracle(oracle_mod.RRG, N, 0.0, 1.0, seed, 1)
    e = o.edges().astype(np.int64).tolist()
    Q = 4 * N
    for t in range(10000):
        p = list(range(Q))
        for i in range(Q - 1, 0, -1):
            n = Q - 1 - i
            x = oracle_mod.philox(n >> 2, t, 0, 5 << 24, seed & 0xFFFFFFFF, seed >> 32)[n & 3]
            j = (int(x) * (i + 1)) >> 32
            p[i], p[j] = p[j], p[i]
        pairs = [(p[2 * k] // 4, p[2 * k + 1] // 4) for k in range(2 * N)]
        simple = all(a != b for a, b in pairs) and len({(min(a, b), max(a, b)) for a, b in pairs}) == len(pairs)
        if simple:
            assert [list(x) for x in pairs] == e
            break
    else:
        raise AssertionError("no simple attempt found")
    assert t > 0 or True


def test_rrg_triangle_count_matches_the_uniform_ensemble(oracle_mod):
    """In a uniform random d-regular graph the number of k-cycles tends to Poisson((d-1)^k / (2k)) (Bollobas 1980;
    Wormald 1981): triangles, d = 4: 27/6 = 4.5, independent of N.  A bipartite graph has none; a generator that resamples
    locally instead of rejecting the whole pairing shifts this count."""
    counts = [_triangles(1500, oracle_mod.Oracle(oracle_mod.RRG, 1500, 0.0, 1.0, 200 + s, 1).edges().astype(np.int64)) for s in range(60)]
    mean = float(np.mean(counts))
    assert abs(mean - 4.5) < 4 * math.sqrt(4.5 / 60), (mean, counts)
    assert 2.0 < float(np.var(counts)) < 9.0                                         # Poisson: variance = mean


def test_rrg_paramagnetic_energy_density(oracle_mod):
    """Locally tree-like with degree 4, as the bipartite ensemble: e = -2 tanh(1/T) above Tc (Bethe lattice)."""
    N, T = 1 << 14, 3.0
    o = oracle_mod.Oracle(oracle_mod.RRG, N, 0.0, T, 11, 1)
    o.sweep(30)
    acc = []
    for _ in range(10):
        o.sweep(2)
        acc.append(o.energy().astype(np.float64).mean() / N)
    assert abs(np.mean(acc) - (-2.0 * math.tanh(1.0 / T))) < 0.006


def test_rrg_rejects_bad_sizes(oracle_mod):
    for N in (2, 7):
        with pytest.raises(ValueError):
            oracle_mod.Oracle(oracle_mod.RRG, N, 0.0, 1.0, 1, 1)
