"""Pins P2-P9, P12: the oracle's dynamics against what the definitions fix.

(a) exact Boltzmann averages, N <= 12, T = 2        BASELINE.json north_star (a)
(b) detailed balance on the full transition matrix   north_star (b)
(c) C(tw,tw) = 1                                     north_star (c)
(d) energy from scratch == accumulated Delta E       north_star (d)
(e) T = 0 never raises the energy                    north_star (e)
(f) T = inf: every proposal accepted (Q21) north_star (f)
"""
import math

import numpy as np
import pytest

from tests import exact

# a fixed small graph with a triangle (frustration possible), a square, a pendant and an isolated site
EDGES10 = np.array([[0, 1], [1, 2], [2, 0], [2, 3], [3, 4], [4, 5], [5, 6], [6, 3], [6, 7], [7, 8], [1, 8], [0, 5]])
N10 = 10  # site 9 is isolated


def _rand_words(rng, n, w=1):
    return rng.integers(0, 1 << 64, size=(n, w), dtype=np.uint64)


# ---------------------------------------------------------------- P2: the enumeration helper itself
def test_enumeration_helper_closed_forms():
    beta = 0.7
    # forest (a path 0-1-2-3 plus a branch 1-4) with mixed signs:
    edges = np.array([[0, 1], [1, 2], [2, 3], [1, 4]])
    J = np.array([1, -1, 1, -1])
    E, corr = exact.exact_averages(5, edges, J, beta)
    t = math.tanh(beta)
    assert abs(E - (-4 * t)) < 1e-12                      # <E> = -M tanh(beta)
    assert abs(corr[0, 3] - (1 * -1 * 1) * t**3) < 1e-12  # product of J tanh along the path
    assert abs(corr[4, 2] - (-1 * -1) * t**2) < 1e-12
    # single triangle: Z = 2e^{3b}+6e^{-b} (unfrustrated) / 6e^{b}+2e^{-3b} (frustrated)
    tri = np.array([[0, 1], [1, 2], [2, 0]])
    for J, Z in [([1, 1, 1], 2 * math.exp(3 * beta) + 6 * math.exp(-beta)),
                 ([1, 1, -1], 6 * math.exp(beta) + 2 * math.exp(-3 * beta))]:
        En = exact.energies(3, tri, np.array(J))
        assert abs(np.exp(-beta * En).sum() - Z) < 1e-9


# ---------------------------------------------------------------- P3: long run vs Boltzmann
def _batch_means(x, nb=40):
    n = (len(x) // nb) * nb
    b = x[:n].reshape(nb, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nb)


def test_vb_long_run_matches_boltzmann(oracle_mod):
    T, beta = 2.0, 0.5
    rng = np.random.default_rng(123)
    kappa = _rand_words(rng, len(EDGES10))
    sigma = _rand_words(rng, N10)
    o = oracle_mod.Oracle.explicit(N10, EDGES10, kappa, sigma, T, seed=77)
    Jl = exact.unpack(kappa)                                   # (M, 64) +-1
    nsw, burn = 24000, 200
    o.sweep(burn)
    Es = np.zeros((nsw, 64))
    pairs = [(0, 1), (2, 3), (0, 4), (7, 8), (3, 9)]
    Cs = np.zeros((nsw, len(pairs), 64))
    for t in range(nsw):
        o.sweep(1)
        S = exact.unpack(o.spins())                            # (N, 64)
        Es[t] = -(Jl * S[EDGES10[:, 0]] * S[EDGES10[:, 1]]).sum(axis=0)
        for q, (i, j) in enumerate(pairs):
            Cs[t, q] = S[i] * S[j]
    z = []
    for lane in range(0, 64, 3):
        Eex, corr = exact.exact_averages(N10, EDGES10, Jl[:, lane], beta)
        m, se = _batch_means(Es[:, lane])
        z.append((m - Eex) / se)
        for q, (i, j) in enumerate(pairs):
            m, se = _batch_means(Cs[:, q, lane])
            z.append((m - corr[i, j]) / max(se, 1e-12))
    z = np.array(z)
    assert np.abs(z).max() < 5.0, z
    assert (z**2).mean() < 1.8, (z**2).mean()                  # no systematic bias across lanes
    # the isolated site 9 flips every sweep at any T (P9): <s_3 s_9> exact value is 0
    S0 = exact.unpack(o.spins())[9]
    o.sweep(1)
    assert np.array_equal(exact.unpack(o.spins())[9], -S0)


# ---------------------------------------------------------------- P4: transition matrix
def test_detailed_balance_with_integer_thresholds(oracle_mod):
    N, T = 8, 1.7
    edges = np.array([[0, 1], [1, 2], [2, 0], [2, 3], [3, 4], [4, 5], [5, 3], [5, 6], [6, 7], [7, 0], [1, 4], [2, 6]])
    J = np.array([1, -1, 1, 1, -1, -1, 1, 1, -1, 1, -1, 1])
    kappa = np.where(J < 0, np.uint64(0xFFFFFFFFFFFFFFFF), np.uint64(0)).reshape(-1, 1)
    o = oracle_mod.Oracle.explicit(N, edges, kappa, np.zeros((N, 1), dtype=np.uint64), T)
    thr = o.thresholds(o.max_degree + 1).astype(np.float64)
    E = exact.energies(N, edges, J)
    pi = exact.boltzmann(E, 1 / T)

    def accept(dE):           # the oracle's integer rule: Delta E = 2k, accept w.p. thr[k]/2^32
        k = int(round(dE / 2))
        return 1.0 if k <= 0 else thr[k] / 2.0**32

    for i in range(N):
        Pi = exact.single_site_matrix(N, edges, J, 1 / T, i, accept)
        flux = pi[:, None] * Pi
        assert np.abs(flux - flux.T).max() <= pi.max() * 2.0**-32 * 1.001
        assert np.allclose(Pi.sum(axis=1), 1.0)
    # the sweep (product in colour order) leaves pi invariant although it is not reversible
    colour = exact.first_fit_colouring(N, edges)
    Ps = exact.sweep_matrix(N, edges, J, 1 / T, exact.colour_order(colour), accept)
    assert np.abs(pi @ Ps - pi).max() < 1e-8
    flux = pi[:, None] * Ps
    assert np.abs(flux - flux.T).max() > 1e-4


def test_one_sweep_transition_frequencies(oracle_mod):
    """Empirical x -> y frequencies of one oracle sweep vs the exact sweep matrix (N=6, all 64 starts).

    Lane b of every word starts in state b; words and sweep indices give independent uniforms."""
    N, T, W = 6, 1.5, 8
    edges = np.array([[0, 1], [1, 2], [2, 0], [2, 3], [3, 4], [4, 5], [5, 0], [1, 4]])
    J = np.array([1, 1, -1, -1, 1, -1, 1, 1])
    kappa = np.repeat(np.where(J < 0, np.uint64(0xFFFFFFFFFFFFFFFF), np.uint64(0)).reshape(-1, 1), W, axis=1)
    start = np.repeat(exact.pack_state_per_lane(N, np.arange(64)), W, axis=1)
    o = oracle_mod.Oracle.explicit(N, edges, kappa, start, T, seed=5, n_words=W)
    colour = exact.first_fit_colouring(N, edges)
    _, _, ocol = o.graph()
    assert np.array_equal(ocol.astype(np.int64), colour)
    Ps = exact.sweep_matrix(N, edges, J, 1 / T, exact.colour_order(colour))
    counts = np.zeros((64, 64))
    reps = 1500
    for t in range(reps):
        o.set_spins(start)
        o.set_sweep_count(1000 + 7 * t)
        o.sweep(1)
        y = exact.state_index_per_lane(o.spins()).reshape(W, 64)
        for w in range(W):
            counts[np.arange(64), y[w]] += 1
    n = reps * W
    exp = n * Ps
    # impossible transitions never happen
    assert np.all(counts[Ps == 0] == 0)
    big = exp > 8
    zz = (counts[big] - exp[big]) / np.sqrt(exp[big] * (1 - Ps[big]))
    assert np.abs(zz).max() < 5.5, np.abs(zz).max()
    # lanes of a word share their uniforms, so the 638 entries are strongly correlated: mean z^2
    # scatters by about +-0.35 around 1 and does not grow with the sample size (a bias would)
    assert 0.35 < (zz**2).mean() < 1.9, (zz**2).mean()


# ---------------------------------------------------------------- P5: correlation
def test_correlation_properties(oracle_mod):
    o = oracle_mod.Oracle(oracle_mod.VB, 777, 4.0, 1.0, 3, 2)
    o.sweep(3)
    o.snapshot(0)
    assert np.all(o.correlation(0) == 0)                       # C(tw,tw) = 1
    A = o.spins()
    o.sweep(5)
    B = o.spins()
    D = o.correlation(0)
    assert np.all(D <= o.N)
    assert np.array_equal(D, (exact.unpack(A) != exact.unpack(B)).sum(axis=0))
    # symmetric in its two arguments
    o.snapshot(1)
    o.set_spins(A)
    assert np.array_equal(o.correlation(1), D)
    with pytest.raises(RuntimeError):
        o.correlation(7)                                       # never written


# ---------------------------------------------------------------- P6 / P7 / P8
@pytest.mark.parametrize("T", [0.0, 0.6, 1.0, 1.4, 5.0, float("inf")])
def test_energy_bookkeeping_every_sweep(oracle_mod, T):
    o = oracle_mod.Oracle(oracle_mod.VB, 600, 4.0, T, 21, 1)
    E0 = o.energy()
    assert np.all((E0 - o.M) % 2 == 0)                         # E = 2U - M
    Eprev = E0
    edges = o.edges()
    Jl = exact.unpack(o.couplings())
    for _ in range(12):
        o.sweep(1)
        E = o.energy()
        assert np.array_equal(E, E0 + o.accumulated_dE())
        # energy from an independent numpy statement of Eq. 3
        S = exact.unpack(o.spins())
        assert np.array_equal(E, -(Jl * S[edges[:, 0]] * S[edges[:, 1]]).sum(axis=0))
        if T == 0.0:
            assert np.all(E <= Eprev)
        if math.isinf(T):
            assert np.array_equal(E, E0)                       # global flip leaves E unchanged
        Eprev = E


def test_T_infinity_alternation(oracle_mod):
    o = oracle_mod.Oracle(oracle_mod.VB, 300, 4.0, float("inf"), 2, 1)
    o.snapshot(0)
    S0 = o.spins()
    for t in range(1, 6):
        o.sweep(1)
        assert np.all(o.last_flips() == o.N)
        D = o.correlation(0)
        assert np.all(D == (o.N if t % 2 else 0))              # C(0,t) = (-1)^t exactly
    o.sweep(1)
    assert np.array_equal(o.spins(), S0)


def test_T_zero_reaches_single_flip_stable_or_zero_dE_moves(oracle_mod):
    o = oracle_mod.Oracle(oracle_mod.VB, 400, 4.0, 0.0, 8, 1)
    o.sweep(200)
    E1 = o.energy()
    o.sweep(1)
    # only Delta E = 0 moves (and isolated sites) survive at T = 0 after relaxation
    assert np.array_equal(o.energy(), E1)


def test_high_T_unflipped_sites_equal_rejections(oracle_mod):
    # at large finite T, sites that did not flip in a sweep = rejected proposals
    o = oracle_mod.Oracle(oracle_mod.VB, 2000, 4.0, 50.0, 6, 1)
    o.snapshot(0)
    o.sweep(1)
    D = o.correlation(0)
    assert np.array_equal(D, o.last_flips())                   # each site proposed once per sweep
    rej = o.N - D.astype(np.int64)
    # expected rejection fraction: E[1-exp(-2k/T)] over kk>0, small but non-zero
    assert rej.min() > 0 and rej.max() < 0.12 * o.N


# ---------------------------------------------------------------- P9: forced cases
def test_forced_flips_and_forced_rejections(oracle_mod):
    # star: centre 0 with 5 leaves; lanes chosen so that all bonds of the centre are unsatisfied
    N = 6
    edges = np.array([[0, j] for j in range(1, 6)])
    kappa = np.zeros((5, 1), dtype=np.uint64)                  # J=+1 everywhere
    sigma = np.zeros((N, 1), dtype=np.uint64)
    sigma[0, 0] = np.uint64(0x00000000FFFFFFFF)                # lanes 0..31: centre = -1, leaves +1 (all unsatisfied)
    o = oracle_mod.Oracle.explicit(N, edges, kappa, sigma, 0.0, seed=3)
    # colour 0 = centre (site 0): updated first.  T=0: lanes 0..31 flip (dE=-10), lanes 32..63 stay (dE=+10)
    o.sweep(1)
    S = o.spins()
    assert int(S[0, 0]) == 0
    assert np.all(S[1:, 0] == 0)                               # leaves see a satisfied bond: no flip at T=0
    assert np.array_equal(o.accumulated_dE(), np.r_[np.full(32, -10), np.zeros(32)].astype(np.int64))


def test_sweep_composition(oracle_mod):
    a = oracle_mod.Oracle(oracle_mod.VB, 500, 4.0, 1.0, 9, 1)
    b = oracle_mod.Oracle(oracle_mod.VB, 500, 4.0, 1.0, 9, 1)
    a.sweep(3)
    a.sweep(4)
    b.sweep(7)
    assert np.array_equal(a.spins(), b.spins()) and a.sweep_count == b.sweep_count == 7
    # different seeds / temperatures differ
    c = oracle_mod.Oracle(oracle_mod.VB, 500, 4.0, 1.0, 10, 1)
    c.sweep(7)
    assert not np.array_equal(a.spins(), c.spins())


# ---------------------------------------------------------------- P12: paramagnet on a tree-like graph
@pytest.mark.parametrize("T,target", [(3.0, -0.6430), (2.5, -0.7599)])
def test_paramagnetic_energy_density(oracle_mod, T, target):
    # e = -(c/2) tanh(1/T) for c=4 on a locally tree-like graph, T > Tc = 1.82
    assert abs(-2 * math.tanh(1 / T) - target) < 1e-4
    N = 1 << 14
    o = oracle_mod.Oracle(oracle_mod.VB, N, 4.0, T, 31, 1)
    o.sweep(25)
    es = []
    for _ in range(6):
        o.sweep(3)
        es.append(o.energy().mean() / N)
    assert abs(np.mean(es) - target) < 0.006, np.mean(es)
