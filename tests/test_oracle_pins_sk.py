"""Pin P13: the SK oracle (Eq. 1 with binary couplings) at small N."""
import math

import numpy as np
import pytest

from tests import exact


def _pairs(N):
    return np.array([[i, j] for i in range(N) for j in range(i + 1, N)])


def test_sk_couplings_layout_and_fairness(oracle_mod):
    N = 64
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, 0.6, 1, 1)
    assert o.M == N * (N - 1) // 2
    K = exact.unpack(o.couplings())
    assert abs((K < 0).mean() - 0.5) < 5 * 0.5 / math.sqrt(K.size)
    # O3: kappa_ij = x0 | x1<<32 of P(c0=j, c1=w, sweep-field=i, tag 2)
    pr = _pairs(N)
    for q in (0, 1, 63, 64, 1000, len(pr) - 1):
        i, j = pr[q]
        x = oracle_mod.philox(int(j), 0, int(i), 2 << 24, 1, 0)
        assert int(o.couplings()[q, 0]) == int(x[0]) | (int(x[1]) << 32)


def test_sk_long_run_matches_boltzmann(oracle_mod):
    N, T = 8, 1.2
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 17, 1)
    pr = _pairs(N)
    Jl = exact.unpack(o.couplings())                   # (pairs, 64)
    beta_eff = 1.0 / (T * math.sqrt(N))                # E = E'/sqrt(N)
    nsw, burn = 20000, 100
    o.sweep(burn)
    Es = np.zeros((nsw, 64))
    C01 = np.zeros((nsw, 64))
    for t in range(nsw):
        o.sweep(1)
        S = exact.unpack(o.spins())
        Es[t] = -(Jl * S[pr[:, 0]] * S[pr[:, 1]]).sum(axis=0)
        C01[t] = S[0] * S[5]
    z = []
    for lane in range(0, 64, 4):
        Eex, corr = exact.exact_averages(N, pr, Jl[:, lane], beta_eff)
        for series, ex in ((Es[:, lane], Eex), (C01[:, lane], corr[0, 5])):
            b = series.reshape(40, -1).mean(axis=1)
            z.append((b.mean() - ex) / (b.std(ddof=1) / math.sqrt(40)))
    z = np.array(z)
    assert np.abs(z).max() < 5.0, z
    assert (z**2).mean() < 1.9


def test_sk_sweep_matrix_leaves_boltzmann_invariant(oracle_mod):
    N, T = 6, 0.9
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 4, 1)
    thr = o.thresholds(N).astype(np.float64)
    pr = _pairs(N)
    J = exact.unpack(o.couplings())[:, 11]
    beta_eff = 1.0 / (T * math.sqrt(N))
    E = exact.energies(N, pr, J)                       # integer numerator E'
    pi = exact.boltzmann(E, beta_eff)

    def accept(dE):                                    # dE' = 2m
        m = int(round(dE / 2))
        return 1.0 if m <= 0 else thr[m] / 2.0**32

    for m in range(1, N):
        assert int(thr[m]) == math.floor(math.exp(-(2.0 * m) / (T * math.sqrt(float(N)))) * 2.0**32)
    Ps = exact.sweep_matrix(N, pr, J, beta_eff, list(range(N)), accept)
    assert np.abs(pi @ Ps - pi).max() < 1e-8


@pytest.mark.parametrize("T", [0.0, 0.6, float("inf")])
def test_sk_energy_bookkeeping(oracle_mod, T):
    N = 96
    o = oracle_mod.Oracle(oracle_mod.SK, N, 0.0, T, 3, 1)
    pr = _pairs(N)
    Jl = exact.unpack(o.couplings())
    E0 = o.energy()
    Eprev = E0
    o.snapshot(0)
    for t in range(1, 7):
        o.sweep(1)
        E = o.energy()
        S = exact.unpack(o.spins())
        assert np.array_equal(E, -(Jl * S[pr[:, 0]] * S[pr[:, 1]]).sum(axis=0))
        assert np.array_equal(E, E0 + o.accumulated_dE())
        # E' = -1/2 sum_i s_i H_i with H_i = sum_{j != i} J'_ij s_j
        for lane in (0, 37):
            Jm = np.zeros((N, N), dtype=np.int64)
            Jm[pr[:, 0], pr[:, 1]] = Jl[:, lane]
            Jm = Jm + Jm.T
            H = Jm @ S[:, lane]
            assert -(S[:, lane] * H).sum() // 2 == E[lane]
        if T == 0.0:
            assert np.all(E <= Eprev)
        if math.isinf(T):
            assert np.all(o.correlation(0) == (N if t % 2 else 0))
        Eprev = E


def test_sk_sweep_is_the_ordered_composition_of_site_updates(oracle_mod):
    """PAPER.md:233 "N single spin updates, performed in a fixed order": or_sk_update_range (used by the GPU tests to
    check windows of the N = 2^15 sweep) composes to or_sweep."""
    a = oracle_mod.Oracle(oracle_mod.SK, 64, 0.0, 0.6, 3, 2)
    b = oracle_mod.Oracle(oracle_mod.SK, 64, 0.0, 0.6, 3, 2)
    for t in range(3):
        a.sweep(1)
        b.sk_update_range(0, 20); b.sk_update_range(20, 21); b.sk_update_range(21, 64)
        b.set_sweep_count(t + 1)
        assert np.array_equal(a.spins(), b.spins())
    c = oracle_mod.Oracle(oracle_mod.SK, 64, 0.0, 0.6, 3, 2)
    c.sk_update_range(10, 30)                       # a different order is a different map
    c.sk_update_range(0, 10); c.sk_update_range(30, 64)
    a2 = oracle_mod.Oracle(oracle_mod.SK, 64, 0.0, 0.6, 3, 2)
    a2.sweep(1)
    assert not np.array_equal(a2.spins(), c.spins())
