"""Exact statistical mechanics of tiny +-J Ising systems, for pinning the oracle.

Independent of oracle/ and of the CUDA path: plain numpy on all 2^N states.
State index x: bit i of x = 1 <=> s_i = -1 (the spin-bit convention, Q14).
"""
from __future__ import annotations

import numpy as np


def all_states(N: int) -> np.ndarray:
    """(2^N, N) array of +-1 spins; row x has s_i = -1 iff bit i of x is set."""
    x = np.arange(1 << N, dtype=np.int64)[:, None]
    bits = (x >> np.arange(N, dtype=np.int64)[None, :]) & 1
    return (1 - 2 * bits).astype(np.int64)


def energies(N: int, edges: np.ndarray, J: np.ndarray) -> np.ndarray:
    """E(x) = -sum_e J_e s_u s_v for every state (PAPER.md:73 Eq. 3; :43 Eq. 1 with integer J)."""
    S = all_states(N)
    E = np.zeros(1 << N, dtype=np.float64)
    for (u, v), j in zip(edges, J):
        E -= j * S[:, u] * S[:, v]
    return E


def boltzmann(E: np.ndarray, beta: float) -> np.ndarray:
    w = np.exp(-beta * (E - E.min()))
    return w / w.sum()


def exact_averages(N, edges, J, beta):
    """<E>, matrix <s_i s_j>."""
    S = all_states(N)
    E = energies(N, edges, J)
    pi = boltzmann(E, beta)
    corr = (S * pi[:, None]).T @ S
    return float((pi * E).sum()), corr


def single_site_matrix(N, edges, J, beta, i, accept=None) -> np.ndarray:
    """Metropolis transition matrix of one update of site i.

    accept(dE) -> acceptance probability; default min(1, exp(-beta dE)).
    """
    E = energies(N, edges, J)
    n = 1 << N
    P = np.zeros((n, n))
    for x in range(n):
        y = x ^ (1 << i)
        dE = E[y] - E[x]
        a = (1.0 if dE <= 0 else float(np.exp(-beta * dE))) if accept is None else accept(dE)
        P[x, y] = a
        P[x, x] = 1.0 - a
    return P


def sweep_matrix(N, edges, J, beta, order, accept=None) -> np.ndarray:
    """Product of single-site matrices in the given site order (row-vector convention)."""
    P = np.eye(1 << N)
    for i in order:
        P = P @ single_site_matrix(N, edges, J, beta, i, accept)
    return P


def first_fit_colouring(N, edges) -> np.ndarray:
    """Smallest colour not used by an already coloured neighbour, natural order (O5)."""
    nbr = [[] for _ in range(N)]
    for u, v in edges:
        nbr[int(u)].append(int(v))
        nbr[int(v)].append(int(u))
    col = -np.ones(N, dtype=np.int64)
    for i in range(N):
        used = {col[j] for j in nbr[i] if col[j] >= 0}
        c = 0
        while c in used:
            c += 1
        col[i] = c
    return col


def colour_order(colour: np.ndarray) -> list[int]:
    """Site order of one sweep: colour classes ascending, sites ascending inside a class (O7)."""
    return [int(i) for k in range(int(colour.max()) + 1) for i in np.nonzero(colour == k)[0]]


def unpack(words: np.ndarray) -> np.ndarray:
    """(N, W) uint64 -> (N, 64W) +-1 int64; bit 1 <=> -1."""
    words = np.asarray(words, dtype=np.uint64)
    N, W = words.shape
    b = (words[:, :, None] >> np.arange(64, dtype=np.uint64)[None, None, :]) & np.uint64(1)
    return (1 - 2 * b.astype(np.int64)).reshape(N, 64 * W)


def pack_state_per_lane(N: int, states: np.ndarray) -> np.ndarray:
    """states: (64,) state indices, one per lane -> (N,1) uint64 spin words."""
    out = np.zeros((N, 1), dtype=np.uint64)
    for lane, x in enumerate(states):
        for i in range(N):
            if (int(x) >> i) & 1:
                out[i, 0] |= np.uint64(1) << np.uint64(lane)
    return out


def state_index_per_lane(words: np.ndarray) -> np.ndarray:
    """(N, W) uint64 -> (64W,) state index per lane."""
    S = unpack(words)  # (N, L)
    N = S.shape[0]
    bits = (S < 0).astype(np.int64)
    return (bits * (1 << np.arange(N, dtype=np.int64))[:, None]).sum(axis=0)
