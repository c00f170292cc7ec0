"""ctypes loader for the CPU oracle (oracle/sg_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
holds no arithmetic of its own: every number comes out of sg_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sg_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

VB, SK, RRBG, RRG = 0, 1, 2, 3   # RRG: random regular graph of degree 4, not bipartite; RRBG: the VB Hamiltonian on a random regular bipartite graph of degree 4
MAX_SLOTS = 64


def build(force: bool = False) -> str:
    """Compile sg_oracle.c with gcc (-O2, no threading, no intrinsics)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", _LIB, _SRC, "-lm"]
        )
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        u64, u32, i32, dbl, vp = C.c_uint64, C.c_uint32, C.c_int32, C.c_double, C.c_void_p
        L.or_philox.argtypes = [u32] * 6 + [vp]
        L.or_philox.restype = None
        L.or_create.argtypes = [C.c_int, u64, dbl, dbl, u64, u32]
        L.or_create.restype = vp
        L.or_create_opt.argtypes = [C.c_int, u64, dbl, dbl, u64, u32, u32, u32, C.c_int]
        L.or_create_opt.restype = vp
        L.or_create_explicit.argtypes = [u64, u64, vp, vp, vp, vp, dbl, u64, u32]
        L.or_create_explicit.restype = vp
        L.or_destroy.argtypes = [vp]
        L.or_destroy.restype = None
        L.or_sweep.argtypes = [vp, u64]
        L.or_sk_update_range.argtypes = [vp, u64, u64]
        L.or_vb_update_sites.argtypes = [vp, vp, u64]
        L.or_snapshot.argtypes = [vp, u32]
        L.or_correlation.argtypes = [vp, u32, vp]
        L.or_energy.argtypes = [vp, vp]
        for name in ("or_sweep_count", "or_num_edges"):
            getattr(L, name).argtypes = [vp]
            getattr(L, name).restype = u64
        for name in ("or_num_colours", "or_max_degree"):
            getattr(L, name).argtypes = [vp]
            getattr(L, name).restype = u32
        L.or_get_spins.argtypes = [vp, i32, vp]
        L.or_set_spins.argtypes = [vp, vp]
        L.or_set_sweep_count.argtypes = [vp, u64]
        L.or_set_sweep_count.restype = None
        L.or_get_graph.argtypes = [vp, vp, vp, vp]
        L.or_get_edges.argtypes = [vp, vp, vp]
        L.or_get_couplings.argtypes = [vp, vp]
        L.or_get_thresholds.argtypes = [vp, vp, u64]
        L.or_get_accumulated_dE.argtypes = [vp, vp]
        L.or_get_last_flips.argtypes = [vp, vp]
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def philox(c0, c1, c2, c3, k0, k1) -> np.ndarray:
    out = np.zeros(4, dtype=np.uint32)
    lib().or_philox(c0, c1, c2, c3, k0, k1, _p(out))
    return out


class Oracle:
    """Thin handle around or_sim*.  Mirrors the sg_* call names."""

    def __init__(self, model: int, N: int, c: float, T: float, seed: int, n_words: int, _handle=None,
                 word0: int = 0, n_clones: int = 1, aligned_start: bool = False):
        self._L = lib()
        self.model, self.N, self.c, self.T, self.seed, self.W = model, int(N), c, T, seed, int(n_words)
        self.word0, self.n_clones, self.aligned_start = int(word0), int(n_clones), bool(aligned_start)
        self._h = _handle if _handle is not None else self._L.or_create_opt(model, N, c, T, seed, n_words, self.word0,
                                                                           self.n_clones, int(self.aligned_start))
        if not self._h:
            raise ValueError("or_create rejected the arguments")
        self.lanes = 64 * self.W * self.n_clones

    @classmethod
    def explicit(cls, N, edges, kappa, sigma, T, seed=0, n_words=1):
        """edges: (M,2) ints; kappa: (M,W) uint64; sigma: (N,W) uint64."""
        L = lib()
        edges = np.asarray(edges, dtype=np.uint32).reshape(-1, 2)
        M = edges.shape[0]
        u = np.ascontiguousarray(edges[:, 0])
        v = np.ascontiguousarray(edges[:, 1])
        kappa = np.ascontiguousarray(np.asarray(kappa, dtype=np.uint64).reshape(M, n_words))
        sigma = np.ascontiguousarray(np.asarray(sigma, dtype=np.uint64).reshape(N, n_words))
        h = L.or_create_explicit(N, M, _p(u), _p(v), _p(kappa), _p(sigma), T, seed, n_words)
        if not h:
            raise ValueError("or_create_explicit rejected the arguments")
        return cls(VB, N, 0.0, T, seed, n_words, _handle=h)

    def close(self):
        if self._h:
            self._L.or_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- the five calls
    def sweep(self, n: int = 1):
        rc = self._L.or_sweep(self._h, n)
        assert rc == 0

    def vb_update_sites(self, sites):
        sites = np.ascontiguousarray(np.asarray(sites, dtype=np.uint32))
        rc = self._L.or_vb_update_sites(self._h, _p(sites), sites.size)
        assert rc == 0

    def sk_update_range(self, i0: int, i1: int):
        rc = self._L.or_sk_update_range(self._h, i0, i1)
        assert rc == 0

    def snapshot(self, slot: int):
        rc = self._L.or_snapshot(self._h, slot)
        if rc != 0:
            raise RuntimeError(f"or_snapshot -> {rc}")

    def correlation(self, slot: int) -> np.ndarray:
        out = np.zeros(self.lanes, dtype=np.uint64)
        rc = self._L.or_correlation(self._h, slot, _p(out))
        if rc != 0:
            raise RuntimeError(f"or_correlation -> {rc}")
        return out

    def energy(self) -> np.ndarray:
        out = np.zeros(self.lanes, dtype=np.int64)
        rc = self._L.or_energy(self._h, _p(out))
        assert rc == 0
        return out

    # --- getters
    @property
    def sweep_count(self) -> int:
        return self._L.or_sweep_count(self._h)

    @property
    def M(self) -> int:
        return self._L.or_num_edges(self._h)

    @property
    def n_colours(self) -> int:
        return self._L.or_num_colours(self._h)

    @property
    def max_degree(self) -> int:
        return self._L.or_max_degree(self._h)

    def spins(self, slot: int = -1) -> np.ndarray:
        out = np.zeros((self.N, self.W * self.n_clones), dtype=np.uint64)
        rc = self._L.or_get_spins(self._h, slot, _p(out))
        if rc != 0:
            raise RuntimeError(f"or_get_spins -> {rc}")
        return out

    def set_spins(self, words: np.ndarray):
        words = np.ascontiguousarray(np.asarray(words, dtype=np.uint64).reshape(self.N, self.W * self.n_clones))
        self._L.or_set_spins(self._h, _p(words))

    def set_sweep_count(self, t: int):
        self._L.or_set_sweep_count(self._h, t)

    def graph(self):
        row_ptr = np.zeros(self.N + 1, dtype=np.uint64)
        col = np.zeros(2 * self.M, dtype=np.uint32)
        colour = np.zeros(self.N, dtype=np.uint32)
        rc = self._L.or_get_graph(self._h, _p(row_ptr), _p(col), _p(colour))
        assert rc == 0
        return row_ptr, col, colour

    def edges(self) -> np.ndarray:
        u = np.zeros(self.M, dtype=np.uint32)
        v = np.zeros(self.M, dtype=np.uint32)
        rc = self._L.or_get_edges(self._h, _p(u), _p(v))
        assert rc == 0
        return np.stack([u, v], axis=1)

    def couplings(self) -> np.ndarray:
        out = np.zeros((self.M, self.W), dtype=np.uint64)
        self._L.or_get_couplings(self._h, _p(out))
        return out

    def thresholds(self, n: int) -> np.ndarray:
        out = np.zeros(n, dtype=np.uint64)
        self._L.or_get_thresholds(self._h, _p(out), n)
        return out

    def accumulated_dE(self) -> np.ndarray:
        out = np.zeros(self.lanes, dtype=np.int64)
        self._L.or_get_accumulated_dE(self._h, _p(out))
        return out

    def last_flips(self) -> np.ndarray:
        out = np.zeros(self.lanes, dtype=np.uint64)
        self._L.or_get_last_flips(self._h, _p(out))
        return out
