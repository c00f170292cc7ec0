"""ctypes binding for libsg.so (include/sg.h).  Same names as the C calls; argument marshalling only.

There is no CPU fallback: if the library has not been built or no CUDA device is present the calls fail.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

SG_MODEL_VB, SG_MODEL_SK, SG_MODEL_RRBG, SG_MODEL_RRG = 0, 1, 2, 3
SG_OK, SG_EINVAL, SG_ENOMEM, SG_ECUDA, SG_ESLOT = 0, -1, -2, -3, -4
SG_MAX_SLOTS = 64

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SG_LIBSG_PATH") or os.path.join(_HERE, "libsg.so")   # the override serves A/B measurements of builds

# every symbol include/sg.h declares: (name, restype, argtypes)
_u64, _u32, _i32, _dbl, _vp = C.c_uint64, C.c_uint32, C.c_int32, C.c_double, C.c_void_p
SYMBOLS = {
    "sg_create": (_vp, [C.c_int, _u64, _dbl, _dbl, _u64, _u32]),
    "sg_create_opt": (_vp, [C.c_int, _u64, _dbl, _dbl, _u64, _u32, _vp]),
    "sg_num_lanes": (_u64, [_vp]),
    "sg_destroy": (None, [_vp]),
    "sg_sweep": (C.c_int, [_vp, _u64]),
    "sg_snapshot": (C.c_int, [_vp, _u32]),
    "sg_correlation": (C.c_int, [_vp, _u32, _vp]),
    "sg_correlation_noalloc": (C.c_int, [_vp, _u32, _vp]),
    "sg_noalloc_max_words": (_u32, []),
    "sg_energy": (C.c_int, [_vp, _vp]),
    "sg_corr_configure": (C.c_int, [_vp, _u32]),
    "sg_corr_accumulate": (C.c_int, [_vp, _u32, _vp, _vp]),
    "sg_corr_fetch": (C.c_int, [_vp, _u32, _u32, _vp, _vp]),
    "sg_class_units": (C.c_int, [_vp, _u32, _vp]),
    "sg_sweep_part": (C.c_int, [_vp, _u32, _u64, _u64]),
    "sg_end_sweep": (C.c_int, [_vp]),
    "sg_part_range": (C.c_int, [_vp, _u32, _u64, _u64, _vp, _vp]),
    "sg_spin_device_pointer": (C.c_int, [_vp, _vp]),
    "sg_export_part": (C.c_int, [_vp, _u64, _u64, _vp]),
    "sg_import_part": (C.c_int, [_vp, _u64, _u64, _vp]),
    "sg_last_error": (C.c_char_p, []),
    "sg_sweep_count": (_u64, [_vp]),
    "sg_num_edges": (_u64, [_vp]),
    "sg_num_colours": (_u32, [_vp]),
    "sg_max_degree": (_u32, [_vp]),
    "sg_get_spins": (C.c_int, [_vp, _i32, _vp]),
    "sg_set_spins": (C.c_int, [_vp, _vp]),
    "sg_set_sweep_count": (C.c_int, [_vp, _u64]),
    "sg_get_graph": (C.c_int, [_vp, _vp, _vp, _vp]),
    "sg_get_edges": (C.c_int, [_vp, _vp, _vp]),
    "sg_get_couplings": (C.c_int, [_vp, _vp]),
    "sg_get_thresholds": (C.c_int, [_vp, _vp, _u64]),
    "sg_kernel_launches": (_u64, []),
    "sg_host_philox": (None, [_u32] * 6 + [_vp]),
    "sg_host_graph_create": (_vp, [C.c_int, _u64, _dbl, _u64, _u32]),
    "sg_host_graph_destroy": (None, [_vp]),
    "sg_host_graph_info": (C.c_int, [_vp, _vp]),
    "sg_host_graph_get": (C.c_int, [_vp] * 19),
}


class SGError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"sg error {code}: {msg}")
        self.code = code


_lib = None


def load_library() -> C.CDLL:
    """Load libsg.so (after torch, whose libc10_cuda provides the allocator and the stream)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1906_11195_b200.build` "
                "(there is no CPU fallback)")
        import torch  # noqa: F401  (loads libc10 / libc10_cuda with RTLD_GLOBAL semantics needed by the glue)

        lib = C.CDLL(LIB_PATH, mode=C.RTLD_GLOBAL)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _err() -> str:
    return (load_library().sg_last_error() or b"").decode()


def _check(rc: int):
    if rc != SG_OK:
        raise SGError(rc, _err())


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


# ---- the five calls, C names --------------------------------------------------------------------
def sg_create(model: int, N: int, c: float, T: float, seed: int, n_words: int) -> int:
    import torch

    if torch.cuda.is_available():
        torch.cuda.init()   # the library takes memory from torch's caching allocator and its current stream
    h = load_library().sg_create(int(model), int(N), float(c), float(T), int(seed), int(n_words))
    if not h:
        raise SGError(SG_EINVAL, _err())
    return h


class sg_options(C.Structure):
    _fields_ = [("word0", _u32), ("n_clones", _u32), ("aligned_start", _u32), ("reserved", _u32)]


def sg_create_opt(model: int, N: int, c: float, T: float, seed: int, n_words: int, word0: int = 0, n_clones: int = 1,
                  aligned_start: bool = False) -> int:
    import torch

    if torch.cuda.is_available():
        torch.cuda.init()
    opt = sg_options(int(word0), int(n_clones), 1 if aligned_start else 0, 0)
    h = load_library().sg_create_opt(int(model), int(N), float(c), float(T), int(seed), int(n_words), C.byref(opt))
    if not h:
        raise SGError(SG_EINVAL, _err())
    return h


def sg_destroy(h: int) -> None:
    load_library().sg_destroy(h)


def sg_sweep(h: int, n: int) -> None:
    _check(load_library().sg_sweep(h, int(n)))


def sg_snapshot(h: int, slot: int) -> None:
    _check(load_library().sg_snapshot(h, int(slot)))


def sg_correlation(h: int, slot: int, out_counts: np.ndarray) -> np.ndarray:
    assert out_counts.dtype == np.uint64 and out_counts.flags.c_contiguous
    _check(load_library().sg_correlation(h, int(slot), _ptr(out_counts)))
    return out_counts


def sg_correlation_noalloc(h: int, slot: int, out_counts: np.ndarray) -> np.ndarray:
    assert out_counts.dtype == np.uint64 and out_counts.flags.c_contiguous
    _check(load_library().sg_correlation_noalloc(h, int(slot), _ptr(out_counts)))
    return out_counts


def sg_noalloc_max_words() -> int:
    return int(load_library().sg_noalloc_max_words())


def sg_energy(h: int, out: np.ndarray) -> np.ndarray:
    assert out.dtype == np.int64 and out.flags.c_contiguous
    _check(load_library().sg_energy(h, _ptr(out)))
    return out


def kernel_launches() -> int:
    return load_library().sg_kernel_launches()


# ---- convenience handle -------------------------------------------------------------------------
class Sim:
    """Owns one sg_sim*.  Methods mirror the C calls one to one."""

    def __init__(self, model: int, N: int, c: float, T: float, seed: int, n_words: int, word0: int = 0, n_clones: int = 1,
                 aligned_start: bool = False):
        self._L = load_library()
        self.model, self.N, self.c, self.T, self.seed, self.W = model, int(N), float(c), float(T), int(seed), int(n_words)
        self.word0, self.n_clones, self.aligned_start = int(word0), int(n_clones), bool(aligned_start)
        self.groups = self.W * self.n_clones          # 64-lane groups per site
        self.lanes = 64 * self.groups
        if word0 == 0 and n_clones == 1 and not aligned_start:
            self._h = sg_create(model, N, c, T, seed, n_words)
        else:
            self._h = sg_create_opt(model, N, c, T, seed, n_words, word0, n_clones, aligned_start)
        assert self._L.sg_num_lanes(self._h) == self.lanes

    def close(self):
        if getattr(self, "_h", None):
            sg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def sweep(self, n: int = 1):
        sg_sweep(self._h, n)

    def snapshot(self, slot: int):
        sg_snapshot(self._h, slot)

    def correlation(self, slot: int, out: np.ndarray | None = None) -> np.ndarray:
        out = np.zeros(self.lanes, dtype=np.uint64) if out is None else out
        return sg_correlation(self._h, slot, out)

    def correlation_noalloc(self, slot: int, out: np.ndarray | None = None) -> np.ndarray:
        """sg_correlation_noalloc: the same counts with the kernel's counters in the library's static device array."""
        out = np.zeros(self.lanes, dtype=np.uint64) if out is None else out
        return sg_correlation_noalloc(self._h, slot, out)

    def energy(self, out: np.ndarray | None = None) -> np.ndarray:
        out = np.zeros(self.lanes, dtype=np.int64) if out is None else out
        return sg_energy(self._h, out)

    def corr_configure(self, nbins: int):
        _check(self._L.sg_corr_configure(self._h, int(nbins)))

    def corr_accumulate(self, slots, bins):
        slots = np.ascontiguousarray(np.asarray(slots, dtype=np.uint32))
        bins = np.ascontiguousarray(np.asarray(bins, dtype=np.uint32))
        assert slots.shape == bins.shape
        _check(self._L.sg_corr_accumulate(self._h, slots.size, _ptr(slots), _ptr(bins)))

    def corr_fetch(self, bin0: int, nbins: int):
        out = np.zeros((nbins, self.lanes), dtype=np.uint64)
        hits = np.zeros(nbins, dtype=np.uint64)
        _check(self._L.sg_corr_fetch(self._h, int(bin0), int(nbins), _ptr(out), _ptr(hits)))
        return out, hits

    # --- site-sharded sweeps (include/sg.h): the backend interface of workloads.sweep_site_sharded
    def class_units(self, k: int) -> int:
        n = C.c_uint64(0)
        _check(self._L.sg_class_units(self._h, int(k), C.byref(n)))
        return int(n.value)

    def sweep_part(self, k: int, unit0: int, n_units: int):
        _check(self._L.sg_sweep_part(self._h, int(k), int(unit0), int(n_units)))

    def end_sweep(self):
        _check(self._L.sg_end_sweep(self._h))

    def part_range(self, k: int, unit0: int, n_units: int):
        a, b = C.c_uint64(0), C.c_uint64(0)
        _check(self._L.sg_part_range(self._h, int(k), int(unit0), int(n_units), C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def export_part(self, k: int, unit0: int, n_units: int) -> np.ndarray:
        first, n = self.part_range(k, unit0, n_units)
        out = np.zeros(n, dtype=np.uint64)
        _check(self._L.sg_export_part(self._h, first, n, _ptr(out)))
        return out

    def import_part(self, k: int, unit0: int, n_units: int, words: np.ndarray):
        first, n = self.part_range(k, unit0, n_units)
        words = np.ascontiguousarray(words, dtype=np.uint64)
        assert words.size == n
        _check(self._L.sg_import_part(self._h, first, n, _ptr(words)))

    def spin_tensor(self):
        """The device spin array as a torch tensor (int64 view of the uint64 words) sharing the library's memory: for
        device-to-device collectives on the ranges of part_range()."""
        import torch

        p = C.c_void_p(0)
        _check(self._L.sg_spin_device_pointer(self._h, C.byref(p)))
        n = self.N * self.W

        class _Arr:
            __cuda_array_interface__ = {"shape": (n,), "typestr": "<i8", "data": (int(p.value), False), "version": 3}

        return torch.as_tensor(_Arr(), device=torch.device("cuda", torch.cuda.current_device()))

    @property
    def sweep_count(self) -> int:
        return self._L.sg_sweep_count(self._h)

    @property
    def M(self) -> int:
        return self._L.sg_num_edges(self._h)

    @property
    def n_colours(self) -> int:
        return self._L.sg_num_colours(self._h)

    @property
    def max_degree(self) -> int:
        return self._L.sg_max_degree(self._h)

    def spins(self, slot: int = -1, out: np.ndarray | None = None) -> np.ndarray:
        if out is None:
            out = np.zeros((self.N, self.groups), dtype=np.uint64)
        assert out.dtype == np.uint64 and out.flags.c_contiguous and out.size == self.N * self.groups
        _check(self._L.sg_get_spins(self._h, slot, _ptr(out)))
        return out

    def set_spins(self, words: np.ndarray):
        words = np.ascontiguousarray(np.asarray(words, dtype=np.uint64).reshape(self.N, self.groups))
        _check(self._L.sg_set_spins(self._h, _ptr(words)))

    def set_sweep_count(self, t: int):
        _check(self._L.sg_set_sweep_count(self._h, int(t)))

    def graph(self):
        row_ptr = np.zeros(self.N + 1, dtype=np.uint64)
        col = np.zeros(2 * self.M, dtype=np.uint32)
        colour = np.zeros(self.N, dtype=np.uint32)
        _check(self._L.sg_get_graph(self._h, _ptr(row_ptr), _ptr(col), _ptr(colour)))
        return row_ptr, col, colour

    def edges(self) -> np.ndarray:
        u = np.zeros(self.M, dtype=np.uint32)
        v = np.zeros(self.M, dtype=np.uint32)
        _check(self._L.sg_get_edges(self._h, _ptr(u), _ptr(v)))
        return np.stack([u, v], axis=1)

    def couplings(self) -> np.ndarray:
        out = np.zeros((self.M, self.W), dtype=np.uint64)
        _check(self._L.sg_get_couplings(self._h, _ptr(out)))
        return out

    def thresholds(self, n: int) -> np.ndarray:
        out = np.zeros(n, dtype=np.uint64)
        _check(self._L.sg_get_thresholds(self._h, _ptr(out), n))
        return out


# ---- host-only helpers (no GPU) --------------------------------------------------------------------
def host_philox(c0, c1, c2, c3, k0, k1) -> np.ndarray:
    out = np.zeros(4, dtype=np.uint32)
    load_library().sg_host_philox(c0, c1, c2, c3, k0, k1, _ptr(out))
    return out


def host_graph(N: int, c: float, seed: int, model: int = SG_MODEL_VB, n_words: int = 1) -> dict:
    """The device layout of a VB instance (include/sg.h, sg_host_graph_*), built by the library's host generator only."""
    L = load_library()
    g = L.sg_host_graph_create(int(model), int(N), float(c), int(seed), int(n_words))
    if not g:
        raise SGError(SG_EINVAL, _err())
    try:
        info = np.zeros(9, dtype=np.uint64)
        _check(L.sg_host_graph_info(g, _ptr(info)))
        M, K, dmax, entries, nslices, N, nJ, it_max, gauge = (int(x) for x in info)
        a = dict(M=M, K=K, dmax=dmax, entries=entries, nslices=nslices, N=N, nJ=nJ, it_max=it_max, gauge=gauge)
        a["u"] = np.zeros(M, np.uint32); a["v"] = np.zeros(M, np.uint32)
        for k in ("colour", "orig", "tpar", "teid", "bfs_pos"):
            a[k] = np.zeros(N, np.uint32)
        a["hdr"] = np.zeros((nslices + 1, 4), np.uint32)
        a["orig_s"] = np.zeros(32 * nslices, np.uint32); a["rp_s"] = np.zeros(32 * nslices, np.uint32)
        a["col"] = np.zeros(entries, np.uint32); a["jeid"] = np.zeros(nJ, np.uint32)
        for k in ("class_pos0", "class_n", "class_slice0", "class_nslices", "class_it", "class_itx"):
            a[k] = np.zeros(K, np.uint64)
        _check(L.sg_host_graph_get(g, *(_ptr(a[k]) for k in ("u", "v", "colour", "orig", "hdr", "orig_s", "rp_s", "col", "jeid", "tpar",
                                                              "teid", "bfs_pos", "class_pos0", "class_n", "class_slice0", "class_nslices", "class_it", "class_itx"))))
        return a
    finally:
        L.sg_host_graph_destroy(g)
