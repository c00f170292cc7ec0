"""CPU tests of the product's host side: the C-ABI library loads and exports every symbol of
include/sg.h; its host Philox and host generator agree with the oracle; the device layout is
self-consistent; without a GPU the compute calls fail loudly (no CPU fallback)."""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sg():
    from paper_1906_11195_b200 import build as b

    b.build()
    import paper_1906_11195_b200 as sg

    return sg


def test_library_exports_every_declared_symbol(sg):
    from paper_1906_11195_b200 import binding

    L = sg.load_library()
    hdr = open(os.path.join(ROOT, "include", "sg.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(sg_[a-z_0-9]+)\s*\(", hdr))
    assert {"sg_create", "sg_sweep", "sg_snapshot", "sg_correlation", "sg_energy", "sg_destroy"} <= declared
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)


def test_no_cpu_fallback(sg):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(sg.SGError) as e:
        sg.Sim(sg.SG_MODEL_VB, 1024, 4.0, 1.0, 1, 1)
    assert "no CUDA device" in str(e.value) or "CUDA" in str(e.value)


def test_bad_arguments_are_rejected_before_touching_the_gpu(sg):
    for args in [(7, 100, 4.0, 1.0, 1, 1), (0, 1, 4.0, 1.0, 1, 1), (0, 100, 4.0, 1.0, 1, 0),
                 (0, 100, 4.0, -0.5, 1, 1), (0, 100, 4.0, float("nan"), 1, 1), (1, 40000, 0.0, 1.0, 1, 1),
                 (0, 1 << 31, 4.0, 1.0, 1, 1), (2, 1001, 0.0, 1.0, 1, 1), (2, 6, 0.0, 1.0, 1, 1)]:
        with pytest.raises(sg.SGError):
            sg.Sim(*args)


def test_host_philox_known_answers(sg):
    from paper_1906_11195_b200 import binding

    for line in open(os.path.join(ROOT, "tests", "golden", "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(x, 16) for x in line.split()]
        assert list(binding.host_philox(*v[:6])) == v[6:]


@pytest.mark.parametrize("model,N,c,seed", [(0, 1024, 4.0, 1), (0, 5000, 4.0, 77), (0, 333, 2.5, 3), (0, 64, 7.0, 5), (0, 100, 0.0, 1),
                                            (2, 8, 0.0, 1), (2, 1024, 0.0, 2), (2, 4102, 0.0, 3)])
def test_host_generator_matches_oracle_and_layout_is_consistent(sg, oracle_mod, model, N, c, seed):
    """model 0: Erdos-Renyi (O2); model 2: random regular bipartite graph of degree 4 (O2b)."""
    from paper_1906_11195_b200 import binding

    g = binding.host_graph(N, c, seed, model)
    o = oracle_mod.Oracle(model, N, c, 1.0, seed, 1)
    assert g["M"] == o.M and g["K"] == o.n_colours and g["dmax"] == o.max_degree
    e = o.edges()
    assert np.array_equal(g["u"], e[:, 0]) and np.array_equal(g["v"], e[:, 1])
    _, _, colour = o.graph()
    assert np.array_equal(g["colour"], colour)
    # positions: class-major; inside a class the valid positions are the class's sites in breadth-first order
    # (roots in label order, rows in edge order), each window of sort_window sites stably sorted by degree;
    # classes start at multiples of 32, gaps are padding (orig = NONE)
    NONE = 0xFFFFFFFF
    P = g["P"]
    assert P % 32 == 0 and g["nslices"] == P // 32
    orig_all = g["orig"].astype(np.int64)
    valid = orig_all != NONE
    orig = orig_all[valid]
    assert np.array_equal(np.sort(orig), np.arange(N))
    degree = np.bincount(e.ravel().astype(np.int64), minlength=N)
    assert np.array_equal(g["deg"][valid], degree[orig]) and np.all(g["deg"][~valid] == 0)
    rows = [[] for _ in range(N)]
    for a, b in e.astype(np.int64).tolist():
        rows[a].append(b); rows[b].append(a)
    bfs, seen = [], np.zeros(N, dtype=bool)
    for r in range(N):
        if seen[r]:
            continue
        seen[r] = True
        bfs.append(r)
        head = len(bfs) - 1
        while head < len(bfs):
            for v_ in rows[bfs[head]]:
                if not seen[v_]:
                    seen[v_] = True
                    bfs.append(v_)
            head += 1
    SW = g["sort_window"]
    for k in range(g["K"]):
        p0, n, s0 = int(g["class_pos0"][k]), int(g["class_n"][k]), int(g["class_slice0"][k])
        assert p0 % 32 == 0 and n % 32 == 0 and s0 == p0 // 32
        members = [i for i in bfs if colour[i] == k]
        assert 0 <= n - len(members) < 32
        expect = []
        for w0 in range(0, len(members), SW):
            expect += sorted(members[w0:w0 + SW], key=lambda i: degree[i])      # sorted() is stable
        assert orig_all[p0:p0 + len(members)].tolist() == expect
        assert np.all(orig_all[p0 + len(members):p0 + n] == NONE)
    pos = np.empty(N, dtype=np.int64)
    pos[orig] = np.nonzero(valid)[0]
    sp = g["slice_ptr"].astype(np.int64)
    # row length of a slice = largest degree in it
    degs = g["deg"].astype(np.int64).reshape(-1, 32)
    assert np.array_equal(np.diff(sp), degs.max(axis=1))
    nbrs = [set() for _ in range(P)]
    for a, b in e.astype(np.int64):
        nbrs[pos[a]].add(pos[b]); nbrs[pos[b]].add(pos[a])
    seen_edges = np.zeros(g["M"], dtype=np.int64)
    for s_ in range(P // 32):
        D = sp[s_ + 1] - sp[s_]
        for j in range(32):
            p = 32 * s_ + j
            ents = 32 * sp[s_] + 32 * np.arange(D) + j
            d = int(g["deg"][p])
            # padding entries (beyond the degree, or a padding position) point at the site itself, no edge
            assert np.all(g["eid"][ents[d:]] == NONE) and np.all(g["col"][ents[d:]] == p)
            if orig_all[p] == NONE:
                assert d == 0
                continue
            assert set(g["col"][ents[:d]].tolist()) == nbrs[p] and len(nbrs[p]) == d
            for q in range(d):
                ed = int(g["eid"][ents[q]])
                a, b = int(e[ed, 0]), int(e[ed, 1])
                assert {pos[a], pos[b]} == {p, int(g["col"][ents[q]])}
                seen_edges[ed] += 1
    assert np.all(seen_edges == 2)                      # every edge stored at both endpoints
    assert g["entries"] == 32 * sp[-1]
    # no edge inside a colour class (the race-freedom condition of the parallel update)
    assert np.all(colour[e[:, 0]] != colour[e[:, 1]])


def test_padding_overhead_is_small(sg):
    from paper_1906_11195_b200 import binding

    g = binding.host_graph(1 << 18, 4.0, 1)
    # padding positions: < 32 per class; padding entries: slices that straddle two degrees inside a sort window
    assert g["P"] - g["N"] < 32 * g["K"]
    assert g["entries"] <= 1.02 * 2 * g["M"]


def test_schedule_counts():
    from paper_1906_11195_b200.workloads import schedule

    ev = schedule(1024)
    assert sum(1 for x in ev if x[1] == "snap") == 11
    assert sum(1 for x in ev if x[1] == "corr") == 100        # 100 pairs at config 1
    assert all(ev[i][0] <= ev[i + 1][0] for i in range(len(ev) - 1))
    snapped = set()
    for t, kind, slot in ev:
        if kind == "snap":
            assert t == 1 << slot
            snapped.add(slot)
        else:
            assert slot in snapped and t > (1 << slot) and bin(t - (1 << slot)).count("1") == 1


def test_window_index_is_the_minor_third_bin():
    """bins (t_m, t_{m+1}] with t_m = 2^(m/4); checked against floating point away from the bin edges and
    exactly at the edges that are integers (t = 2^k = t_{4k} belongs to bin 4k - 1)."""
    import math

    from paper_1906_11195_b200.workloads import window_index

    assert window_index(1) == -1
    for k in range(1, 40):
        assert window_index(1 << k) == 4 * k - 1
        if k >= 3:
            assert window_index((1 << k) + 1) == 4 * k
    for t in list(range(2, 5000)) + [10**6 + 7, 2**25 - 1]:
        m = window_index(t)
        assert 2.0 ** (m / 4) < t <= 2.0 ** ((m + 1) / 4) * (1 + 1e-12)
    # the bins of 1..T partition the times, and bin widths grow by 2^(1/4)
    T = 4096
    seen = {}
    for t in range(2, T + 1):
        seen.setdefault(window_index(t), []).append(t)
    assert sum(len(v) for v in seen.values()) == T - 1
    big = [m for m in seen if m >= 40 and m + 1 in seen and max(seen[m + 1]) < T]
    for m in big:
        assert abs(len(seen[m + 1]) / len(seen[m]) - 2 ** 0.25) < 0.15


def test_windowed_protocol_on_the_oracle(oracle_mod):
    """run_windowed against a direct recomputation from stored configurations (small N, the oracle as the simulator)."""
    from paper_1906_11195_b200.workloads import run_windowed, window_index

    N, S = 512, 80
    o = oracle_mod.Oracle(oracle_mod.RRBG, N, 0.0, 1.2149, 3, 1)
    res = run_windowed(o, S, tws=(4, 16, 64, 256))
    o2 = oracle_mod.Oracle(oracle_mod.RRBG, N, 0.0, 1.2149, 3, 1)
    from tests import exact
    states = {0: exact.unpack(o2.spins())}
    for t in range(1, S + 1):
        o2.sweep(1)
        states[t] = exact.unpack(o2.spins())
    expect = {}
    for tw in (4, 16, 64):
        for t in range(tw + 1, S + 1):
            key = (tw, window_index(t))
            d = (states[t] != states[tw]).sum(axis=0).astype(np.uint64)
            expect[key] = (expect[key][0] + d, expect[key][1] + 1) if key in expect else (d, 1)
    assert res.keys() == expect.keys()
    for k in res:
        assert res[k][1] == expect[k][1] and np.array_equal(res[k][0], expect[k][0]), k
