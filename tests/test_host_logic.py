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
                 (0, (1 << 31) - 2, 4.0, 1.0, 1, 1), (2, 1001, 0.0, 1.0, 1, 1), (2, 6, 0.0, 1.0, 1, 1), (3, 6, 0.0, 1.0, 1, 1), (4, 100, 4.0, 1.0, 1, 1)]:
        with pytest.raises(sg.SGError):
            sg.Sim(*args)


def test_host_philox_known_answers(sg):
    from paper_1906_11195_b200 import binding

    for line in open(os.path.join(ROOT, "tests", "golden", "philox_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(x, 16) for x in line.split()]
        assert list(binding.host_philox(*v[:6])) == v[6:]


def _bfs_forest(N, e):
    """Breadth-first forest over the whole graph, roots in label order, rows in edge order: order, parent, parent edge."""
    rows = [[] for _ in range(N)]
    for k, (a, b) in enumerate(e.astype(np.int64).tolist()):
        rows[a].append((b, k)); rows[b].append((a, k))
    order, par, par_e, seen = [], [-1] * N, [-1] * N, np.zeros(N, dtype=bool)
    for r in range(N):
        if seen[r]:
            continue
        seen[r] = True
        order.append(r)
        head = len(order) - 1
        while head < len(order):
            u_ = order[head]
            for v_, k in rows[u_]:
                if not seen[v_]:
                    seen[v_] = True
                    par[v_], par_e[v_] = u_, k
                    order.append(v_)
            head += 1
    return rows, order, par, par_e


def _decode_rows(g):
    """Walk the slices exactly as the kernels do: per position the tree list, the other list (neighbour position,
    coupling-entry index), and the label the slice carries for the site."""
    N = g["N"]
    T = [[] for _ in range(N)]
    X = [[] for _ in range(N)]
    label = np.full(N, -1, dtype=np.int64)
    hdr = g["hdr"].astype(np.int64)
    it_of = np.zeros(g["nslices"], dtype=np.int64)
    itx_of = np.zeros(g["nslices"], dtype=np.int64)
    for k in range(g["K"]):
        s0, ns = int(g["class_slice0"][k]), int(g["class_nslices"][k])
        it_of[s0:s0 + ns] = int(g["class_it"][k]); itx_of[s0:s0 + ns] = int(g["class_itx"][k])
    for s_ in range(g["nslices"]):
        pos0, col_off, j_off, counts = hdr[s_]
        n, nXs, nE = counts & 63, (counts >> 6) & 1023, (counts >> 16) & 4095
        assert 1 <= n <= 32 and nE <= 32 * it_of[s_] and nXs <= 32 * itx_of[s_] and nXs <= nE
        assert hdr[s_ + 1][1] == col_off + nE and hdr[s_ + 1][2] == j_off + nXs
        x_run, t_run = 0, nXs                                      # one run: the X entries, then the T entries
        for j in range(32):
            rp = int(g["rp_s"][32 * s_ + j])
            if j >= n:
                assert g["orig_s"][32 * s_ + j] == 0xFFFFFFFF and rp == 0
                continue
            p = pos0 + j
            label[p] = int(g["orig_s"][32 * s_ + j])
            xOff, tOff, nX, nT = rp & 255, (rp >> 8) & 511, (rp >> 17) & 31, rp >> 22
            assert tOff == t_run and xOff == x_run                 # site order, no gaps
            T[p] = [int(q) for q in g["col"][col_off + tOff:col_off + tOff + nT]]
            X[p] = [(int(g["col"][col_off + xOff + r]), int(j_off + xOff + r)) for r in range(nX)]
            t_run += nT; x_run += nX
        assert x_run == nXs and t_run == nE
    return T, X, label


@pytest.mark.parametrize("model,N,c,seed,W", [(0, 1024, 4.0, 1, 1), (0, 5000, 4.0, 77, 4), (0, 333, 2.5, 3, 1), (0, 64, 7.0, 5, 2), (0, 100, 0.0, 1, 1),
                                              (0, 3000, 14.0, 9, 1), (2, 8, 0.0, 1, 1), (2, 1024, 0.0, 2, 1), (2, 4102, 0.0, 3, 16), (3, 8, 0.0, 4, 1), (3, 2500, 0.0, 5, 2)])
def test_host_generator_matches_oracle_and_layout_is_consistent(sg, oracle_mod, model, N, c, seed, W):
    """model 0: Erdos-Renyi (O2); model 2: random regular bipartite graph of degree 4 (O2b); model 3: random regular graph
    of degree 4 (O2c).  The layout rules of
    include/sg.h (sg_host_graph_*) are re-derived here in plain Python from the oracle's edge list and colouring."""
    from paper_1906_11195_b200 import binding

    g = binding.host_graph(N, c, seed, model, W)
    o = oracle_mod.Oracle(model, N, c, 1.0, seed, 1)
    assert g["M"] == o.M and g["K"] == o.n_colours and g["dmax"] == o.max_degree
    e = o.edges()
    assert np.array_equal(g["u"], e[:, 0]) and np.array_equal(g["v"], e[:, 1])
    _, _, colour = o.graph()
    assert np.array_equal(g["colour"], colour)
    NONE = 0xFFFFFFFF
    K = g["K"]
    assert g["gauge"] == 1
    orig = g["orig"].astype(np.int64)
    assert np.array_equal(np.sort(orig), np.arange(N))
    pos = np.empty(N, dtype=np.int64)
    pos[orig] = np.arange(N)
    degree = np.bincount(e.ravel().astype(np.int64), minlength=N)
    rows, order, par, par_e = _bfs_forest(N, e)
    # positions: class-major; inside a class breadth-first order, every window of 4096 sites stably sorted by
    # (demand, shape); demand 0: a neighbour in a class of fewer than N/32 sites, 1: fewer than N/8, 2: fewer than N/4, 3: none;
    # shape 0: at most 2 X and 2 T entries, 1: at most 4 and 4, 2: longer rows (T = forest edges, X = the others)
    csize = np.bincount(colour, minlength=K)

    def demand(i):
        return min([3] + [0 if 32 * csize[colour[v_]] < N else 1 if 8 * csize[colour[v_]] < N else 2 if 4 * csize[colour[v_]] < N else 3
                          for v_, _ in rows[i]])
    nT_lab = np.zeros(N, dtype=np.int64)
    for i in range(N):
        if par[i] >= 0:
            nT_lab[i] += 1; nT_lab[par[i]] += 1

    def shape(nx, nt):
        return 0 if (nx <= 2 and nt <= 2) else 1 if (nx <= 4 and nt <= 4) else 2
    p0 = 0
    for k in range(K):
        members = [i for i in order if colour[i] == k]
        members = [i for a in range(0, len(members), 4096)
                   for i in sorted(members[a:a + 4096], key=lambda i: (demand(i), shape(degree[i] - nT_lab[i], nT_lab[i])))]
        assert int(g["class_pos0"][k]) == p0 and int(g["class_n"][k]) == len(members)
        assert orig[p0:p0 + len(members)].tolist() == members
        p0 += len(members)
    # forest arrays
    for p in range(N):
        i = orig[p]
        if par[i] < 0:
            assert g["tpar"][p] == NONE and g["teid"][p] == NONE
        else:
            assert g["tpar"][p] == pos[par[i]] and g["teid"][p] == par_e[i]
    assert np.array_equal(g["bfs_pos"], pos[np.array(order, dtype=np.int64)])
    # rows: T = parent first, then children by position; X = the other neighbours by position; every coupling
    # entry carries its edge id; every non-tree edge is stored at both endpoints, every tree edge at none
    T, X, label = _decode_rows(g)
    assert np.array_equal(label, orig)
    seen_edges = np.zeros(g["M"], dtype=np.int64)
    nT = np.zeros(N, dtype=np.int64)
    for p in range(N):
        i = orig[p]
        children = sorted(pos[v_] for v_, k in rows[i] if par_e[v_] == k and par[v_] == i)
        assert T[p] == ([pos[par[i]]] if par[i] >= 0 else []) + children
        nT[p] = len(T[p])
        tree_edges = {par_e[i]} | {k for v_, k in rows[i] if par_e[v_] == k and par[v_] == i}
        others = sorted((pos[v_], k) for v_, k in rows[i] if k not in tree_edges)
        assert [q for q, _ in X[p]] == [q for q, _ in others]
        for (q, x), (_, k) in zip(X[p], others):
            assert g["jeid"][x] == k
            seen_edges[k] += 1
    is_tree = np.zeros(g["M"], dtype=bool)
    is_tree[[k for k in par_e if k >= 0]] = True
    assert np.all(seen_edges[~is_tree] == 2) and np.all(seen_edges[is_tree] == 0)
    assert g["entries"] == 2 * g["M"] and g["nJ"] == 2 * int((~is_tree).sum())
    # slices: greedy cut of every class into runs of <= 32 sites within the class's budgets (32*it entries, 32*itx X
    # entries), never across classes; the budget is the first of include/sg.h's list within 30 % of the last one's slice count
    def cut(k, it, itx):
        runs = []
        p, pend = int(g["class_pos0"][k]), int(g["class_pos0"][k]) + int(g["class_n"][k])
        while p < pend:
            n = sE = sX = 0
            while p + n < pend and n < 32:
                d_, x = degree[orig[p + n]], degree[orig[p + n]] - nT[p + n]
                if n > 0 and (sE + d_ > 32 * it or sX + x > 32 * itx):
                    break
                sE += d_; sX += x; n += 1
            runs.append((p, n, sX, sE))
            p += n
        return runs
    budgets = [(6, 4), (8, 6)] if W % 2 else [(4, 3)]
    hdr = g["hdr"].astype(np.int64)
    s_ = 0
    for k in range(K):
        assert int(g["class_slice0"][k]) == s_
        best = next(b_ for b_ in budgets if 100 * len(cut(k, *b_)) <= 130 * len(cut(k, *budgets[-1])))
        assert (int(g["class_it"][k]), int(g["class_itx"][k])) == best
        for p, n, sX, sE in cut(k, *best):
            sh = max(shape(degree[orig[q]] - nT[q], nT[q]) for q in range(p, p + n))
            assert hdr[s_][0] == p and hdr[s_][3] == (n | sX << 6 | sE << 16 | sh << 28)
            s_ += 1
        assert int(g["class_nslices"][k]) == s_ - int(g["class_slice0"][k])
    assert s_ == g["nslices"] and hdr[s_][0] == N and g["it_max"] == max(int(x) for x in g["class_it"])
    # no edge inside a colour class (the race-freedom condition of the parallel update)
    assert np.all(colour[e[:, 0]] != colour[e[:, 1]])


def test_gauged_layout_reproduces_the_oracle_sweep(sg, oracle_mod):
    """The gauge transformation changes no output (include/sg.h): a plain-Python sweep over the device layout, with the
    transformed spins sigma ^ eps and couplings kappa ^ eps_i ^ eps_j and NO coupling word on tree entries, gives
    the oracle's configurations once eps is undone.  Pins the host side of the gauge before any kernel runs."""
    from paper_1906_11195_b200 import binding

    N, c, T_, seed = 600, 4.0, 1.0, 4
    g = binding.host_graph(N, c, seed, 0)
    o = oracle_mod.Oracle(0, N, c, T_, seed, 1)
    kappa = [int(x) for x in o.couplings()[:, 0]]
    sigma = [int(x) for x in o.spins()[:, 0]]
    thr = [int(x) for x in o.thresholds(o.max_degree + 1)] + [0] * 40
    NONE = 0xFFFFFFFF
    orig = g["orig"].astype(np.int64)
    eps = [0] * N
    for p in g["bfs_pos"].tolist():
        if g["tpar"][p] != NONE:
            eps[p] = eps[int(g["tpar"][p])] ^ kappa[int(g["teid"][p])]
    T, X, _ = _decode_rows(g)
    spin = [sigma[orig[p]] ^ eps[p] for p in range(N)]
    J = [0] * g["nJ"]
    for p in range(N):
        for q, x in X[p]:
            J[x] = kappa[int(g["jeid"][x])] ^ eps[p] ^ eps[q]
    M64 = (1 << 64) - 1
    for t in range(3):
        for k in range(g["K"]):
            p0, n = int(g["class_pos0"][k]), int(g["class_n"][k])
            for p in range(p0, p0 + n):
                r = int(oracle_mod.philox(int(orig[p]), 0, t, 0, seed & 0xFFFFFFFF, seed >> 32)[0])
                bonds = [spin[p] ^ spin[q] for q in T[p]] + [spin[p] ^ spin[q] ^ J[x] for q, x in X[p]]
                d = len(bonds)
                flip = 0
                for b in range(64):
                    u_ = sum((m >> b) & 1 for m in bonds)
                    kk = d - 2 * u_
                    if kk <= 0 or r < thr[kk]:
                        flip |= 1 << b
                spin[p] ^= flip & M64
        o.sweep(1)
        got = np.zeros(N, dtype=np.uint64)
        for p in range(N):
            got[orig[p]] = spin[p] ^ eps[p]
        assert np.array_equal(got, o.spins()[:, 0]), f"sweep {t}"


def test_layout_overhead_is_small(sg):
    from paper_1906_11195_b200 import binding

    g = binding.host_graph(1 << 18, 4.0, 1)
    # no padding entries at all; the forest's N - (number of components) edges carry no coupling word; almost all
    # slices are full (32 sites): the per-slice arrays hold little more than one slot per site
    assert g["entries"] == 2 * g["M"]
    assert g["nJ"] < 0.52 * g["entries"]
    assert 32 * g["nslices"] < 1.08 * g["N"]


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


def test_tritone_index_is_the_papers_lump():
    """"we lump together the data for the same value of floor(ln((t+tw)/4)/(0.5 ln 2)) ... e.g. we lump
    together the t + tw = {4, 5} data"."""
    import math

    from paper_1906_11195_b200.workloads import tritone_index

    assert tritone_index(4) == tritone_index(5) == 0 and tritone_index(6) == 1
    for x in range(4, 20000):
        v = math.log(x / 4) / (0.5 * math.log(2))
        if abs(v - round(v)) > 1e-9:                      # away from the lump edges floating point is safe
            assert tritone_index(x) == math.floor(v), x
    for k in range(2, 40):                                # the edges that are integers: x = 2^k -> index 2k - 4
        assert tritone_index(1 << k) == 2 * k - 4 and tritone_index((1 << k) - 1) == 2 * k - 5
    sizes = {}
    for x in range(4, 1 << 16):
        sizes[tritone_index(x)] = sizes.get(tritone_index(x), 0) + 1
    for m in range(14, 24):                               # lump widths grow by sqrt(2): "tritone" intervals
        assert abs(sizes[m + 1] / sizes[m] - 2 ** 0.5) < 0.02


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


def test_sweep_kernels_read_no_spin_before_the_dependent_launch_wait(sg):
    """The sweep launches are programmatic dependent launches: a CTA may start while the previous colour class is still
    running, reads its read-only streams, and must not touch a spin word before `griddepcontrol.wait` (SASS: ACQBULK).
    ptxas is kept from hoisting the wait above the stream loads by a never-taken exit (csrc/sg_vb_sweep.cu); this
    test pins the resulting order in the shipped binary: in every k_vb_sweep instantiation, every global load in
    front of ACQBULK is a read-only (.CONSTANT) load, there are at least four of them, the first plain load (a spin
    word) and the only store come after it."""
    import shutil
    import subprocess

    from paper_1906_11195_b200 import binding

    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", binding.LIB_PATH], capture_output=True, text=True, check=True).stdout
    funcs = re.split(r"\n\s*Function : ", sass)[1:]
    sweeps = [f for f in funcs if "k_vb_sweep" in f.split("\n", 1)[0]]
    assert len(sweeps) >= 6                                    # G = 1 (W = 1 and general), 2, 4, each narrow and wide
    for f in sweeps:
        name = f.split("\n", 1)[0]
        ops = re.findall(r"/\*[0-9a-f]{4}\*/\s+(?:@!?U?P\d\s+)?([A-Z0-9_.]+)", f)
        assert ops.count("ACQBULK") == 1, name
        k = ops.index("ACQBULK")
        before, after = ops[:k], ops[k + 1:]
        loads_before = [o for o in before if o.startswith("LDG")]
        assert len(loads_before) >= 4 and all(".CONSTANT" in o for o in loads_before), (name, loads_before)
        assert not any(o.startswith(("STG", "ATOM", "RED")) for o in before), name
        assert any(o.startswith("LDG") and ".CONSTANT" not in o for o in after), name      # the spin reads
        assert sum(1 for o in after if o.startswith("STG")) >= 1, name
