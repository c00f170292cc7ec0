// sg_host.cpp -- host side of sg_create: Philox, the seeded instance generator (row a1 of
// SURVEY.md section 8(a)), thresholds.  Conventions: DESIGN.md section 3 (O1, O2, O5, O6).
// Independent of oracle/: nothing here is shared with or derived from it.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <numeric>

#include "sg_internal.h"

// ---- O1: Philox4x32-10 ------------------------------------------------------------------------
Philox4 sg_philox_host(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
    constexpr uint64_t MUL_A = 0xD2511F53ull, MUL_B = 0xCD9E8D57ull;
    for (int r = 0; r < 10; ++r) {
        const uint64_t pa = MUL_A * c0, pb = MUL_B * c2;
        const uint32_t y0 = uint32_t(pb >> 32) ^ c1 ^ k0;
        const uint32_t y2 = uint32_t(pa >> 32) ^ c3 ^ k1;
        c1 = uint32_t(pb);
        c3 = uint32_t(pa);
        c0 = y0;
        c2 = y2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return Philox4{{c0, c1, c2, c3}};
}

// ---- O6: integer acceptance thresholds ----------------------------------------------------------
static uint64_t acceptance_threshold(double two_k, double denom)
{
    const double p = std::exp(-two_k / denom);       // T=0: -x/0 = -inf -> 0 ; T=inf: -x/inf = -0 -> 1
    return (uint64_t)std::floor(std::ldexp(p, 32));  // kept in 64 bits: p = 1 gives 2^32
}

std::vector<uint64_t> sg_vb_thresholds(double T, uint32_t dmax)
{
    std::vector<uint64_t> thr(dmax + 1, 0);
    for (uint32_t k = 1; k <= dmax; ++k) thr[k] = acceptance_threshold((double)(2 * (int)k), T);
    return thr;
}

std::vector<uint64_t> sg_sk_thresholds(double T, uint64_t N)
{
    std::vector<uint64_t> thr(N, 0);
    const double denom = T * std::sqrt((double)N);
    for (uint64_t m = 1; m < N; ++m) thr[m] = acceptance_threshold((double)(2 * (int64_t)m), denom);
    return thr;
}

// ---- O2: edge list ------------------------------------------------------------------------------
// Open-addressing set of unordered pairs, key = lo<<32 | hi (never 0xFFFF... since lo < hi < 2^32).
namespace {
struct PairSet {
    std::vector<uint64_t> slot;
    uint64_t mask;
    explicit PairSet(uint64_t expected)
    {
        uint64_t cap = 16;
        while (cap < 2 * expected + 16) cap <<= 1;
        slot.assign(cap, ~0ull);
        mask = cap - 1;
    }
    static uint64_t mix(uint64_t x)
    {
        x ^= x >> 33; x *= 0xff51afd7ed558ccdull; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull; x ^= x >> 33;
        return x;
    }
    // true if inserted, false if already present
    bool insert(uint64_t key)
    {
        uint64_t h = mix(key) & mask;
        while (true) {
            const uint64_t s = slot[h];
            if (s == ~0ull) { slot[h] = key; return true; }
            if (s == key) return false;
            h = (h + 1) & mask;
        }
    }
};
}  // namespace

// O2b: random regular bipartite graph of degree 4 as the union of four permutations of
// half A = {0..H-1} onto half B = {H..N-1}, H = N/2, without a repeated pair.  Permutation a = 0..3: attempts
// t = 0,1,2,... (one counter over all four); an attempt is a Fisher-Yates shuffle of the identity, for i = H-1 down
// to 1: j = (x*(i+1)) >> 32 with x = word n&3 of P(n>>2, t, 0, tag 4), n = H-1-i, swap(perm[i], perm[j]); it is
// accepted if it differs from every earlier accepted permutation at every i.  Edge e = a*H + i joins i and H + perm_a[i].
static bool build_rrbg_edges(uint64_t N, uint64_t seed, VBHostGraph &g)
{
    if (N < 8 || (N & 1)) { sg_set_error("sg_create: the RRBG model needs an even N >= 8"); return false; }
    const uint64_t H = N / 2;
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    g.N = N; g.M = 4 * H;
    g.eu.resize(g.M); g.ev.resize(g.M);
    std::vector<uint32_t> perm(H);
    uint64_t t = 0;
    for (uint32_t a = 0; a < 4; ++a) {
        for (;; ++t) {
            std::iota(perm.begin(), perm.end(), 0u);
            Philox4 x{{0, 0, 0, 0}};
            for (uint64_t i = H - 1; i >= 1; --i) {
                const uint64_t n = H - 1 - i;
                if ((n & 3) == 0) x = sg_philox_host((uint32_t)(n >> 2), (uint32_t)t, 0u, 4u << 24, k0, k1);
                const uint64_t j = ((uint64_t)x.x[n & 3] * (i + 1)) >> 32;
                std::swap(perm[i], perm[j]);
            }
            bool clash = false;
            for (uint32_t b = 0; b < a && !clash; ++b)
                for (uint64_t i = 0; i < H; ++i)
                    if (g.ev[(uint64_t)b * H + i] == (uint32_t)(H + perm[i])) { clash = true; break; }
            if (!clash) { ++t; break; }
        }
        for (uint64_t i = 0; i < H; ++i) {
            g.eu[(uint64_t)a * H + i] = (uint32_t)i;
            g.ev[(uint64_t)a * H + i] = (uint32_t)(H + perm[i]);
        }
    }
    return true;
}

// O2: Erdos-Renyi G(N, M), M = floor(c N / 2 + 0.5), self-loops and repeated pairs rejected
static bool build_er_edges(uint64_t N, double c, uint64_t seed, VBHostGraph &g)
{
    if (!(c >= 0.0) || !std::isfinite(c)) { sg_set_error("sg_create: c must be finite and >= 0"); return false; }
    const double pairs = 0.5 * (double)N * (double)(N - 1);
    const double Md = std::floor(c * (double)N / 2.0 + 0.5);
    if (Md > pairs) { sg_set_error("sg_create: c*N/2 exceeds the number of site pairs"); return false; }
    if (Md >= 2147483648.0) { sg_set_error("sg_create: more than 2^31 edges are not supported"); return false; }
    const uint64_t M = (uint64_t)Md;
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    g.N = N; g.M = M;
    g.eu.resize(M); g.ev.resize(M);
    PairSet seen(M);
    uint64_t e = 0;
    for (uint64_t a = 0; e < M; ++a) {
        const Philox4 x = sg_philox_host((uint32_t)a, (uint32_t)(a >> 32), 0u, 3u << 24, k0, k1);
        const uint32_t u = (uint32_t)(((uint64_t)x.x[0] * N) >> 32);
        const uint32_t v = (uint32_t)(((uint64_t)x.x[1] * N) >> 32);
        if (u == v) continue;
        const uint64_t key = u < v ? ((uint64_t)u << 32 | v) : ((uint64_t)v << 32 | u);
        if (!seen.insert(key)) continue;
        g.eu[e] = u; g.ev[e] = v; ++e;
    }
    return true;
}

bool sg_build_vb_graph(int model, uint64_t N, double c, uint64_t seed, VBHostGraph &g)
{
    if (model == SG_MODEL_RRBG ? !build_rrbg_edges(N, seed, g) : !build_er_edges(N, c, seed, g)) return false;
    const uint64_t M = g.M;
    // CSR in original labels, rows in increasing edge id
    g.row_ptr.assign(N + 1, 0);
    for (uint64_t e = 0; e < M; ++e) { g.row_ptr[g.eu[e] + 1]++; g.row_ptr[g.ev[e] + 1]++; }
    uint64_t dmax = 0;
    for (uint64_t i = 0; i < N; ++i) { dmax = std::max(dmax, g.row_ptr[i + 1]); g.row_ptr[i + 1] += g.row_ptr[i]; }
    if (dmax > 31) { sg_set_error("sg_create: maximum degree above 31 is not supported (5 count bit-planes)"); return false; }
    g.dmax = (uint32_t)dmax;
    g.adj.resize(2 * M); g.adj_e.resize(2 * M);
    {
        std::vector<uint64_t> fill(g.row_ptr.begin(), g.row_ptr.end() - 1);
        for (uint64_t e = 0; e < M; ++e) {
            const uint32_t u = g.eu[e], v = g.ev[e];
            g.adj[fill[u]] = v; g.adj_e[fill[u]++] = (uint32_t)e;
            g.adj[fill[v]] = u; g.adj_e[fill[v]++] = (uint32_t)e;
        }
    }
    // O5: first-fit colouring in natural order (bit mask of colours used by lower-numbered neighbours)
    g.colour.assign(N, 0);
    uint32_t K = 0;
    for (uint64_t i = 0; i < N; ++i) {
        uint64_t used = 0;
        for (uint64_t a = g.row_ptr[i]; a < g.row_ptr[i + 1]; ++a)
            if (g.adj[a] < i) used |= 1ull << g.colour[g.adj[a]];
        const uint32_t col = (uint32_t)__builtin_ctzll(~used);
        g.colour[i] = (uint8_t)col;
        K = std::max(K, col + 1);
    }
    g.K = K;
    // Locality order (the "locality-improving relabelling within each colour class" of BASELINE.json): breadth-first
    // index over the whole graph, roots in label order, rows in stored order.  The graph is locally tree-like, so
    // a site's tree parent and children get nearby indices; since a class keeps this order, the gathers along the
    // N-1 tree edges (half of all gathers at c = 4) walk through every other class's block monotonically and find
    // their 32-byte sectors still in L2 (or L1) instead of costing a DRAM row activation each.
    // (SG_VB_ORDER=label keeps the label order instead: a measurement knob, see profiles/; outputs are identical.)
    std::vector<uint32_t> bfs; bfs.reserve(N);
    const char *order_env = std::getenv("SG_VB_ORDER");
    if (order_env && !std::strcmp(order_env, "label")) {
        bfs.resize(N);
        std::iota(bfs.begin(), bfs.end(), 0u);
    } else {
        std::vector<uint8_t> seen(N, 0);
        for (uint64_t r = 0; r < N; ++r) {
            if (seen[r]) continue;
            seen[r] = 1;
            size_t head = bfs.size();
            bfs.push_back((uint32_t)r);
            while (head < bfs.size()) {
                const uint32_t u = bfs[head++];
                for (uint64_t a = g.row_ptr[u]; a < g.row_ptr[u + 1]; ++a) {
                    const uint32_t v = g.adj[a];
                    if (!seen[v]) { seen[v] = 1; bfs.push_back(v); }
                }
            }
        }
    }
    // Positions: class-major; inside a class the sites keep the BFS order, except that every window of
    // SG_SORT_WINDOW consecutive sites is stably sorted by degree, so that the 32 sites of a slice have (almost
    // always) one degree and the sliced-ELL rows carry ~1 % padding.  Classes start at multiples of 32; the gap
    // positions are padding (orig = NONE, spin word 0, never written).
    std::vector<uint64_t> ccount(K, 0);
    for (uint64_t i = 0; i < N; ++i) ccount[g.colour[i]]++;
    g.cls.assign(K, VBClass{});
    uint64_t P = 0;
    for (uint32_t k = 0; k < K; ++k) {
        g.cls[k].pos0 = P;
        g.cls[k].n = (ccount[k] + 31) / 32 * 32;
        P += g.cls[k].n;
    }
    if (P >= (1ull << 31)) { sg_set_error("sg_create: too many sites"); return false; }
    g.P = P;
    g.orig.assign(P, SG_NONE); g.pos.resize(N); g.deg.assign(P, 0);
    {
        std::vector<uint64_t> fill(K);
        for (uint32_t k = 0; k < K; ++k) fill[k] = g.cls[k].pos0;
        for (uint64_t q = 0; q < N; ++q) g.orig[fill[g.colour[bfs[q]]]++] = bfs[q];
        const uint64_t SW = SG_SORT_WINDOW;
        std::vector<uint32_t> tmp(SW);
        for (uint32_t k = 0; k < K; ++k) {
            const uint64_t p0 = g.cls[k].pos0, p1 = p0 + ccount[k];
            for (uint64_t w0 = p0; w0 < p1; w0 += SW) {
                const uint64_t w1 = std::min<uint64_t>(p1, w0 + SW);
                uint32_t hist[33] = {0};
                for (uint64_t p = w0; p < w1; ++p) hist[g.row_ptr[g.orig[p] + 1] - g.row_ptr[g.orig[p]] + 1]++;
                for (int d = 0; d < 32; ++d) hist[d + 1] += hist[d];
                for (uint64_t p = w0; p < w1; ++p) tmp[hist[g.row_ptr[g.orig[p] + 1] - g.row_ptr[g.orig[p]]]++] = g.orig[p];
                std::copy(tmp.begin(), tmp.begin() + (w1 - w0), g.orig.begin() + w0);
            }
        }
        for (uint64_t p = 0; p < P; ++p)
            if (g.orig[p] != SG_NONE) {
                g.pos[g.orig[p]] = (uint32_t)p;
                g.deg[p] = (uint8_t)(g.row_ptr[g.orig[p] + 1] - g.row_ptr[g.orig[p]]);
            }
    }
    std::vector<uint32_t>().swap(bfs);
    // sliced ELL: slice s = positions 32 s .. 32 s + 31, row length = the largest degree in the slice
    const uint64_t nslices = P / 32;
    g.slice_ptr.assign(nslices + 1, 0);
    for (uint64_t s = 0; s < nslices; ++s) {
        uint32_t D = 0;
        for (uint32_t j = 0; j < 32; ++j) D = std::max<uint32_t>(D, g.deg[32 * s + j]);
        const uint64_t next = (uint64_t)g.slice_ptr[s] + D;
        if (next > 0x7FFFFFFull) { sg_set_error("sg_create: instance too large for 32-bit entry indices"); return false; }
        g.slice_ptr[s + 1] = (uint32_t)next;
    }
    for (uint32_t k = 0; k < K; ++k) { g.cls[k].slice0 = g.cls[k].pos0 / 32; g.cls[k].nslices = g.cls[k].n / 32; }
    const uint64_t entries = 32ull * g.slice_ptr[nslices];
    g.col.resize(entries); g.eid.assign(entries, SG_NONE);
    g.entry_of_edge.assign(M, 0);
    const bool sort_rows = std::getenv("SG_VB_ROWS") == nullptr || std::strcmp(std::getenv("SG_VB_ROWS"), "edge") != 0;   // measurement knob
    for (uint64_t s = 0; s < nslices; ++s) {
        const uint64_t base = 32ull * g.slice_ptr[s];
        const uint32_t D = g.slice_ptr[s + 1] - g.slice_ptr[s];
        for (uint32_t j = 0; j < 32; ++j) {
            const uint64_t p = 32 * s + j;
            const uint32_t i = g.orig[p];
            const uint32_t d = g.deg[p];
            // a row lists its neighbours by ascending position (= by class, then by BFS index): the 32 sites of a
            // slice are close in BFS index, so their k-th neighbours tend to share 128-byte lines
            uint64_t key[32];
            if (i != SG_NONE) {
                const uint64_t r0 = g.row_ptr[i];
                for (uint32_t q = 0; q < d; ++q) key[q] = (uint64_t)g.pos[g.adj[r0 + q]] << 32 | g.adj_e[r0 + q];
                if (sort_rows) std::sort(key, key + d);
            }
            for (uint32_t q = 0; q < D; ++q) {
                const uint64_t ent = base + 32ull * q + j;
                if (i != SG_NONE && q < d) {
                    g.col[ent] = (uint32_t)(key[q] >> 32);
                    const uint32_t e = (uint32_t)key[q];
                    g.eid[ent] = e;
                    if (g.eu[e] == i) g.entry_of_edge[e] = (uint32_t)ent;
                } else {
                    g.col[ent] = (uint32_t)p;   // padding entry: points at its own position, coupling word 0
                }
            }
        }
    }
    return true;
}

// ---- host-only C entry points (include/sg.h) ------------------------------------------------------
struct sg_host_graph { VBHostGraph g; };

extern "C" void sg_host_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t *out)
{
    const Philox4 x = sg_philox_host(c0, c1, c2, c3, k0, k1);
    for (int q = 0; q < 4; ++q) out[q] = x.x[q];
}

extern "C" sg_host_graph *sg_host_graph_create(int model, uint64_t N, double c, uint64_t seed)
{
    if (model != SG_MODEL_VB && model != SG_MODEL_RRBG) { sg_set_error("sg_host_graph_create: graph model required"); return nullptr; }
    if (N < 2 || N >= (1ull << 32)) { sg_set_error("sg_host_graph_create: N must satisfy 2 <= N < 2^32"); return nullptr; }
    sg_host_graph *h = new sg_host_graph();
    if (!sg_build_vb_graph(model, N, c, seed, h->g)) { delete h; return nullptr; }
    return h;
}

extern "C" void sg_host_graph_destroy(sg_host_graph *g) { delete g; }

extern "C" int sg_host_graph_info(const sg_host_graph *h, uint64_t *info)
{
    if (!h || !info) return SG_EINVAL;
    info[0] = h->g.M; info[1] = h->g.K; info[2] = h->g.dmax; info[3] = h->g.col.size();
    info[4] = h->g.slice_ptr.size() - 1; info[5] = h->g.N; info[6] = h->g.P; info[7] = SG_SORT_WINDOW;
    return SG_OK;
}

extern "C" int sg_host_graph_get(const sg_host_graph *h, uint32_t *u, uint32_t *v, uint32_t *colour, uint32_t *orig,
                                 uint32_t *deg, uint32_t *slice_ptr, uint32_t *col, uint32_t *eid,
                                 uint64_t *class_pos0, uint64_t *class_n, uint64_t *class_slice0)
{
    if (!h) return SG_EINVAL;
    const VBHostGraph &g = h->g;
    if (u) std::copy(g.eu.begin(), g.eu.end(), u);
    if (v) std::copy(g.ev.begin(), g.ev.end(), v);
    if (colour) std::copy(g.colour.begin(), g.colour.end(), colour);
    if (orig) std::copy(g.orig.begin(), g.orig.end(), orig);
    if (deg) std::copy(g.deg.begin(), g.deg.end(), deg);
    if (slice_ptr) std::copy(g.slice_ptr.begin(), g.slice_ptr.end(), slice_ptr);
    if (col) std::copy(g.col.begin(), g.col.end(), col);
    if (eid) std::copy(g.eid.begin(), g.eid.end(), eid);
    for (uint32_t k = 0; k < g.K; ++k) {
        if (class_pos0) class_pos0[k] = g.cls[k].pos0;
        if (class_n) class_n[k] = g.cls[k].n;
        if (class_slice0) class_slice0[k] = g.cls[k].slice0;
    }
    return SG_OK;
}
