// sg_host.cpp -- host side of sg_create: Philox, the seeded instance generator (row a1 of
// SURVEY.md section 8(a)), thresholds.  Conventions: DESIGN.md section 3 (O1, O2, O5, O6).
// Independent of oracle/: nothing here is shared with or derived from it.
#include <algorithm>
#include <cmath>
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

bool sg_build_vb_graph(uint64_t N, double c, uint64_t seed, VBHostGraph &g)
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
    {
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
    }
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
    // Positions: sites sorted by (colour, degree, original label).  Every (colour, degree) bucket starts
    // at a multiple of 32 positions; the gap positions are padding (orig = NONE, spin word 0, never
    // written), so a slice of 32 positions holds sites of ONE degree: no padded neighbour slots, and the
    // degree of a site is the slice's row length.
    const uint32_t DB = g.dmax + 1;
    std::vector<uint64_t> cnt((uint64_t)K * DB, 0), start((uint64_t)K * DB + 1, 0);
    for (uint64_t i = 0; i < N; ++i) cnt[(uint64_t)g.colour[i] * DB + (g.row_ptr[i + 1] - g.row_ptr[i])]++;
    for (size_t b = 0; b < cnt.size(); ++b) start[b + 1] = start[b] + ((cnt[b] + 31) / 32) * 32;
    const uint64_t P = start[cnt.size()];
    if (P >= (1ull << 31)) { sg_set_error("sg_create: too many sites"); return false; }
    g.P = P;
    g.cls.assign(K, VBClass{});
    for (uint32_t k = 0; k < K; ++k) {
        g.cls[k].pos0 = start[(uint64_t)k * DB];
        g.cls[k].n = start[(uint64_t)(k + 1) * DB] - start[(uint64_t)k * DB];
    }
    g.orig.assign(P, SG_NONE); g.pos.resize(N); g.deg.assign(P, 0);
    for (uint32_t k = 0; k < K; ++k)
        for (uint32_t d = 0; d < DB; ++d)
            for (uint64_t p = start[(uint64_t)k * DB + d]; p < start[(uint64_t)k * DB + d + 1]; ++p) g.deg[p] = (uint8_t)d;
    {
        std::vector<uint64_t> fill(start.begin(), start.end() - 1);
        for (uint64_t i = 0; i < N; ++i) {
            const uint64_t p = fill[(uint64_t)g.colour[i] * DB + (g.row_ptr[i + 1] - g.row_ptr[i])]++;
            g.orig[p] = (uint32_t)i; g.pos[i] = (uint32_t)p;
        }
    }
    // sliced ELL: slice s of the whole position space = positions 32 s .. 32 s + 31, row length deg[32 s]
    const uint64_t nslices = P / 32;
    g.slice_ptr.assign(nslices + 1, 0);
    for (uint64_t s = 0; s < nslices; ++s) {
        const uint64_t next = (uint64_t)g.slice_ptr[s] + g.deg[32 * s];
        if (next > 0x7FFFFFFull) { sg_set_error("sg_create: instance too large for 32-bit entry indices"); return false; }
        g.slice_ptr[s + 1] = (uint32_t)next;
    }
    for (uint32_t k = 0; k < K; ++k) { g.cls[k].slice0 = g.cls[k].pos0 / 32; g.cls[k].nslices = g.cls[k].n / 32; }
    const uint64_t entries = 32ull * g.slice_ptr[nslices];
    g.col.resize(entries); g.eid.assign(entries, SG_NONE);
    g.entry_of_edge.assign(M, 0);
    for (uint64_t s = 0; s < nslices; ++s) {
        const uint64_t base = 32ull * g.slice_ptr[s];
        const uint32_t D = g.slice_ptr[s + 1] - g.slice_ptr[s];
        for (uint32_t j = 0; j < 32; ++j) {
            const uint64_t p = 32 * s + j;
            const uint32_t i = g.orig[p];
            for (uint32_t q = 0; q < D; ++q) {
                const uint64_t ent = base + 32ull * q + j;
                if (i != SG_NONE) {
                    const uint64_t r0 = g.row_ptr[i];
                    g.col[ent] = g.pos[g.adj[r0 + q]];
                    const uint32_t e = g.adj_e[r0 + q];
                    g.eid[ent] = e;
                    if (g.eu[e] == i) g.entry_of_edge[e] = (uint32_t)ent;
                } else {
                    g.col[ent] = (uint32_t)p;   // padding position: points at itself, coupling word 0
                }
            }
        }
    }
    // tiles for the staged sweep kernel: consecutive slices of one class, at most SG_TILE_SLICES slices
    // and SG_TILE_ENT32 neighbour columns (32 entries each)
    g.tiles.clear();
    for (uint32_t k = 0; k < K; ++k) {
        g.cls[k].tile0 = g.tiles.size();
        uint64_t s = g.cls[k].slice0;
        const uint64_t send = s + g.cls[k].nslices;
        while (s < send) {
            VBTile t{g.slice_ptr[s], (uint32_t)(32 * s), 0};
            uint32_t ns = 0, cols = 0;
            while (s + ns < send && ns < SG_TILE_SLICES) {
                const uint32_t D = g.slice_ptr[s + ns + 1] - g.slice_ptr[s + ns];
                if (ns > 0 && cols + D > SG_TILE_ENT32) break;
                t.packed |= (uint64_t)D << (4 + 5 * ns);
                cols += D; ++ns;
            }
            t.packed |= ns;
            g.tiles.push_back(t);
            s += ns;
        }
        g.cls[k].ntiles = g.tiles.size() - g.cls[k].tile0;
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

extern "C" sg_host_graph *sg_host_graph_create(uint64_t N, double c, uint64_t seed)
{
    if (N < 2 || N >= (1ull << 32)) { sg_set_error("sg_host_graph_create: N must satisfy 2 <= N < 2^32"); return nullptr; }
    sg_host_graph *h = new sg_host_graph();
    if (!sg_build_vb_graph(N, c, seed, h->g)) { delete h; return nullptr; }
    return h;
}

extern "C" void sg_host_graph_destroy(sg_host_graph *g) { delete g; }

extern "C" int sg_host_graph_info(const sg_host_graph *h, uint64_t *info)
{
    if (!h || !info) return SG_EINVAL;
    info[0] = h->g.M; info[1] = h->g.K; info[2] = h->g.dmax; info[3] = h->g.col.size();
    info[4] = h->g.slice_ptr.size() - 1; info[5] = h->g.N; info[6] = h->g.P; info[7] = h->g.tiles.size();
    return SG_OK;
}

extern "C" int sg_host_graph_get(const sg_host_graph *h, uint32_t *u, uint32_t *v, uint32_t *colour, uint32_t *orig,
                                 uint32_t *deg, uint32_t *slice_ptr, uint32_t *col, uint32_t *eid,
                                 uint64_t *class_pos0, uint64_t *class_n, uint64_t *class_slice0, uint64_t *tiles)
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
    if (tiles) std::memcpy(tiles, g.tiles.data(), g.tiles.size() * sizeof(VBTile));
    if (tiles) std::memcpy(tiles, g.tiles.data(), g.tiles.size() * sizeof(VBTile));
    return SG_OK;
}
