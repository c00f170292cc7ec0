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

// O2b: random regular bipartite graph of degree 4: four perfect matchings between half
// A = {0..H-1} and half B = {H..N-1}, H = N/2, no pair matched twice.  DESIGN.md O2b fixes the draw: candidate number t
// (t = 0, 1, 2, ... over all four matchings) is the identity run through the swap sequence
//   position H-1-n  <->  position (x_n * (H-n)) >> 32,   n = 0 .. H-2,   x_n = word n&3 of P(n>>2, t, 0, tag 4),
// and a candidate is kept if no A-vertex gets a partner it already has.  Edge e = a*H + i joins i and H + m_a(i).
namespace {
// the swap targets of candidate t, one Philox block per four consecutive swaps
void rrbg_swap_targets(uint64_t H, uint64_t t, uint32_t k0, uint32_t k1, std::vector<uint32_t> &target)
{
    target.resize(H > 0 ? H - 1 : 0);
    for (uint64_t n0 = 0; n0 + 1 < H; n0 += 4) {
        const Philox4 blk = sg_philox_host((uint32_t)(n0 >> 2), (uint32_t)t, 0u, 4u << 24, k0, k1);
        for (uint64_t n = n0; n < std::min<uint64_t>(n0 + 4, H - 1); ++n)
            target[n] = (uint32_t)(((uint64_t)blk.x[n - n0] * (H - n)) >> 32);
    }
}
}  // namespace

static bool build_rrbg_edges(uint64_t N, uint64_t seed, VBHostGraph &g)
{
    if (N < 8 || (N & 1)) { sg_set_error("sg_create: the RRBG model needs an even N >= 8"); return false; }
    const uint64_t H = N / 2;
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    g.N = N; g.M = 4 * H;
    g.eu.resize(g.M); g.ev.resize(g.M);
    std::vector<uint32_t> partner(4 * H);          // partner[4 i + a] = B-index matched to A-vertex i by matching a
    std::vector<uint32_t> cand(H), target;
    uint32_t kept = 0;
    for (uint64_t t = 0; kept < 4; ++t) {
        rrbg_swap_targets(H, t, k0, k1, target);
        for (uint64_t i = 0; i < H; ++i) cand[i] = (uint32_t)i;
        for (uint64_t n = 0; n + 1 < H; ++n) std::swap(cand[H - 1 - n], cand[target[n]]);
        bool fresh = true;
        for (uint64_t i = 0; i < H && fresh; ++i)
            for (uint32_t a = 0; a < kept; ++a)
                if (partner[4 * i + a] == cand[i]) { fresh = false; break; }
        if (!fresh) continue;
        for (uint64_t i = 0; i < H; ++i) {
            partner[4 * i + kept] = cand[i];
            g.eu[(uint64_t)kept * H + i] = (uint32_t)i;
            g.ev[(uint64_t)kept * H + i] = (uint32_t)(H + cand[i]);
        }
        ++kept;
    }
    return true;
}

// O2c: random regular graph of degree 4, not bipartite, by the pairing model (O2c): the
// 4N half-edges ("points", point q on vertex q/4) are shuffled -- candidate t applies, to the identity, the swaps
//   position 4N-1-n  <->  position (x_n * (4N-n)) >> 32,   n = 0 .. 4N-2,   x_n = word n&3 of P(n>>2, t, 0, tag 5)
// -- and read off in consecutive pairs; the first candidate that is a simple graph is taken.  Edge k joins the vertices of
// the points at positions 2k and 2k+1.
static bool build_rrg_edges(uint64_t N, uint64_t seed, VBHostGraph &g)
{
    if (N < 8 || N >= (1ull << 30)) { sg_set_error("sg_create: the RRG model needs 8 <= N < 2^30"); return false; }
    const uint64_t Q = 4 * N, M = 2 * N;
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    g.N = N; g.M = M;
    g.eu.resize(M); g.ev.resize(M);
    std::vector<uint32_t> point(Q);
    std::vector<uint64_t> keys(M);
    for (uint64_t t = 0;; ++t) {
        std::iota(point.begin(), point.end(), 0u);
        for (uint64_t n0 = 0; n0 + 1 < Q; n0 += 4) {
            const Philox4 blk = sg_philox_host((uint32_t)(n0 >> 2), (uint32_t)t, 0u, 5u << 24, k0, k1);
            for (uint64_t n = n0; n < std::min<uint64_t>(n0 + 4, Q - 1); ++n)
                std::swap(point[Q - 1 - n], point[((uint64_t)blk.x[n - n0] * (Q - n)) >> 32]);
        }
        // simple <=> no pair inside one vertex and no two pairs on the same two vertices: sort the pair keys
        bool simple = true;
        for (uint64_t k = 0; k < M && simple; ++k) {
            const uint32_t u = point[2 * k] >> 2, v = point[2 * k + 1] >> 2;
            simple = u != v;
            keys[k] = u < v ? ((uint64_t)u << 32 | v) : ((uint64_t)v << 32 | u);
        }
        if (!simple) continue;
        std::sort(keys.begin(), keys.end());
        if (std::adjacent_find(keys.begin(), keys.end()) != keys.end()) continue;
        for (uint64_t k = 0; k < M; ++k) { g.eu[k] = point[2 * k] >> 2; g.ev[k] = point[2 * k + 1] >> 2; }
        return true;
    }
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

bool sg_build_vb_graph(int model, uint64_t N, double c, uint64_t seed, uint32_t n_words, VBHostGraph &g)
{
    if (model == SG_MODEL_RRBG ? !build_rrbg_edges(N, seed, g) : model == SG_MODEL_RRG ? !build_rrg_edges(N, seed, g) : !build_er_edges(N, c, seed, g))
        return false;
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
    // N-1 tree edges (half of all gathers at c = 4) walk through every other class's block monotonically: the
    // lanes of a warp share 128-byte lines and the lines are still in L1/L2 when the next slices need them.
    // The same forest fixes the gauge (see sg_internal.h): its edges need no coupling word.
    // (SG_VB_ORDER=label keeps the label order for the positions: a measurement knob; outputs are identical.)
    std::vector<uint32_t> bfs; bfs.reserve(N);
    std::vector<uint32_t> par(N, SG_NONE), par_e(N, SG_NONE);
    {
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
                    if (!seen[v]) { seen[v] = 1; par[v] = u; par_e[v] = g.adj_e[a]; bfs.push_back(v); }
                }
            }
        }
    }
    const char *order_env = std::getenv("SG_VB_ORDER");
    const bool label_order = order_env && !std::strcmp(order_env, "label");
    const char *gauge_env = std::getenv("SG_VB_GAUGE");
    g.gauge = !(gauge_env && !std::strcmp(gauge_env, "0"));                 // measurement knob: keep every coupling word
    // per site: tree entries nT (parent + children); the others are X entries
    std::vector<uint8_t> nT(N, 0);
    if (g.gauge)
        for (uint64_t i = 0; i < N; ++i)
            if (par[i] != SG_NONE) { nT[i]++; nT[par[i]]++; }
    std::vector<uint64_t> ccount(K, 0);
    for (uint64_t i = 0; i < N; ++i) ccount[g.colour[i]]++;
    auto shape_of = [&](uint32_t i) { return sg_vb_shape((uint32_t)(g.row_ptr[i + 1] - g.row_ptr[i]) - nT[i], nT[i]); };
    const char *dem_env = std::getenv("SG_VB_DEMAND");                      // measurement knob: 0 = sort by shape only
    const bool use_demand = !(dem_env && !std::strcmp(dem_env, "0"));
    const uint64_t demand2_div = (dem_env && !std::strcmp(dem_env, "2")) ? (1ull << 40) : 4;      // "2": only the two smaller brackets
    auto bucket_of = [&](uint32_t i) {
        uint32_t demand = 3;
        if (use_demand)
            for (uint64_t a = g.row_ptr[i]; a < g.row_ptr[i + 1]; ++a) {
                const uint64_t nk = ccount[g.colour[g.adj[a]]];
                demand = std::min(demand, nk * 32 < N ? 0u : nk * 8 < N ? 1u : nk * demand2_div < N ? 2u : 3u);
            }
        return demand * 3 + shape_of(i);
    };
    const char *win_env = std::getenv("SG_VB_WIN");                         // measurement knob: 0 = no sort
    const uint64_t win = win_env ? (uint64_t)std::max(0, std::atoi(win_env)) : 4096;
    // positions: (class, window of the breadth-first index, shape, breadth-first index)
    g.cls.assign(K, VBClass{});
    {
        uint64_t p0 = 0;
        for (uint32_t k = 0; k < K; ++k) { g.cls[k].pos0 = p0; g.cls[k].n = ccount[k]; p0 += ccount[k]; }
    }
    g.orig.resize(N); g.pos.resize(N);
    {
        std::vector<uint64_t> fill(K);
        for (uint32_t k = 0; k < K; ++k) fill[k] = g.cls[k].pos0;
        if (label_order) for (uint64_t i = 0; i < N; ++i) g.orig[fill[g.colour[i]]++] = (uint32_t)i;
        else for (uint64_t q = 0; q < N; ++q) g.orig[fill[g.colour[bfs[q]]]++] = bfs[q];
        // Buckets: every window of `win` consecutive sites of a class (in the order above) is stably sorted by
        // (demand, shape).  demand: 0 = the site has a neighbour in a class of fewer than N/32 sites, 1 = in a class
        // of fewer than N/8 sites, 2 = of fewer than N/4 sites, 3 = none of these: the smaller classes gather from a
        // part of the sites only, and with those packed together their gathers use whole 128-byte lines and a smaller
        // part of L2.  shape (sg_vb_shape): 0 = at
        // most 2 X and 2 T entries, 1 = at most 4 and 4, 2 = longer rows: almost every slice then holds sites of one
        // shape and the kernels run the count that fits it.  The breadth-first order survives inside each run.
        if (win > 1) {
            std::vector<uint32_t> tmp(win);
            for (uint32_t k = 0; k < K; ++k)
                for (uint64_t a = g.cls[k].pos0, end = a + g.cls[k].n; a < end; a += win) {
                    const uint64_t len = std::min<uint64_t>(win, end - a);
                    uint64_t at[13] = {0};
                    for (uint64_t q = 0; q < len; ++q) at[bucket_of(g.orig[a + q]) + 1]++;
                    for (int b = 0; b < 12; ++b) at[b + 1] += at[b];
                    for (uint64_t q = 0; q < len; ++q) tmp[at[bucket_of(g.orig[a + q])]++] = g.orig[a + q];
                    std::copy(tmp.begin(), tmp.begin() + len, g.orig.begin() + a);
                }
        }
        for (uint64_t p = 0; p < N; ++p) g.pos[g.orig[p]] = (uint32_t)p;
    }
    g.tpar.assign(N, SG_NONE); g.teid.assign(N, SG_NONE);
    g.bfs_pos.resize(N);
    for (uint64_t q = 0; q < N; ++q) g.bfs_pos[q] = g.pos[bfs[q]];
    std::vector<uint32_t>().swap(bfs);
    for (uint64_t p = 0; p < N; ++p) {
        const uint32_t i = g.orig[p];
        if (par[i] != SG_NONE) { g.tpar[p] = g.pos[par[i]]; g.teid[p] = par_e[i]; }
    }
    // per-class entry budgets (sg_internal.h): the smallest budget the kernels are compiled for whose greedy cut needs at
    // most 30 % more slices than the largest budget's (measured: the small budget's 12 resident CTAs per SM beat the large
    // budget's fuller slices up to there)
    // (SG_VB_IT=<it> forces one budget for all classes: a measurement knob; outputs are identical)
    const char *it_env = std::getenv("SG_VB_IT");
    const char *slack_env = std::getenv("SG_VB_SLACK");                     // measurement knob: the percentage above
    const uint64_t slack_pct = slack_env ? (uint64_t)std::atoi(slack_env) : 130;
    auto count_slices = [&](uint32_t k, VBBudget bud) {
        uint64_t ns = 0, p = g.cls[k].pos0;
        const uint64_t pend = p + g.cls[k].n;
        while (p < pend) {
            uint32_t n = 0, sE = 0, sX = 0;
            while (p < pend && n < 32) {
                const uint32_t i = g.orig[p];
                const uint32_t d = (uint32_t)(g.row_ptr[i + 1] - g.row_ptr[i]), x = d - nT[i];
                if (n > 0 && (sE + d > 32 * bud.it || sX + x > 32 * bud.itx)) break;
                sE += d; sX += x; ++n; ++p;
            }
            ++ns;
        }
        return ns;
    };
    g.it_max = g.itx_max = 0;
    for (uint32_t k = 0; k < K; ++k) {
        const uint32_t G = sg_vb_group(n_words);
        VBBudget best = G == 4 ? SG_VB_BUDGET_G4 : SG_VB_BUDGET_G2;
        if (G == 1) {
            constexpr size_t NB = sizeof(SG_VB_BUDGETS_G1) / sizeof(SG_VB_BUDGETS_G1[0]);
            best = SG_VB_BUDGETS_G1[NB - 1];
            const uint64_t fewest = count_slices(k, best);
            for (size_t b = 0; b + 1 < NB; ++b)
                if (count_slices(k, SG_VB_BUDGETS_G1[b]) * 100 <= fewest * slack_pct) { best = SG_VB_BUDGETS_G1[b]; break; }
            if (it_env)
                for (const VBBudget bud : SG_VB_BUDGETS_G1)
                    if ((uint32_t)std::atoi(it_env) == bud.it) best = bud;
        }
        g.cls[k].it = best.it; g.cls[k].itx = best.itx;
        g.it_max = std::max(g.it_max, best.it); g.itx_max = std::max(g.itx_max, best.itx);
    }
    // slices: greedy runs of <= 32 positions of one class within the class's budgets
    g.hdr.clear(); g.orig_s.clear(); g.rp_s.clear();
    g.col.clear(); g.col.reserve(2 * M); g.jeid.clear();
    std::vector<uint32_t> rowT, rowX;            // the slice's T entries are appended after its X entries
    std::vector<uint32_t> rowXe;
    for (uint32_t k = 0; k < K; ++k) {
        g.cls[k].slice0 = g.hdr.size();
        uint64_t p = g.cls[k].pos0;
        const uint64_t pend = p + g.cls[k].n;
        const uint32_t capE = 32 * g.cls[k].it, capX = 32 * g.cls[k].itx;
        while (p < pend) {
            SGHdr h{(uint32_t)p, (uint32_t)g.col.size(), (uint32_t)g.jeid.size(), 0u};
            uint32_t n = 0, sT = 0, sX = 0, shape = 0;
            rowT.clear(); rowX.clear(); rowXe.clear();
            const size_t base = g.orig_s.size();
            g.orig_s.resize(base + 32, SG_NONE); g.rp_s.resize(base + 32, 0u);
            while (p < pend && n < 32) {
                const uint32_t i = g.orig[p];
                const uint32_t d = (uint32_t)(g.row_ptr[i + 1] - g.row_ptr[i]), t = nT[i], x = d - t;
                if (n > 0 && (sT + sX + d > capE || sX + x > capX)) break;
                // tree entries: parent first, then children by position; other entries by position
                uint64_t keyT[32], keyX[32];
                uint32_t cT = 0, cX = 0;
                for (uint64_t a = g.row_ptr[i]; a < g.row_ptr[i + 1]; ++a) {
                    const uint32_t v = g.adj[a], e = g.adj_e[a];
                    const uint64_t key = (uint64_t)g.pos[v] << 32 | e;
                    if (g.gauge && par_e[i] == e) { std::memmove(keyT + 1, keyT, cT * sizeof(uint64_t)); keyT[0] = key; cT++; }
                    else if (g.gauge && par_e[v] == e) keyT[cT++] = key;
                    else keyX[cX++] = key;
                }
                std::sort(keyT + ((g.gauge && par_e[i] != SG_NONE) ? 1 : 0), keyT + cT);
                std::sort(keyX, keyX + cX);
                g.orig_s[base + n] = i;
                g.rp_s[base + n] = sX | sT << 8 | cX << 17 | cT << 22;          // tOff is made absolute below
                for (uint32_t q = 0; q < cT; ++q) rowT.push_back((uint32_t)(keyT[q] >> 32));
                for (uint32_t q = 0; q < cX; ++q) { rowX.push_back((uint32_t)(keyX[q] >> 32)); rowXe.push_back((uint32_t)keyX[q]); }
                shape = std::max(shape, sg_vb_shape(cX, cT));
                sT += cT; sX += cX; ++n; ++p;
            }
            for (uint32_t j = 0; j < n; ++j) g.rp_s[base + j] += sX << 8;       // T entries follow the slice's X entries
            h.counts = n | sX << 6 | (sT + sX) << 16 | shape << 28;
            g.hdr.push_back(h);
            g.col.insert(g.col.end(), rowX.begin(), rowX.end());
            g.col.insert(g.col.end(), rowT.begin(), rowT.end());
            g.jeid.insert(g.jeid.end(), rowXe.begin(), rowXe.end());
            if (g.col.size() >= (1ull << 32)) { sg_set_error("sg_create: instance too large for 32-bit entry indices"); return false; }
        }
        g.cls[k].nslices = g.hdr.size() - g.cls[k].slice0;
    }
    g.hdr.push_back(SGHdr{(uint32_t)N, (uint32_t)g.col.size(), (uint32_t)g.jeid.size(), 0u});
    return true;
}

uint32_t sg_vb_group(uint32_t n_words)
{
    // two words (16-byte accesses) whenever n_words is even: measured 25-30 % faster than four words per thread, whose 96
    // registers leave 20 warps per SM (profiles/r02_sweep.md)
    uint32_t G = n_words % 2 == 0 ? 2u : 1u;
    if (const char *e = std::getenv("SG_VB_G")) {
        const uint32_t want = (uint32_t)std::atoi(e);
        if ((want == 1 || want == 2 || want == 4) && n_words % want == 0) G = want;
    }
    return G;
}

// ---- host-only C entry points (include/sg.h) ------------------------------------------------------
struct sg_host_graph { VBHostGraph g; };

extern "C" void sg_host_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t *out)
{
    const Philox4 x = sg_philox_host(c0, c1, c2, c3, k0, k1);
    for (int q = 0; q < 4; ++q) out[q] = x.x[q];
}

extern "C" sg_host_graph *sg_host_graph_create(int model, uint64_t N, double c, uint64_t seed, uint32_t n_words)
{
    if (model != SG_MODEL_VB && model != SG_MODEL_RRBG && model != SG_MODEL_RRG) { sg_set_error("sg_host_graph_create: graph model required"); return nullptr; }
    if (N < 2 || N >= (1ull << 31) - 2) { sg_set_error("sg_host_graph_create: N must satisfy 2 <= N < 2^31 - 2"); return nullptr; }
    if (n_words == 0) { sg_set_error("sg_host_graph_create: n_words must be >= 1"); return nullptr; }
    sg_host_graph *h = new sg_host_graph();
    if (!sg_build_vb_graph(model, N, c, seed, n_words, h->g)) { delete h; return nullptr; }
    return h;
}

extern "C" void sg_host_graph_destroy(sg_host_graph *g) { delete g; }

extern "C" int sg_host_graph_info(const sg_host_graph *h, uint64_t *info)
{
    if (!h || !info) return SG_EINVAL;
    const VBHostGraph &g = h->g;
    info[0] = g.M; info[1] = g.K; info[2] = g.dmax; info[3] = g.col.size();
    info[4] = g.hdr.size() - 1; info[5] = g.N; info[6] = g.jeid.size(); info[7] = g.it_max; info[8] = g.gauge ? 1 : 0;
    return SG_OK;
}

extern "C" int sg_host_graph_get(const sg_host_graph *h, uint32_t *u, uint32_t *v, uint32_t *colour, uint32_t *orig,
                                 uint32_t *hdr, uint32_t *orig_s, uint32_t *rp_s, uint32_t *col, uint32_t *jeid,
                                 uint32_t *tpar, uint32_t *teid, uint32_t *bfs_pos,
                                 uint64_t *class_pos0, uint64_t *class_n, uint64_t *class_slice0, uint64_t *class_nslices,
                                 uint64_t *class_it, uint64_t *class_itx)
{
    if (!h) return SG_EINVAL;
    const VBHostGraph &g = h->g;
    if (u) std::copy(g.eu.begin(), g.eu.end(), u);
    if (v) std::copy(g.ev.begin(), g.ev.end(), v);
    if (colour) std::copy(g.colour.begin(), g.colour.end(), colour);
    if (orig) std::copy(g.orig.begin(), g.orig.end(), orig);
    if (hdr) std::memcpy(hdr, g.hdr.data(), g.hdr.size() * sizeof(SGHdr));
    if (orig_s) std::copy(g.orig_s.begin(), g.orig_s.end(), orig_s);
    if (rp_s) std::copy(g.rp_s.begin(), g.rp_s.end(), rp_s);
    if (col) std::copy(g.col.begin(), g.col.end(), col);
    if (jeid) std::copy(g.jeid.begin(), g.jeid.end(), jeid);
    if (tpar) std::copy(g.tpar.begin(), g.tpar.end(), tpar);
    if (teid) std::copy(g.teid.begin(), g.teid.end(), teid);
    if (bfs_pos) std::copy(g.bfs_pos.begin(), g.bfs_pos.end(), bfs_pos);
    for (uint32_t k = 0; k < g.K; ++k) {
        if (class_pos0) class_pos0[k] = g.cls[k].pos0;
        if (class_n) class_n[k] = g.cls[k].n;
        if (class_slice0) class_slice0[k] = g.cls[k].slice0;
        if (class_nslices) class_nslices[k] = g.cls[k].nslices;
        if (class_it) class_it[k] = g.cls[k].it;
        if (class_itx) class_itx[k] = g.cls[k].itx;
    }
    return SG_OK;
}
