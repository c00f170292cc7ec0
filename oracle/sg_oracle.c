/*
 * sg_oracle.c -- THE ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, single-threaded, obviously-correct CPU statement of what the
 * hot path of arXiv:1906.11195 computes, in the conventions of DESIGN.md §3
 * (which restate SURVEY.md §8(c) O1-O10).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load this file's
 * library.  It shares no code, header, table or helper with the CUDA path
 * (paper_1906_11195_b200/csrc): both sides restate the same written spec.
 *
 * What it follows, passage by passage:
 *   - VB Hamiltonian H = -sum_{(ij) in E} J_ij s_i s_j, J = +-1     PAPER.md:73-75 (Eq. 3)
 *   - SK Hamiltonian H = -sum_{i<j} J_ij s_i s_j, binary J=+-1/sqrt N PAPER.md:43 (Eq. 1), :233
 *   - "classic single spin flip Metropolis ... fixed temperature ... taking the
 *     update of the whole graph as unit of time", random start
 *   - SK: "N single spin updates, performed in a fixed order"
 *   - parallel update needs a partition with no internal edges
 *     (here: first-fit colour classes, reading Q1/Q4)
 *   - 64 samples per word share the graph, independent couplings and
 *     initial spins
 *   - C(t,t') = (1/N) sum_i s_i(t) s_i(t')
 *   - energy and correlations are the observables
 *   - model 2 (RRBG): the same Hamiltonian on a bipartite random regular graph of
 *     degree 4, the paper's own ensemble
 *   - model 3 (RRG): ... on a random regular graph of degree 4, not bipartite: the
 *     ensemble of the main text, which Fig. S3 shows to be equivalent
 *
 * Representation: spins are UNPACKED +-1 int8, one per (site, lane), in the
 * original site labels; every lane is updated on its own with explicit
 * integer arithmetic; no bit tricks, no blocking, no reordering beyond what the
 * spec states.  Coupling words are kept as drawn (O3) and read one bit at a
 * time through jbit().
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): Philox known answers (P1),
 * exact enumeration / Boltzmann (P3), full transition matrix and detailed
 * balance (P4), C(tw,tw)=1 (P5), energy bookkeeping (P6), T=0 (P7), T=inf
 * (P8), forced cases (P9), generator statistics (P10), paramagnet energy (P12),
 * SK small-N (P13), word offset / clones / aligned start (P15).  Unpinned by the
 * paper: the numerical values of C(tw,tw+t) themselves (no number is printed;
 * see DESIGN.md).
 *
 * Options (or_create_opt; readings Q24-Q26), all neutral at their defaults:
 *   word0    the handle simulates words word0 .. word0+W-1 of the instance: every
 *            Philox counter that takes a word index takes word0 + w (Q16: words
 *            are independent given the graph, so a W-word run is W one-word runs)
 *   clones   SK: "two clones (i.e. replicas with the same
 *            couplings)": clone c shares the coupling words of word w and draws
 *            its initial spins and its Metropolis uniforms as the virtual word
 *            w + c * 2^20 (Q25)
 *   aligned  PAPER.md:231: "the initial configuration has all the spins
 *            aligned": every spin +1 at t = 0 (Q26)
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

#define OR_VB 0
#define OR_SK 1
#define OR_RRBG 2   /* VB Hamiltonian on a random regular bipartite graph of degree 4 */
#define OR_RRG 3    /* ... on a random regular graph of degree 4, not bipartite (Fig. S3) */
#define OR_MAX_SLOTS 64

typedef struct or_sim {
    int       model;
    uint64_t  N, M;
    uint32_t  W;        /* words per site; lanes L = 64*W */
    uint64_t  L;
    double    T;
    uint64_t  seed;
    uint64_t  sweep;    /* number of completed sweeps */
    /* VB graph, original labels */
    uint32_t *eu, *ev;  /* edge e = (eu[e], ev[e]) in acceptance order (O2) */
    uint64_t *row_ptr;  /* N+1 */
    uint32_t *adj;      /* 2M neighbour labels */
    uint64_t *adj_e;    /* 2M edge ids */
    uint32_t *colour;   /* N */
    uint32_t  K;        /* number of colours */
    uint32_t  dmax;
    /* couplings: VB kappa[e*W+w]; SK kappa[pair(i,j)*W+w], i<j */
    uint64_t *kappa;
    /* thresholds: VB thr[k], k=0..dmax ; SK thr[m], m=0..N-1 (index 0 unused) */
    uint64_t *thr;
    uint64_t  nthr;
    int8_t   *s;        /* N*L spins, s[i*L + lane] = +1 / -1 */
    int8_t   *slot[OR_MAX_SLOTS];
    int64_t  *dE;       /* per-lane accumulated energy change (VB: units of J; SK: numerator) */
    uint64_t *nflip;    /* per-lane number of accepted flips in the last sweep */
    uint32_t  word0;    /* first word of the instance this handle simulates */
    uint32_t  clones;   /* replicas sharing the couplings: lane = c*64*W + 64*w + b */
    int       aligned;  /* all spins +1 initially */
} or_sim;

#define OR_CLONE_STRIDE (1u << 20)   /* virtual word of clone c of word w: w + c * 2^20 */

/* word index that the Philox counters of spins and uniforms use for lane group (clone c, word w) */
static uint32_t virtual_word(const or_sim *h, uint32_t c, uint32_t w)
{
    return h->word0 + w + c * OR_CLONE_STRIDE;
}

/* ------------------------------------------------------------------ O1 */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 10 rounds of
 *   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
 * with the key bumped by (0x9E3779B9, 0xBB67AE85) between rounds. */
void or_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
               uint32_t k0, uint32_t k1, uint32_t out[4])
{
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* P(c0, c1, sweep, tag): counter layout of O1.  c2 = sweep low 32 bits,
 * c3 = tag<<24 | sweep>>32 ; key = (seed low, seed high). */
static void P(const or_sim *h, uint32_t c0, uint32_t c1, uint64_t sweep, uint32_t tag,
              uint32_t out[4])
{
    or_philox(c0, c1, (uint32_t)(sweep & 0xFFFFFFFFu),
              (tag << 24) | (uint32_t)(sweep >> 32),
              (uint32_t)(h->seed & 0xFFFFFFFFu), (uint32_t)(h->seed >> 32), out);
}

/* ------------------------------------------------------------------ O6 */
static uint64_t threshold(double arg_numer, double denom)
{
    /* floor(2^32 * exp(-numer/denom)), kept in 64 bits (T=inf gives 2^32) */
    double p = exp(-arg_numer / denom);
    return (uint64_t)floor(ldexp(p, 32));
}

/* coupling sign of a stored coupling word for one lane: bit 1 <=> J = -1 (Q14) */
static int jbit(const uint64_t *kappa_words, uint64_t lane)
{
    uint64_t word = kappa_words[lane >> 6];
    return ((word >> (lane & 63)) & 1u) ? -1 : +1;
}
/* the clones of a word share its couplings: coupling lane of lane l = l mod 64*W */
#define CL(h, lane) ((lane) % (64ull * (h)->W))

static uint64_t sk_pair(uint64_t N, uint64_t i, uint64_t j)
{
    /* index of the unordered pair i<j in row-major upper-triangular order */
    return i * N - i * (i + 1) / 2 + (j - i - 1);
}

/* ---------------------------------------------------------------- build */
static int build_csr_colour_thr(or_sim *h)
{
    uint64_t N = h->N, M = h->M;
    h->row_ptr = (uint64_t *)calloc(N + 1, sizeof(uint64_t));
    h->adj = (uint32_t *)malloc((2 * M + 1) * sizeof(uint32_t));
    h->adj_e = (uint64_t *)malloc((2 * M + 1) * sizeof(uint64_t));
    h->colour = (uint32_t *)malloc(N * sizeof(uint32_t));
    if (!h->row_ptr || !h->adj || !h->adj_e || !h->colour) return -1;
    uint64_t *deg = (uint64_t *)calloc(N, sizeof(uint64_t));
    for (uint64_t e = 0; e < M; ++e) { deg[h->eu[e]]++; deg[h->ev[e]]++; }
    h->dmax = 0;
    for (uint64_t i = 0; i < N; ++i) {
        h->row_ptr[i + 1] = h->row_ptr[i] + deg[i];
        if (deg[i] > h->dmax) h->dmax = (uint32_t)deg[i];
        deg[i] = 0;
    }
    /* rows list the incident edges in increasing edge id */
    for (uint64_t e = 0; e < M; ++e) {
        uint32_t u = h->eu[e], v = h->ev[e];
        h->adj[h->row_ptr[u] + deg[u]] = v; h->adj_e[h->row_ptr[u] + deg[u]] = e; deg[u]++;
        h->adj[h->row_ptr[v] + deg[v]] = u; h->adj_e[h->row_ptr[v] + deg[v]] = e; deg[v]++;
    }
    free(deg);
    /* O5: first-fit colouring in natural order */
    h->K = 0;
    uint8_t *used = (uint8_t *)malloc((size_t)h->dmax + 2);
    for (uint64_t i = 0; i < N; ++i) {
        memset(used, 0, (size_t)h->dmax + 2);
        for (uint64_t a = h->row_ptr[i]; a < h->row_ptr[i + 1]; ++a) {
            uint32_t j = h->adj[a];
            if (j < i && h->colour[j] <= h->dmax) used[h->colour[j]] = 1;
        }
        uint32_t col = 0;
        while (used[col]) col++;
        h->colour[i] = col;
        if (col + 1 > h->K) h->K = col + 1;
    }
    free(used);
    /* O6 */
    h->nthr = (uint64_t)h->dmax + 1;
    h->thr = (uint64_t *)calloc(h->nthr, sizeof(uint64_t));
    for (uint32_t k = 1; k <= h->dmax; ++k)
        h->thr[k] = threshold((double)(2 * (int)k), h->T);
    return 0;
}

static int alloc_state(or_sim *h)
{
    if (h->clones == 0) h->clones = 1;
    h->L = 64ull * h->W * h->clones;
    h->s = (int8_t *)malloc(h->N * h->L);
    h->dE = (int64_t *)calloc(h->L, sizeof(int64_t));
    h->nflip = (uint64_t *)calloc(h->L, sizeof(uint64_t));
    return (h->s && h->dE && h->nflip) ? 0 : -1;
}

void or_destroy(or_sim *h)
{
    if (!h) return;
    free(h->eu); free(h->ev); free(h->row_ptr); free(h->adj); free(h->adj_e);
    free(h->colour); free(h->kappa); free(h->thr); free(h->s); free(h->dE); free(h->nflip);
    for (int k = 0; k < OR_MAX_SLOTS; ++k) free(h->slot[k]);
    free(h);
}

/* O4: initial spins.  bit 1 <=> s = -1 */
static void draw_initial_spins(or_sim *h)
{
    for (uint64_t i = 0; i < h->N; ++i)
        for (uint32_t c = 0; c < h->clones; ++c)
            for (uint32_t w = 0; w < h->W; ++w) {
                uint32_t x[4];
                P(h, (uint32_t)i, virtual_word(h, c, w), 0, 1, x);
                uint64_t sigma = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
                for (int b = 0; b < 64; ++b)
                    h->s[i * h->L + 64ull * (c * h->W + w) + b] = (!h->aligned && ((sigma >> b) & 1u)) ? -1 : +1;
            }
}

or_sim *or_create_opt(int model, uint64_t N, double c, double T, uint64_t seed, uint32_t n_words,
                      uint32_t word0, uint32_t clones, int aligned)
{
    if (N < 2 || N >= (1ull << 32) || n_words == 0) return NULL;
    if (model != OR_VB && model != OR_SK && model != OR_RRBG && model != OR_RRG) return NULL;
    if (model == OR_RRG && (N < 8 || N >= (1ull << 30))) return NULL;
    if (model == OR_RRBG && (N < 8 || (N & 1))) return NULL;   /* two halves of N/2 >= 4 vertices */
    if (!(T >= 0.0)) return NULL;
    if (clones < 1 || clones > 2 || (clones > 1 && model != OR_SK)) return NULL;
    if ((uint64_t)word0 + n_words > OR_CLONE_STRIDE) return NULL;
    or_sim *h = (or_sim *)calloc(1, sizeof(or_sim));
    h->model = model; h->N = N; h->W = n_words; h->T = T; h->seed = seed; h->sweep = 0;
    h->word0 = word0; h->clones = clones; h->aligned = aligned;
    if (alloc_state(h)) { or_destroy(h); return NULL; }

    if (model == OR_RRBG) {
        /* O2b: random regular bipartite graph of degree 4, "all of them are in the same half of the lattice"
         * (PAPER.md:318), as the union of four permutations of one half onto the other without a repeated pair.
         * Halves A = {0..H-1}, B = {H..N-1}, H = N/2.  Permutation a = 0..3: attempts t = 0,1,2,... (one global
         * counter); an attempt is a Fisher-Yates shuffle of the identity, for i = H-1 down to 1:
         * j = (x*(i+1)) >> 32 with x = word n&3 of P(n>>2, t, 0, tag 4), n = H-1-i, swap(perm[i], perm[j]);
         * it is accepted if perm[i] differs from every earlier accepted permutation at every i.
         * Edge e = a*H + i joins i and H + perm_a[i]. */
        const uint64_t H = N / 2;
        h->M = 4 * H;
        h->eu = (uint32_t *)malloc((h->M + 1) * sizeof(uint32_t));
        h->ev = (uint32_t *)malloc((h->M + 1) * sizeof(uint32_t));
        uint32_t *perm = (uint32_t *)malloc(H * sizeof(uint32_t));
        uint64_t t = 0;
        for (uint32_t a = 0; a < 4; ++a) {
            for (;; ++t) {
                for (uint64_t i = 0; i < H; ++i) perm[i] = (uint32_t)i;
                uint32_t x[4] = {0, 0, 0, 0};
                for (uint64_t i = H - 1; i >= 1; --i) {
                    const uint64_t n = H - 1 - i;
                    if ((n & 3) == 0) P(h, (uint32_t)(n >> 2), (uint32_t)t, 0, 4, x);
                    const uint64_t j = ((uint64_t)x[n & 3] * (i + 1)) >> 32;
                    const uint32_t tmp = perm[i]; perm[i] = perm[j]; perm[j] = tmp;
                }
                int clash = 0;
                for (uint32_t b = 0; b < a && !clash; ++b)
                    for (uint64_t i = 0; i < H; ++i)
                        if (h->ev[(uint64_t)b * H + i] == (uint32_t)(H + perm[i])) { clash = 1; break; }
                if (!clash) { ++t; break; }
            }
            for (uint64_t i = 0; i < H; ++i) {
                h->eu[(uint64_t)a * H + i] = (uint32_t)i;
                h->ev[(uint64_t)a * H + i] = (uint32_t)(H + perm[i]);
            }
        }
        free(perm);
        h->model = OR_VB;   /* from here on: the VB Hamiltonian (Eq. 3) on this edge list */
        if (build_csr_colour_thr(h)) { or_destroy(h); return NULL; }
        const uint64_t M = h->M;
        h->kappa = (uint64_t *)malloc((M * h->W + 1) * sizeof(uint64_t));
        for (uint64_t f = 0; f < M; ++f)
            for (uint32_t w = 0; w < h->W; ++w) {
                uint32_t x[4];
                P(h, (uint32_t)f, h->word0 + w, 0, 2, x);
                h->kappa[f * h->W + w] = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
            }
    } else if (model == OR_RRG) {
        /* O2c (Q27): random regular graph of degree 4 ("random regular graphs with fixed degree
         * z = 4"; :262 Fig. S3 compares it with the bipartite one) by the pairing model: 4N points, point q belongs to
         * vertex q / 4; attempt t = 0, 1, 2, ... is a Fisher-Yates shuffle of the points, for i = 4N-1 down to 1:
         * j = (x * (i+1)) >> 32 with x = word n&3 of P(n>>2, t, 0, tag 5), n = 4N-1-i, swap(p[i], p[j]); the shuffled
         * points are paired (p[2k], p[2k+1]), k < 2N; the first attempt without a loop and without a repeated pair is
         * the graph (uniform over simple 4-regular graphs); edge k joins p[2k]/4 and p[2k+1]/4. */
        const uint64_t Q = 4 * N, M = 2 * N;
        h->M = M;
        h->eu = (uint32_t *)malloc((M + 1) * sizeof(uint32_t));
        h->ev = (uint32_t *)malloc((M + 1) * sizeof(uint32_t));
        uint32_t *pt = (uint32_t *)malloc(Q * sizeof(uint32_t));
        uint32_t *nbr = (uint32_t *)malloc(Q * sizeof(uint32_t));   /* up to 4 neighbours per vertex */
        uint8_t *cnt = (uint8_t *)malloc(N);
        for (uint64_t t = 0;; ++t) {
            for (uint64_t q = 0; q < Q; ++q) pt[q] = (uint32_t)q;
            uint32_t x[4] = {0, 0, 0, 0};
            for (uint64_t i = Q - 1; i >= 1; --i) {
                const uint64_t n = Q - 1 - i;
                if ((n & 3) == 0) P(h, (uint32_t)(n >> 2), (uint32_t)t, 0, 5, x);
                const uint64_t j = ((uint64_t)x[n & 3] * (i + 1)) >> 32;
                const uint32_t tmp = pt[i]; pt[i] = pt[j]; pt[j] = tmp;
            }
            memset(cnt, 0, N);
            int simple = 1;
            for (uint64_t k = 0; k < M && simple; ++k) {
                const uint32_t u = pt[2 * k] / 4, v = pt[2 * k + 1] / 4;
                if (u == v) { simple = 0; break; }
                for (uint32_t a = 0; a < cnt[u]; ++a)
                    if (nbr[4ull * u + a] == v) { simple = 0; break; }
                nbr[4ull * u + cnt[u]++] = v;
                nbr[4ull * v + cnt[v]++] = u;
                h->eu[k] = u; h->ev[k] = v;
            }
            if (simple) break;
        }
        free(pt); free(nbr); free(cnt);
        h->model = OR_VB;   /* from here on: the VB Hamiltonian (Eq. 3) on this edge list */
        if (build_csr_colour_thr(h)) { or_destroy(h); return NULL; }
        h->kappa = (uint64_t *)malloc((M * h->W + 1) * sizeof(uint64_t));
        for (uint64_t f = 0; f < M; ++f)
            for (uint32_t w = 0; w < h->W; ++w) {
                uint32_t x[4];
                P(h, (uint32_t)f, h->word0 + w, 0, 2, x);
                h->kappa[f * h->W + w] = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
            }
    } else if (model == OR_VB) {
        /* O2: G(N, M), M = floor(c N / 2 + 0.5); attempts a = 0,1,2,... */
        if (!(c >= 0.0)) { or_destroy(h); return NULL; }
        double pairs = 0.5 * (double)N * (double)(N - 1);
        uint64_t M = (uint64_t)floor(c * (double)N / 2.0 + 0.5);
        if ((double)M > pairs) { or_destroy(h); return NULL; }
        h->M = M;
        h->eu = (uint32_t *)malloc((M + 1) * sizeof(uint32_t));
        h->ev = (uint32_t *)malloc((M + 1) * sizeof(uint32_t));
        /* duplicate test by walking per-vertex chains of already accepted edges */
        int64_t *head = (int64_t *)malloc(N * sizeof(int64_t));
        int64_t *nxt = (int64_t *)malloc((2 * M + 1) * sizeof(int64_t));
        for (uint64_t i = 0; i < N; ++i) head[i] = -1;
        uint64_t e = 0;
        for (uint64_t a = 0; e < M; ++a) {
            uint32_t x[4];
            P(h, (uint32_t)(a & 0xFFFFFFFFu), (uint32_t)(a >> 32), 0, 3, x);
            uint32_t u = (uint32_t)(((uint64_t)x[0] * N) >> 32);
            uint32_t v = (uint32_t)(((uint64_t)x[1] * N) >> 32);
            if (u == v) continue;
            int dup = 0;
            for (int64_t q = head[u]; q >= 0; q = nxt[q]) {
                uint64_t f = (uint64_t)q >> 1;
                uint32_t other = ((uint64_t)q & 1u) ? h->eu[f] : h->ev[f];
                if (other == v) { dup = 1; break; }
            }
            if (dup) continue;
            h->eu[e] = u; h->ev[e] = v;
            nxt[2 * e] = head[u]; head[u] = (int64_t)(2 * e);        /* entry 2e: seen from eu, other = ev */
            nxt[2 * e + 1] = head[v]; head[v] = (int64_t)(2 * e + 1);/* entry 2e+1: seen from ev, other = eu */
            e++;
        }
        free(head); free(nxt);
        if (build_csr_colour_thr(h)) { or_destroy(h); return NULL; }
        /* O3 */
        h->kappa = (uint64_t *)malloc((M * h->W + 1) * sizeof(uint64_t));
        for (uint64_t f = 0; f < M; ++f)
            for (uint32_t w = 0; w < h->W; ++w) {
                uint32_t x[4];
                P(h, (uint32_t)f, h->word0 + w, 0, 2, x);
                h->kappa[f * h->W + w] = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
            }
    } else {
        if (N > 32768) { or_destroy(h); return NULL; }   /* Q22 */
        uint64_t pairs = N * (N - 1) / 2;
        h->M = pairs;
        h->kappa = (uint64_t *)malloc(pairs * h->W * sizeof(uint64_t));
        for (uint64_t i = 0; i < N; ++i)
            for (uint64_t j = i + 1; j < N; ++j)
                for (uint32_t w = 0; w < h->W; ++w) {
                    uint32_t x[4];
                    P(h, (uint32_t)j, h->word0 + w, i, 2, x);
                    h->kappa[sk_pair(N, i, j) * h->W + w] = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
                }
        h->nthr = N;
        h->thr = (uint64_t *)calloc(N, sizeof(uint64_t));
        for (uint64_t m = 1; m < N; ++m)
            h->thr[m] = threshold((double)(2 * (int64_t)m), h->T * sqrt((double)N));
    }
    draw_initial_spins(h);
    return h;
}

or_sim *or_create(int model, uint64_t N, double c, double T, uint64_t seed, uint32_t n_words)
{
    return or_create_opt(model, N, c, T, seed, n_words, 0, 1, 0);
}

/* Explicit VB instance for the pins: edges (u[e],v[e]), coupling words
 * kappa[e*W+w] (bit 1 <=> J=-1), initial spin words sigma[i*W+w]
 * (bit 1 <=> s=-1).  Colouring, thresholds and dynamics are the same code
 * as for or_create. */
or_sim *or_create_explicit(uint64_t N, uint64_t M, const uint32_t *u, const uint32_t *v,
                           const uint64_t *kappa, const uint64_t *sigma,
                           double T, uint64_t seed, uint32_t n_words)
{
    if (N < 1 || n_words == 0 || !(T >= 0.0)) return NULL;
    or_sim *h = (or_sim *)calloc(1, sizeof(or_sim));
    h->model = OR_VB; h->N = N; h->M = M; h->W = n_words; h->T = T; h->seed = seed;
    if (alloc_state(h)) { or_destroy(h); return NULL; }
    h->eu = (uint32_t *)malloc((M + 1) * sizeof(uint32_t));
    h->ev = (uint32_t *)malloc((M + 1) * sizeof(uint32_t));
    h->kappa = (uint64_t *)malloc((M * n_words + 1) * sizeof(uint64_t));
    for (uint64_t e = 0; e < M; ++e) {
        if (u[e] >= N || v[e] >= N || u[e] == v[e]) { or_destroy(h); return NULL; }
        h->eu[e] = u[e]; h->ev[e] = v[e];
    }
    memcpy(h->kappa, kappa, M * n_words * sizeof(uint64_t));
    if (build_csr_colour_thr(h)) { or_destroy(h); return NULL; }
    for (uint64_t i = 0; i < N; ++i)
        for (uint64_t lane = 0; lane < h->L; ++lane)
            h->s[i * h->L + lane] = ((sigma[i * n_words + (lane >> 6)] >> (lane & 63)) & 1u) ? -1 : +1;
    return h;
}

/* ------------------------------------------------------------ O7 / O8 */
/* Metropolis uniform of (site i, word w) in sweep t: r = x_{w&3} of
 * P(i, w>>2, t, tag 0); shared by the 64 lanes of the word (Q6). */
static uint32_t uniform_for(const or_sim *h, uint64_t i, uint32_t w, uint64_t t)
{
    /* w counts lane groups of 64: w = c*W + (word inside the handle) */
    uint32_t vw = virtual_word(h, w / h->W, w % h->W);
    uint32_t x[4];
    P(h, (uint32_t)i, vw >> 2, t, 0, x);
    return x[vw & 3];
}

static void vb_update_site(or_sim *h, uint64_t i, uint64_t t)
{
    uint64_t L = h->L;
    int64_t d = (int64_t)(h->row_ptr[i + 1] - h->row_ptr[i]);
    for (uint32_t w = 0; w < h->W * h->clones; ++w) {
        uint32_t r = uniform_for(h, i, w, t);
        for (int b = 0; b < 64; ++b) {
            uint64_t lane = 64ull * w + b;
            int64_t u = 0;   /* unsatisfied bonds: s_i s_j J = -1 */
            for (uint64_t a = h->row_ptr[i]; a < h->row_ptr[i + 1]; ++a) {
                uint64_t j = h->adj[a];
                int J = jbit(&h->kappa[h->adj_e[a] * h->W], CL(h, lane));
                if ((int)h->s[i * L + lane] * (int)h->s[j * L + lane] * J == -1) u++;
            }
            int64_t kk = d - 2 * u;          /* Delta E = 2*kk */
            if (kk <= 0 || (uint64_t)r < h->thr[kk]) {
                h->s[i * L + lane] = (int8_t)(-h->s[i * L + lane]);
                h->dE[lane] += 2 * kk;
                h->nflip[lane]++;
            }
        }
    }
}

static void sk_update_site(or_sim *h, uint64_t i, uint64_t t)
{
    uint64_t L = h->L, N = h->N;
    for (uint32_t w = 0; w < h->W * h->clones; ++w) {
        uint32_t r = uniform_for(h, i, w, t);
        for (int b = 0; b < 64; ++b) {
            uint64_t lane = 64ull * w + b;
            int64_t H = 0;                   /* integer local field, from scratch */
            for (uint64_t j = 0; j < N; ++j) {
                if (j == i) continue;
                uint64_t p = (i < j) ? sk_pair(N, i, j) : sk_pair(N, j, i);
                H += (int64_t)jbit(&h->kappa[p * h->W], CL(h, lane)) * (int64_t)h->s[j * L + lane];
            }
            int64_t m = (int64_t)h->s[i * L + lane] * H;   /* Delta E = 2 m / sqrt N */
            if (m <= 0 || (uint64_t)r < h->thr[m]) {
                h->s[i * L + lane] = (int8_t)(-h->s[i * L + lane]);
                h->dE[lane] += 2 * m;
                h->nflip[lane]++;
            }
        }
    }
}

int or_sweep(or_sim *h, uint64_t n)
{
    if (!h) return -1;
    for (uint64_t it = 0; it < n; ++it) {
        uint64_t t = h->sweep;
        memset(h->nflip, 0, h->L * sizeof(uint64_t));
        if (h->model == OR_VB) {
            for (uint32_t k = 0; k < h->K; ++k)
                for (uint64_t i = 0; i < h->N; ++i)
                    if (h->colour[i] == k) vb_update_site(h, i, t);
        } else {
            for (uint64_t i = 0; i < h->N; ++i) sk_update_site(h, i, t);
        }
        h->sweep = t + 1;
    }
    return 0;
}

/* VB only: the Metropolis update of the listed sites, in the listed order, at the current sweep index; the sweep
 * counter does not move.  A sweep is the composition of its site updates in colour-class order (O7), so a test can
 * let several ranks each update a part of a class and exchange the results. */
int or_vb_update_sites(or_sim *h, const uint32_t *sites, uint64_t n)
{
    if (!h || h->model != OR_VB) return -1;
    for (uint64_t q = 0; q < n; ++q) {
        if (sites[q] >= h->N) return -1;
        vb_update_site(h, sites[q], h->sweep);
    }
    return 0;
}

/* SK only: the updates of sites i0 .. i1-1 of the sweep with the current index, in order, on the current
 * configuration; the sweep counter does not move.  A sweep is the composition of its N site updates ("N
 * single spin updates, performed in a fixed order"), so tests can check a window of a very large instance: sites
 * below i0 already carry their new values, the others their old ones. */
int or_sk_update_range(or_sim *h, uint64_t i0, uint64_t i1)
{
    if (!h || h->model != OR_SK || i0 > i1 || i1 > h->N) return -1;
    for (uint64_t i = i0; i < i1; ++i) sk_update_site(h, i, h->sweep);
    return 0;
}

/* ------------------------------------------------------------------ O9 */
int or_snapshot(or_sim *h, uint32_t slot)
{
    if (!h || slot >= OR_MAX_SLOTS) return -1;
    if (!h->slot[slot]) h->slot[slot] = (int8_t *)malloc(h->N * h->L);
    if (!h->slot[slot]) return -2;
    memcpy(h->slot[slot], h->s, h->N * h->L);
    return 0;
}

/* out_counts[lane] = D_lane = #{ i : s_i(now) != s_i(slot) };  C = 1 - 2D/N */
int or_correlation(or_sim *h, uint32_t slot, uint64_t *out_counts)
{
    if (!h || slot >= OR_MAX_SLOTS || !h->slot[slot]) return -4;
    for (uint64_t lane = 0; lane < h->L; ++lane) {
        uint64_t D = 0;
        for (uint64_t i = 0; i < h->N; ++i)
            if (h->s[i * h->L + lane] != h->slot[slot][i * h->L + lane]) D++;
        out_counts[lane] = D;
    }
    return 0;
}

/* VB: E_lane = -sum_e J_e s_i s_j.   SK: E'_lane = -sum_{i<j} J'_ij s_i s_j (numerator; E = E'/sqrt N) */
int or_energy(or_sim *h, int64_t *out)
{
    if (!h) return -1;
    uint64_t L = h->L;
    for (uint64_t lane = 0; lane < L; ++lane) {
        int64_t E = 0;
        if (h->model == OR_VB) {
            for (uint64_t e = 0; e < h->M; ++e)
                E -= (int64_t)jbit(&h->kappa[e * h->W], CL(h, lane))
                   * (int64_t)h->s[(uint64_t)h->eu[e] * L + lane]
                   * (int64_t)h->s[(uint64_t)h->ev[e] * L + lane];
        } else {
            for (uint64_t i = 0; i < h->N; ++i)
                for (uint64_t j = i + 1; j < h->N; ++j)
                    E -= (int64_t)jbit(&h->kappa[sk_pair(h->N, i, j) * h->W], CL(h, lane))
                       * (int64_t)h->s[i * L + lane] * (int64_t)h->s[j * L + lane];
        }
        out[lane] = E;
    }
    return 0;
}

/* ------------------------------------------------------------- getters */
uint64_t or_sweep_count(const or_sim *h) { return h->sweep; }
uint64_t or_num_edges(const or_sim *h) { return h->M; }
uint32_t or_num_colours(const or_sim *h) { return h->K; }
uint32_t or_max_degree(const or_sim *h) { return h->dmax; }

/* packed spin words in original site order, word-minor: out[i*W+w], bit 1 <=> s=-1.
 * slot = -1: current configuration.  With clones: out[i*(W*clones) + c*W + w]. */
int or_get_spins(const or_sim *h, int32_t slot, uint64_t *out)
{
    const int8_t *src = h->s;
    if (slot >= 0) {
        if (slot >= OR_MAX_SLOTS || !h->slot[slot]) return -4;
        src = h->slot[slot];
    }
    const uint64_t G = h->L / 64;    /* lane groups per site: W * clones, clone-major */
    for (uint64_t i = 0; i < h->N; ++i)
        for (uint64_t w = 0; w < G; ++w) {
            uint64_t word = 0;
            for (int b = 0; b < 64; ++b)
                if (src[i * h->L + 64ull * w + b] < 0) word |= (1ull << b);
            out[i * G + w] = word;
        }
    return 0;
}

/* overwrite the current configuration from packed words (tests only) */
int or_set_spins(or_sim *h, const uint64_t *in)
{
    for (uint64_t i = 0; i < h->N; ++i)
        for (uint64_t lane = 0; lane < h->L; ++lane)
            h->s[i * h->L + lane] = ((in[i * (h->L / 64) + (lane >> 6)] >> (lane & 63)) & 1u) ? -1 : +1;
    return 0;
}

void or_set_sweep_count(or_sim *h, uint64_t t) { h->sweep = t; }

int or_get_graph(const or_sim *h, uint64_t *row_ptr, uint32_t *col, uint32_t *colour)
{
    if (h->model != OR_VB) return -1;
    memcpy(row_ptr, h->row_ptr, (h->N + 1) * sizeof(uint64_t));
    memcpy(col, h->adj, 2 * h->M * sizeof(uint32_t));
    memcpy(colour, h->colour, h->N * sizeof(uint32_t));
    return 0;
}

int or_get_edges(const or_sim *h, uint32_t *u, uint32_t *v)
{
    if (h->model != OR_VB) return -1;
    memcpy(u, h->eu, h->M * sizeof(uint32_t));
    memcpy(v, h->ev, h->M * sizeof(uint32_t));
    return 0;
}

/* VB: M*W words in edge order.  SK: N(N-1)/2*W words in pair order (i<j row-major). */
int or_get_couplings(const or_sim *h, uint64_t *out)
{
    memcpy(out, h->kappa, h->M * h->W * sizeof(uint64_t));
    return 0;
}

int or_get_thresholds(const or_sim *h, uint64_t *out, uint64_t n)
{
    for (uint64_t k = 0; k < n; ++k) out[k] = (k < h->nthr) ? h->thr[k] : 0;
    return 0;
}

int or_get_accumulated_dE(const or_sim *h, int64_t *out)
{
    memcpy(out, h->dE, h->L * sizeof(int64_t));
    return 0;
}

int or_get_last_flips(const or_sim *h, uint64_t *out)
{
    memcpy(out, h->nflip, h->L * sizeof(uint64_t));
    return 0;
}
