// sg_internal.h -- shared declarations of the CUDA path (host generator, kernels, C-ABI).
// Not part of the public interface; include/sg.h is.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "sg.h"

typedef struct CUstream_st *cudaStream_t;

// ---- torch glue (sg_torch_glue.cpp): the only place that sees torch headers -------------------
void *sgx_alloc(size_t bytes);   // c10 CUDACachingAllocator::raw_alloc; nullptr + error on failure
void sgx_free(void *p);
cudaStream_t sgx_stream();       // c10::cuda::getCurrentCUDAStream()
int sgx_device_ok(std::string *why);

void sg_set_error(const std::string &msg);

// ---- host-side Philox (sg_host.cpp) -----------------------------------------------------------
struct Philox4 { uint32_t x[4]; };
Philox4 sg_philox_host(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1);

// ---- VB instance layout -----------------------------------------------------------------------
// Sites are relabelled to "positions" p = 0..N-1: class-major (colour 0, 1, ...), and inside a class in
// breadth-first index order (BFS over the whole graph, roots in label order, rows in edge order): the
// locality-improving relabelling.  It is free: the order inside a colour class changes no output (Q15).
// Gauge fixing: the breadth-first forest's edges carry J = +1 in every lane after the transformation
// s_i -> eps_i s_i, J_ij -> eps_i J_ij eps_j with eps_child = eps_parent * J_(parent,child) (eps_root = +1), which
// changes no bond state, hence no flip decision, energy or correlation count.  The device stores the
// transformed spins and couplings; tree entries ("T") need no coupling word at all, the others ("X") do.
// Inside a class, every window of 4096 consecutive sites (in breadth-first order) is stably sorted by (demand, shape):
// demand 0 = the site has a neighbour in a class of fewer than N/32 sites, 1 = in a class of fewer than N/8 sites,
// 2 = neither (the gathers of the small classes then use whole lines); shape = sg_vb_shape below, so that the sites of a
// slice almost always share one.
// A class is cut into slices: runs of at most 32 consecutive positions with at most capE = 32*it entries, of which at
// most capX = 32*itx X entries (it, itx: per class, the smallest budget the kernels are compiled for that needs at most
// 30 % more slices than the largest one; a single site always fits).  A slice is one warp's work:
//   hdr[g]           = first position, first index in `col`, first index in the coupling array, and
//                      n | nXs << 6 | nE << 16 | shape << 28  (sites, X entries, all entries of the slice, the largest
//                      shape of its sites);
//   col              = for every slice ONE run of nE neighbour positions: first its X entries in site order (inside a
//                      site by position), then its T entries in site order (parent first, then children by position);
//                      the coupling array follows the X order, so entry e < nXs of the run has coupling j_off + e;
//   orig_s[32 g + j] = original label of the j-th site of slice g (SG_NONE for j >= n): the Philox counter;
//   rp_s[32 g + j]   = xOff | tOff << 8 | nX << 17 | nT << 22: where the site's X / T entries start inside the slice's
//                      run (tOff counts from the start of the run, so nXs <= tOff <= nE <= 256: nine bits), and how many
//                      there are.
// The kernels read a slice's run with one lane per ENTRY, 32 entries per step (every lane busy whatever the degrees,
// streams coalesced, neighbouring entries gather from neighbouring words), park spin ^ coupling in shared memory, and
// finish with one lane per SITE.
constexpr uint32_t SG_NONE = 0xFFFFFFFFu;

struct VBClass {
    uint64_t pos0;     // first position of the class
    uint64_t n;        // sites in the class
    uint64_t slice0;   // first slice
    uint64_t nslices;
    uint32_t it;       // entry budget of a slice of this class, in steps of 32 entries (capE = 32 * it)
    uint32_t itx;      // budget of X entries, in steps of 32 (capX = 32 * itx)
};

struct alignas(16) SGHdr { uint32_t pos0, col_off, j_off, counts; };
// shape of a site with nX X entries and nT T entries: which count the kernels run for it
constexpr uint32_t sg_vb_shape(uint32_t nX, uint32_t nT) { return (nX <= 2 && nT <= 2) ? 0u : (nX <= 4 && nT <= 4) ? 1u : 2u; }

struct VBHostGraph {
    uint64_t N = 0, M = 0;
    uint32_t K = 0, dmax = 0;
    uint32_t it_max = 0, itx_max = 0;      // largest per-class budgets (steps of 32 entries)
    bool gauge = true;
    std::vector<uint32_t> eu, ev;          // M edges in generation order (original labels)
    std::vector<uint64_t> row_ptr;         // N+1 (original labels)
    std::vector<uint32_t> adj;             // 2M neighbours, rows in increasing edge id
    std::vector<uint32_t> adj_e;           // 2M edge ids
    std::vector<uint8_t> colour;           // N
    std::vector<uint32_t> orig;            // position -> original label
    std::vector<uint32_t> pos;             // original label -> position
    std::vector<VBClass> cls;              // K classes
    std::vector<SGHdr> hdr;                // per slice, plus one sentinel (pos0 = N, offsets = totals, counts = 0)
    std::vector<uint32_t> orig_s, rp_s;    // 32 per slice
    std::vector<uint32_t> col;             // 2M neighbour positions
    std::vector<uint32_t> jeid;            // edge id of every coupling entry
    std::vector<uint32_t> tpar, teid;      // per position: parent position / tree edge id (SG_NONE: root)
    std::vector<uint32_t> bfs_pos;         // positions in breadth-first order (parents before children)
};

// Builds everything above.  Returns false and sets the error string on bad arguments.
bool sg_build_vb_graph(int model /* SG_MODEL_VB or SG_MODEL_RRBG */, uint64_t N, double c, uint64_t seed, uint32_t n_words, VBHostGraph &g);
// the (it, itx) budgets the kernels are compiled for, by words per thread G = 4, 2, 1 (W % 4 == 0, W % 2 == 0, else)
struct VBBudget { uint32_t it, itx; };
constexpr VBBudget SG_VB_BUDGETS_G1[] = {{6, 4}, {8, 6}};
constexpr VBBudget SG_VB_BUDGET_G2 = {4, 3}, SG_VB_BUDGET_G4 = {4, 2};
// words a thread of the sweep kernel owns for an instance of n_words words per site: 2 if n_words is even, else 1
// (SG_VB_G=<1|2|4> chooses another divisor of n_words: a measurement knob; outputs are identical)
uint32_t sg_vb_group(uint32_t n_words);

std::vector<uint64_t> sg_vb_thresholds(double T, uint32_t dmax);   // thr[0..dmax], thr[0]=0
std::vector<uint64_t> sg_sk_thresholds(double T, uint64_t N);      // thr[0..N-1]

// ---- device launchers (sg_kernels.cu) ---------------------------------------------------------
struct VBDevice {
    uint64_t *spin = nullptr;       // N*W words, position-major word-minor, gauge-transformed (sigma ^ eps)
    uint64_t *eps = nullptr;        // N*W words: the gauge (all 0 without gauge fixing); getters/setters only
    uint64_t *J = nullptr;          // nJ*W transformed coupling words (X entries only)
    uint32_t *col = nullptr;        // neighbour positions
    uint32_t *orig = nullptr;       // N: position -> label (getters / setters)
    uint32_t *orig_s = nullptr;     // 32 per slice
    uint32_t *rp_s = nullptr;       // 32 per slice
    SGHdr *hdr = nullptr;           // nslices+1
    uint32_t nslices = 0, it_max = 0, itx_max = 0;
    uint64_t thr_host[32] = {0};    // thresholds thr[k], k=0..31 (beyond dmax = 0): passed to the kernels by value
};

struct SGSeed { uint32_t k0, k1; };

int sgk_init_spins(uint64_t *spin, const uint32_t *orig, const uint64_t *eps, uint64_t N, uint32_t W, uint32_t word0, bool aligned, SGSeed key,
                   cudaStream_t st);
// draws every coupling entry (O3) and applies the gauge; jeid: device, edge id per coupling entry
int sgk_init_vb_couplings(const VBDevice &d, const uint32_t *jeid, uint32_t W, uint32_t word0, SGSeed key, cudaStream_t st);
// one colour class of one sweep; N, nJ = sizes of the whole instance (choose 32- or 64-bit index arithmetic);
// reverse = walk the class from its last slice to its first (callers alternate it from launch to launch)
int sgk_vb_sweep_class(const VBDevice &d, const VBClass &c, uint64_t N, uint64_t nJ, uint32_t W, uint32_t word0, uint64_t sweep, SGSeed key,
                       bool reverse, cudaStream_t st);
// counts[64*W] (device, u64) += per-lane number of set bits of (a XOR b) over n_sites*W words
int sgk_xor_popcount(const uint64_t *a, const uint64_t *b, uint64_t n_sites, uint32_t W, uint64_t *counts, cudaStream_t st);
// the same with the counters in the library's static device array (no allocation anywhere); out_host: HOST, 64*W uint64
constexpr uint32_t SG_NOALLOC_MAX_WORDS = 64;
int sgk_xor_popcount_noalloc(const uint64_t *a, const uint64_t *b, uint64_t n_sites, uint32_t W, uint64_t *out_host, cudaStream_t st);
// the same against up to 3 stored configurations in one pass: counts[s][64*W] += D(a, b[s])
int sgk_xor_popcount_multi(const uint64_t *a, const uint64_t *const *b, uint32_t n, uint64_t n_sites, uint32_t W, uint64_t *const *counts,
                           cudaStream_t st);
// counts[64*W] += per-lane sum over all sites of u_i (unsatisfied incident bonds): one launch over the whole instance
int sgk_vb_unsat(const VBDevice &d, uint64_t N, uint64_t nJ, uint32_t W, uint64_t *counts, cudaStream_t st);
int sgk_permute_words(const uint64_t *src, uint64_t *dst, const uint32_t *map, const uint64_t *eps, uint64_t N, uint32_t W, bool scatter,
                      cudaStream_t st);

// SK
struct SKDevice {
    uint64_t *spin = nullptr;    // N*W words
    uint32_t *rows = nullptr;    // lanes * N * (N/32) bits: rows[(lane*N + i)*NW32 + j/32] bit j%32 = 1 <=> J'_ij = -1
    int16_t *H = nullptr;        // lanes * N local fields H_i = sum_j J'_ij s_j
    uint64_t *thr = nullptr;     // N thresholds
    uint32_t *thr32 = nullptr;   // compact: thr clipped to u32, length nthr_nz (first index with 0 onwards omitted)
    uint32_t nthr_nz = 0;
    bool accept_all = false;     // T = inf
};

uint64_t sgk_launch_count();
