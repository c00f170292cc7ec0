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
// Sites are relabelled to "positions" p: class-major (colour 0, 1, ...), every class starting at a multiple of
// 32 (gap positions are padding: orig = SG_NONE, spin word 0, never written).  Inside a class the sites keep
// their breadth-first index order (the locality-improving relabelling), except that every window of
// SG_SORT_WINDOW consecutive sites is stably sorted by degree.  Slice g = positions 32g..32g+31 stores its rows
// column-major (sliced ELL) with row length D_g = the largest degree in the slice: the k-th neighbour of the
// j-th site of the slice lives at index 32*slice_ptr[g] + 32*k + j of `col` (neighbour position) and, times
// n_words plus w, of the coupling array.  Entries beyond a site's degree (and all entries of padding positions)
// point at the site's own position with coupling word 0.
constexpr uint32_t SG_NONE = 0xFFFFFFFFu;
constexpr uint32_t SG_SORT_WINDOW = 16384;

struct VBClass {
    uint64_t pos0;     // first position of the class (multiple of 32)
    uint64_t n;        // positions in the class, padding included (multiple of 32)
    uint64_t slice0;   // first slice = pos0 / 32
    uint64_t nslices;  // n / 32
};

struct VBHostGraph {
    uint64_t N = 0, M = 0;
    uint64_t P = 0;                        // positions including padding (multiple of 32)
    uint32_t K = 0, dmax = 0;
    std::vector<uint32_t> eu, ev;          // M edges in generation order (original labels)
    std::vector<uint64_t> row_ptr;         // N+1 (original labels)
    std::vector<uint32_t> adj;             // 2M neighbours, rows in increasing edge id
    std::vector<uint32_t> adj_e;           // 2M edge ids
    std::vector<uint8_t> colour;           // N
    std::vector<uint32_t> orig;            // position -> original label, SG_NONE for padding positions
    std::vector<uint32_t> pos;             // original label -> position
    std::vector<VBClass> cls;              // K classes
    std::vector<uint32_t> slice_ptr;       // nslices_total+1, units of 32 entries
    std::vector<uint32_t> col;             // 32*slice_ptr.back() entries: neighbour positions
    std::vector<uint32_t> eid;             // same length: edge id or 0xFFFFFFFF for padding
    std::vector<uint8_t> deg;              // per position (padding positions: 0)
    std::vector<uint32_t> entry_of_edge;   // M: entry index of edge e at endpoint eu[e]
};

// Builds everything above.  Returns false and sets the error string on bad arguments.
bool sg_build_vb_graph(int model /* SG_MODEL_VB or SG_MODEL_RRBG */, uint64_t N, double c, uint64_t seed, VBHostGraph &g);

std::vector<uint64_t> sg_vb_thresholds(double T, uint32_t dmax);   // thr[0..dmax], thr[0]=0
std::vector<uint64_t> sg_sk_thresholds(double T, uint64_t N);      // thr[0..N-1]

// ---- device launchers (sg_kernels.cu) ---------------------------------------------------------
struct VBDevice {
    uint64_t *spin = nullptr;       // P*W words, position-major word-minor
    uint64_t *J = nullptr;          // entries*W coupling words
    uint32_t *col = nullptr;        // entries
    uint32_t *orig = nullptr;       // P (SG_NONE = padding)
    uint32_t *slice_ptr = nullptr;  // nslices+1
    uint64_t *thr = nullptr;        // 32 thresholds (thr[k], k=0..31; beyond dmax = 0)
};

struct SGSeed { uint32_t k0, k1; };

int sgk_init_spins(uint64_t *spin, const uint32_t *orig, uint64_t N, uint32_t W, SGSeed key, cudaStream_t st);
int sgk_init_vb_couplings(uint64_t *J, const uint32_t *eid, uint64_t entries, uint32_t W, SGSeed key, cudaStream_t st);
// one colour class of one sweep; P, entries = sizes of the whole instance (choose 32- or 64-bit index arithmetic);
// reverse = walk the class from its last slice to its first (callers alternate it from launch to launch)
int sgk_vb_sweep_class(const VBDevice &d, const VBClass &c, uint64_t P, uint64_t entries, uint32_t W, uint64_t sweep, SGSeed key,
                       bool reverse, cudaStream_t st);
// counts[64*W] (device, u64) += per-lane number of set bits of (a XOR b) over n_sites*W words
int sgk_xor_popcount(const uint64_t *a, const uint64_t *b, uint64_t n_sites, uint32_t W, uint64_t *counts, cudaStream_t st);
// counts[64*W] += per-lane sum over the class's sites of u_i (unsatisfied incident bonds)
int sgk_vb_unsat_class(const VBDevice &d, const VBClass &c, uint32_t W, uint64_t *counts, cudaStream_t st);
int sgk_permute_words(const uint64_t *src, uint64_t *dst, const uint32_t *map, uint64_t N, uint32_t W, bool scatter, cudaStream_t st);

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
int sgk_sk_init_rows(const SKDevice &d, uint64_t N, uint32_t W, SGSeed key, cudaStream_t st);
int sgk_sk_init_fields(const SKDevice &d, uint64_t N, uint32_t W, cudaStream_t st);
int sgk_sk_sweep(const SKDevice &d, uint64_t N, uint32_t W, uint64_t sweep, uint64_t nsweeps, SGSeed key, cudaStream_t st);
int sgk_sk_energy(const SKDevice &d, uint64_t N, uint32_t W, int64_t *out_dev, cudaStream_t st);

uint64_t sgk_launch_count();
