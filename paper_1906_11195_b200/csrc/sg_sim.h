// sg_sim.h -- the handle behind the opaque sg_sim of include/sg.h, and small CUDA host helpers.
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "sg_internal.h"

struct sg_sim {
    int model = SG_MODEL_VB;                 // SG_MODEL_VB (also for RRBG instances) or SG_MODEL_SK
    int graph_model = SG_MODEL_VB;           // the graph ensemble: SG_MODEL_VB (Erdos-Renyi) or SG_MODEL_RRBG
    uint64_t N = 0, M = 0;
    uint32_t W = 0;
    uint32_t word0 = 0, clones = 1;         // sg_options
    bool aligned = false;
    uint64_t lanes = 0;                      // 64 * W * clones
    double c = 0, T = 0;
    uint64_t seed = 0;
    uint64_t sweep = 0;
    int device = -1;                         // the CUDA device the handle was created on: every call checks it
    SGSeed key{0, 0};
    // VB
    VBHostGraph g;
    VBDevice vb;
    std::vector<uint64_t> thr_host;
    bool vb_reverse = false;                 // direction of the next colour-class launch (alternates)
    uint64_t vb_nJ = 0;                      // coupling entries
    // SK
    SKDevice sk;
    // common
    uint64_t spin_words = 0;                 // words in one configuration (device layout)
    uint64_t *slot[SG_MAX_SLOTS] = {nullptr};
    uint64_t *counts_dev = nullptr;          // 64*W
    uint64_t *scratch = nullptr;             // one configuration, for getters
    uint64_t *corr_acc = nullptr;            // windowed protocol: corr_bins x lanes accumulated counts
    uint32_t corr_bins = 0;
    std::vector<uint64_t> corr_n;            // accumulations per bin
    std::vector<void *> owned;               // every device allocation
};


inline bool cuda_ok(cudaError_t e, const char *what)
{
    if (e == cudaSuccess) return true;
    sg_set_error(std::string(what) + ": " + cudaGetErrorString(e));
    return false;
}

template <class T>
T *dev_alloc(sg_sim *h, uint64_t count)
{
    void *p = sgx_alloc(count * sizeof(T));
    if (p) h->owned.push_back(p);
    return (T *)p;
}

template <class T>
bool upload(T *dst, const std::vector<T> &src, cudaStream_t st)
{
    if (src.empty()) return true;
    return cuda_ok(cudaMemcpyAsync(dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, st), "host-to-device copy");
}

// SK entry points (sg_sk.cu)
int sg_sk_create_impl(sg_sim *h);
int sg_sk_sweep_impl(sg_sim *h, uint64_t n);
int sg_sk_energy_impl(sg_sim *h, int64_t *out);
int sg_sk_correlation_impl(sg_sim *h, const uint64_t *slot_dev, uint64_t *out);
int sg_sk_corr_accumulate_impl(sg_sim *h, const uint64_t *slot_dev, uint64_t *acc_dev);
int sg_sk_get_spins_impl(sg_sim *h, const uint64_t *src_dev, uint64_t *out);
int sg_sk_set_spins_impl(sg_sim *h, const uint64_t *in);
int sg_sk_get_couplings_impl(sg_sim *h, uint64_t *out);
