// sg_api.cu -- the C-ABI of include/sg.h: handle, argument checks, buffer ownership, call
// sequencing.  Every step of the path runs in the kernels of sg_kernels.cu / sg_sk.cu.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <new>
#include <string>
#include <vector>

#include <algorithm>

#include "sg_internal.h"
#include "sg_sim.h"

static thread_local std::string g_err;
void sg_set_error(const std::string &msg) { g_err = msg; }
extern "C" const char *sg_last_error(void) { return g_err.c_str(); }
extern "C" uint64_t sg_kernel_launches(void) { return sgk_launch_count(); }

namespace {

// A handle's buffers live on the device that was current at sg_create; launching on another device (after a
// torch.cuda.set_device, say) would be an error that CUDA reports late and far away.
bool on_own_device(const sg_sim *h, const char *who)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) {
        sg_set_error(std::string(who) + ": the current CUDA device is not the one the handle was created on");
        return false;
    }
    return true;
}

void destroy_impl(sg_sim *h)
{
    if (!h) return;
    cudaStreamSynchronize(sgx_stream());
    for (void *p : h->owned) sgx_free(p);
    delete h;
}

// kappa_e[w] of DESIGN.md O3 on the host (the gauge needs the tree edges' couplings before anything is on the device)
uint64_t host_coupling_word(uint32_t e, uint32_t w, SGSeed key)
{
    const Philox4 x = sg_philox_host(e, w, 0u, 2u << 24, key.k0, key.k1);
    return (uint64_t)x.x[0] | ((uint64_t)x.x[1] << 32);
}

int create_vb(sg_sim *h)
{
    cudaStream_t st = sgx_stream();
    if (!sg_build_vb_graph(h->graph_model, h->N, h->c, h->seed, h->W, h->g)) return SG_EINVAL;
    VBHostGraph &g = h->g;
    h->M = g.M;
    const uint64_t W = h->W, N = g.N;
    const uint64_t nslices = g.hdr.size() - 1, entries = g.col.size(), nJ = g.jeid.size();
    h->spin_words = N * W;
    h->vb_nJ = nJ;
    h->vb.nslices = (uint32_t)nslices;
    h->vb.it_max = g.it_max; h->vb.itx_max = g.itx_max;
    h->vb.spin = dev_alloc<uint64_t>(h, N * W);
    h->vb.eps = dev_alloc<uint64_t>(h, N * W);
    h->vb.J = dev_alloc<uint64_t>(h, nJ * W + 4);
    h->vb.col = dev_alloc<uint32_t>(h, entries + 1);
    h->vb.orig = dev_alloc<uint32_t>(h, N);
    h->vb.orig_s = dev_alloc<uint32_t>(h, 32 * nslices);
    h->vb.rp_s = dev_alloc<uint32_t>(h, 32 * nslices);
    h->vb.hdr = dev_alloc<SGHdr>(h, nslices + 1);
    uint32_t *jeid_dev = dev_alloc<uint32_t>(h, nJ + 1);
    if (!h->vb.spin || !h->vb.eps || !h->vb.J || !h->vb.col || !h->vb.orig || !h->vb.orig_s || !h->vb.rp_s || !h->vb.hdr || !jeid_dev)
        return SG_ENOMEM;
    h->thr_host = sg_vb_thresholds(h->T, g.dmax);
    for (size_t k = 0; k < h->thr_host.size() && k < 32; ++k) h->vb.thr_host[k] = h->thr_host[k];
    // the gauge: eps_root = 0, eps_child = eps_parent ^ kappa_(tree edge), parents before children (sg_internal.h)
    std::vector<uint64_t> eps(N * W, 0);
    if (g.gauge)
        for (uint64_t q = 0; q < N; ++q) {
            const uint64_t p = g.bfs_pos[q], par = g.tpar[p];
            if (par == SG_NONE) continue;
            for (uint32_t w = 0; w < W; ++w) eps[p * W + w] = eps[par * W + w] ^ host_coupling_word(g.teid[p], h->word0 + w, h->key);
        }
    if (!upload(h->vb.col, g.col, st) || !upload(h->vb.orig, g.orig, st) || !upload(h->vb.orig_s, g.orig_s, st) ||
        !upload(h->vb.rp_s, g.rp_s, st) || !upload(h->vb.hdr, g.hdr, st) ||
        !upload(jeid_dev, g.jeid, st) || !upload(h->vb.eps, eps, st))
        return SG_ECUDA;
    int rc = sgk_init_vb_couplings(h->vb, jeid_dev, h->W, h->word0, h->key, st);
    if (rc) return rc;
    rc = sgk_init_spins(h->vb.spin, h->vb.orig, h->vb.eps, N, h->W, h->word0, h->aligned, h->key, st);
    if (rc) return rc;
    if (!cuda_ok(cudaStreamSynchronize(st), "sg_create")) return SG_ECUDA;
    // the entry->edge table is only needed to draw the couplings; the large host copies are not needed any more
    sgx_free(jeid_dev);
    h->owned.erase(std::find(h->owned.begin(), h->owned.end(), (void *)jeid_dev));
    std::vector<uint32_t>().swap(g.jeid);
    std::vector<uint32_t>().swap(g.col);
    std::vector<uint32_t>().swap(g.bfs_pos);
    std::vector<uint32_t>().swap(g.orig_s);
    return SG_OK;
}

}  // namespace

extern "C" sg_sim *sg_create(int model, uint64_t N, double c, double T, uint64_t seed, uint32_t n_words)
{
    return sg_create_opt(model, N, c, T, seed, n_words, nullptr);
}

extern "C" uint64_t sg_num_lanes(const sg_sim *h) { return h ? h->lanes : 0; }

extern "C" sg_sim *sg_create_opt(int model, uint64_t N, double c, double T, uint64_t seed, uint32_t n_words, const sg_options *opt)
{
    g_err.clear();
    sg_options o{0, 1, 0, 0};
    if (opt) o = *opt;
    if (o.n_clones == 0) o.n_clones = 1;
    if (o.reserved != 0 || o.aligned_start > 1) { sg_set_error("sg_create_opt: bad options"); return nullptr; }
    if (o.n_clones > 2 || (o.n_clones == 2 && model != SG_MODEL_SK)) { sg_set_error("sg_create_opt: n_clones must be 1, or 2 for the SK model"); return nullptr; }
    if (o.word0 % 4 != 0 || (uint64_t)o.word0 + n_words > (1u << 20)) { sg_set_error("sg_create_opt: word0 must be a multiple of 4 and word0 + n_words <= 2^20"); return nullptr; }
    if (model != SG_MODEL_VB && model != SG_MODEL_SK && model != SG_MODEL_RRBG && model != SG_MODEL_RRG) { sg_set_error("sg_create: unknown model"); return nullptr; }
    if (N < 2 || N >= (1ull << 31) - 2) { sg_set_error("sg_create: N must satisfy 2 <= N < 2^31 - 2"); return nullptr; }
    if (n_words == 0 || n_words > 65535) { sg_set_error("sg_create: n_words must satisfy 1 <= n_words <= 65535"); return nullptr; }
    if (!(T >= 0.0)) { sg_set_error("sg_create: T must be >= 0 (T = inf allowed)"); return nullptr; }
    if (model == SG_MODEL_SK && N > 32768) { sg_set_error("sg_create: SK needs N <= 32768 (int16 local fields)"); return nullptr; }
    std::string why;
    if (!sgx_device_ok(&why)) { sg_set_error("sg_create: " + why); return nullptr; }
    sg_sim *h = new (std::nothrow) sg_sim();
    if (!h) { sg_set_error("sg_create: out of host memory"); return nullptr; }
    // RRBG and RRG are the VB Hamiltonian on other graph ensembles: only the host generator tells them apart
    h->graph_model = model;
    if (model == SG_MODEL_RRBG || model == SG_MODEL_RRG) model = SG_MODEL_VB;
    h->model = model; h->N = N; h->W = n_words; h->c = c; h->T = T; h->seed = seed;
    h->word0 = o.word0; h->clones = o.n_clones; h->aligned = o.aligned_start != 0;
    h->lanes = 64ull * n_words * o.n_clones;
    h->key = SGSeed{(uint32_t)seed, (uint32_t)(seed >> 32)};
    cudaGetDevice(&h->device);
    int rc;
    try {
        rc = (model == SG_MODEL_VB) ? create_vb(h) : sg_sk_create_impl(h);
        if (rc == SG_OK) {
            h->counts_dev = dev_alloc<uint64_t>(h, h->lanes);
            if (!h->counts_dev) rc = SG_ENOMEM;
        }
    } catch (const std::bad_alloc &) {
        sg_set_error("sg_create: out of host memory");
        rc = SG_ENOMEM;
    }
    if (rc != SG_OK) { destroy_impl(h); return nullptr; }
    return h;
}

extern "C" void sg_destroy(sg_sim *h) { destroy_impl(h); }

extern "C" int sg_sweep(sg_sim *h, uint64_t n)
{
    if (!h) { sg_set_error("sg_sweep: null handle"); return SG_EINVAL; }
    if (!on_own_device(h, "sg_sweep")) return SG_EINVAL;
    if (h->sweep + n >= (1ull << 56)) { sg_set_error("sg_sweep: sweep counter would exceed 2^56"); return SG_EINVAL; }
    if (h->model == SG_MODEL_SK) return sg_sk_sweep_impl(h, n);
    cudaStream_t st = sgx_stream();
    for (uint64_t it = 0; it < n; ++it) {
        for (uint32_t k = 0; k < h->g.K; ++k) {
            const int rc = sgk_vb_sweep_class(h->vb, h->g.cls[k], h->g.N, h->vb_nJ, h->W, h->word0, h->sweep, h->key, h->vb_reverse, st);
            h->vb_reverse = !h->vb_reverse;
            if (rc) return rc;
        }
        h->sweep++;
    }
    return SG_OK;
}

// ---- site-sharded sweeps -----------------------------------------------------------------------------
static bool vb_part_ok(sg_sim *h, uint32_t k, uint64_t unit0, uint64_t n, const char *who)
{
    if (!h || h->model != SG_MODEL_VB) { sg_set_error(std::string(who) + ": VB handle required"); return false; }
    if (k >= h->g.K || unit0 + n > h->g.cls[k].nslices) { sg_set_error(std::string(who) + ": class or unit range out of bounds"); return false; }
    return true;
}

extern "C" int sg_class_units(sg_sim *h, uint32_t k, uint64_t *n_units)
{
    if (!n_units || !vb_part_ok(h, k, 0, 0, "sg_class_units")) return SG_EINVAL;
    *n_units = h->g.cls[k].nslices;
    return SG_OK;
}

extern "C" int sg_sweep_part(sg_sim *h, uint32_t k, uint64_t unit0, uint64_t n_units)
{
    if (!vb_part_ok(h, k, unit0, n_units, "sg_sweep_part")) return SG_EINVAL;
    if (n_units == 0) return SG_OK;
    VBClass part = h->g.cls[k];
    part.slice0 += unit0;
    part.nslices = n_units;
    part.n = 1;       // non-empty (the kernels take their positions from the slice headers)
    return sgk_vb_sweep_class(h->vb, part, h->g.N, h->vb_nJ, h->W, h->word0, h->sweep, h->key, false, sgx_stream());
}

extern "C" int sg_end_sweep(sg_sim *h)
{
    if (!h || h->sweep + 1 >= (1ull << 56)) { sg_set_error("sg_end_sweep: bad handle or counter overflow"); return SG_EINVAL; }
    h->sweep++;
    return SG_OK;
}

extern "C" int sg_part_range(sg_sim *h, uint32_t k, uint64_t unit0, uint64_t n_units, uint64_t *first_word, uint64_t *n_words)
{
    if (!first_word || !n_words || !vb_part_ok(h, k, unit0, n_units, "sg_part_range")) return SG_EINVAL;
    const uint64_t s0 = h->g.cls[k].slice0 + unit0;
    const uint64_t p0 = h->g.hdr[s0].pos0;
    // the next slice of the same class starts where this range ends; after the last slice of the class the class ends
    const uint64_t p1 = unit0 + n_units < h->g.cls[k].nslices ? h->g.hdr[s0 + n_units].pos0 : h->g.cls[k].pos0 + h->g.cls[k].n;
    *first_word = p0 * h->W;
    *n_words = (n_units ? p1 - p0 : 0) * h->W;
    return SG_OK;
}

extern "C" int sg_spin_device_pointer(sg_sim *h, void **ptr)
{
    if (!h || !ptr || h->model != SG_MODEL_VB) { sg_set_error("sg_spin_device_pointer: VB handle required"); return SG_EINVAL; }
    *ptr = h->vb.spin;
    return SG_OK;
}

extern "C" int sg_export_part(sg_sim *h, uint64_t first_word, uint64_t n_words, uint64_t *out)
{
    if (!h || h->model != SG_MODEL_VB || (n_words && !out) || first_word + n_words > h->spin_words) { sg_set_error("sg_export_part: bad argument"); return SG_EINVAL; }
    cudaStream_t st = sgx_stream();
    if (n_words && (!cuda_ok(cudaMemcpyAsync(out, h->vb.spin + first_word, n_words * 8, cudaMemcpyDeviceToHost, st), "sg_export_part") ||
                    !cuda_ok(cudaStreamSynchronize(st), "sg_export_part")))
        return SG_ECUDA;
    return SG_OK;
}

extern "C" int sg_import_part(sg_sim *h, uint64_t first_word, uint64_t n_words, const uint64_t *in)
{
    if (!h || h->model != SG_MODEL_VB || (n_words && !in) || first_word + n_words > h->spin_words) { sg_set_error("sg_import_part: bad argument"); return SG_EINVAL; }
    cudaStream_t st = sgx_stream();
    if (n_words && (!cuda_ok(cudaMemcpyAsync(h->vb.spin + first_word, in, n_words * 8, cudaMemcpyHostToDevice, st), "sg_import_part") ||
                    !cuda_ok(cudaStreamSynchronize(st), "sg_import_part")))
        return SG_ECUDA;
    return SG_OK;
}

static uint64_t *current_config(sg_sim *h) { return h->model == SG_MODEL_VB ? h->vb.spin : h->sk.spin; }

extern "C" int sg_snapshot(sg_sim *h, uint32_t slot)
{
    if (!h) { sg_set_error("sg_snapshot: null handle"); return SG_EINVAL; }
    if (!on_own_device(h, "sg_snapshot")) return SG_EINVAL;
    if (slot >= SG_MAX_SLOTS) { sg_set_error("sg_snapshot: slot out of range"); return SG_EINVAL; }
    if (!h->slot[slot]) {
        h->slot[slot] = dev_alloc<uint64_t>(h, h->spin_words);
        if (!h->slot[slot]) return SG_ENOMEM;
    }
    if (!cuda_ok(cudaMemcpyAsync(h->slot[slot], current_config(h), h->spin_words * 8, cudaMemcpyDeviceToDevice, sgx_stream()),
                 "sg_snapshot"))
        return SG_ECUDA;
    return SG_OK;
}

extern "C" int sg_correlation(sg_sim *h, uint32_t slot, uint64_t *out_counts)
{
    if (!h || !out_counts) { sg_set_error("sg_correlation: null argument"); return SG_EINVAL; }
    if (!on_own_device(h, "sg_correlation")) return SG_EINVAL;
    if (slot >= SG_MAX_SLOTS) { sg_set_error("sg_correlation: slot out of range"); return SG_EINVAL; }
    if (!h->slot[slot]) { sg_set_error("sg_correlation: slot was never written"); return SG_ESLOT; }
    cudaStream_t st = sgx_stream();
    const uint64_t lanes = h->lanes;
    if (!cuda_ok(cudaMemsetAsync(h->counts_dev, 0, lanes * 8, st), "sg_correlation")) return SG_ECUDA;
    if (h->model == SG_MODEL_SK) return sg_sk_correlation_impl(h, h->slot[slot], out_counts);
    // position order in both operands (the same permutation), so no relabelling is needed
    const int rc = sgk_xor_popcount(current_config(h), h->slot[slot], h->g.N, h->W, h->counts_dev, st);
    if (rc) return rc;
    if (!cuda_ok(cudaMemcpyAsync(out_counts, h->counts_dev, lanes * 8, cudaMemcpyDeviceToHost, st), "sg_correlation") ||
        !cuda_ok(cudaStreamSynchronize(st), "sg_correlation"))
        return SG_ECUDA;
    return SG_OK;
}

// sg_correlation for callers that must not allocate: the counters live in the library's static device array
extern "C" uint32_t sg_noalloc_max_words(void) { return SG_NOALLOC_MAX_WORDS; }

extern "C" int sg_correlation_noalloc(sg_sim *h, uint32_t slot, uint64_t *out_counts)
{
    if (!h || !out_counts) { sg_set_error("sg_correlation_noalloc: null argument"); return SG_EINVAL; }
    if (!on_own_device(h, "sg_correlation_noalloc")) return SG_EINVAL;
    if (h->model != SG_MODEL_VB) { sg_set_error("sg_correlation_noalloc: graph models only (VB, RRBG, RRG)"); return SG_EINVAL; }
    if (slot >= SG_MAX_SLOTS) { sg_set_error("sg_correlation_noalloc: slot out of range"); return SG_EINVAL; }
    if (!h->slot[slot]) { sg_set_error("sg_correlation_noalloc: slot was never written"); return SG_ESLOT; }
    return sgk_xor_popcount_noalloc(current_config(h), h->slot[slot], h->g.N, h->W, out_counts, sgx_stream());
}

// ---- windowed protocol: device-side accumulation of correlation counts ---------------------
extern "C" int sg_corr_configure(sg_sim *h, uint32_t nbins)
{
    if (!h || nbins == 0 || nbins > (1u << 20)) { sg_set_error("sg_corr_configure: bad argument"); return SG_EINVAL; }
    cudaStream_t st = sgx_stream();
    if (nbins > h->corr_bins) {
        // (the old block stays with the handle until sg_destroy; reconfiguring to a larger size is rare)
        h->corr_acc = dev_alloc<uint64_t>(h, (uint64_t)nbins * h->lanes);
        if (!h->corr_acc) { h->corr_bins = 0; return SG_ENOMEM; }
        h->corr_bins = nbins;
    }
    h->corr_n.assign(h->corr_bins, 0);
    if (!cuda_ok(cudaMemsetAsync(h->corr_acc, 0, (uint64_t)h->corr_bins * h->lanes * 8, st), "sg_corr_configure")) return SG_ECUDA;
    return SG_OK;
}

extern "C" int sg_corr_accumulate(sg_sim *h, uint32_t n, const uint32_t *slots, const uint32_t *bins)
{
    if (!h || (n && (!slots || !bins))) { sg_set_error("sg_corr_accumulate: null argument"); return SG_EINVAL; }
    if (!on_own_device(h, "sg_corr_accumulate")) return SG_EINVAL;
    if (!h->corr_acc) { sg_set_error("sg_corr_accumulate: call sg_corr_configure first"); return SG_EINVAL; }
    for (uint32_t k = 0; k < n; ++k) {
        if (slots[k] >= SG_MAX_SLOTS || bins[k] >= h->corr_bins) { sg_set_error("sg_corr_accumulate: slot or bin out of range"); return SG_EINVAL; }
        if (!h->slot[slots[k]]) { sg_set_error("sg_corr_accumulate: slot was never written"); return SG_ESLOT; }
        for (uint32_t q = 0; q < k; ++q)
            if (bins[q] == bins[k]) { sg_set_error("sg_corr_accumulate: the bins of one call must be distinct"); return SG_EINVAL; }
    }
    cudaStream_t st = sgx_stream();
    for (uint32_t k0 = 0; k0 < n; k0 += 3) {
        const uint32_t m = std::min<uint32_t>(3, n - k0);
        const uint64_t *b[3];
        uint64_t *c[3];
        for (uint32_t q = 0; q < m; ++q) { b[q] = h->slot[slots[k0 + q]]; c[q] = h->corr_acc + (uint64_t)bins[k0 + q] * h->lanes; }
        int rc = SG_OK;
        if (h->model == SG_MODEL_SK) {
            for (uint32_t q = 0; q < m && rc == SG_OK; ++q) rc = sg_sk_corr_accumulate_impl(h, b[q], c[q]);
        } else {
            rc = sgk_xor_popcount_multi(current_config(h), b, m, h->g.N, h->W, c, st);
        }
        if (rc) return rc;
    }
    for (uint32_t k = 0; k < n; ++k) h->corr_n[bins[k]]++;
    return SG_OK;
}

extern "C" int sg_corr_fetch(sg_sim *h, uint32_t bin0, uint32_t nbins, uint64_t *out, uint64_t *n_out)
{
    if (!h || !out) { sg_set_error("sg_corr_fetch: null argument"); return SG_EINVAL; }
    if (!h->corr_acc || (uint64_t)bin0 + nbins > h->corr_bins) { sg_set_error("sg_corr_fetch: bins out of range"); return SG_EINVAL; }
    cudaStream_t st = sgx_stream();
    if (nbins && (!cuda_ok(cudaMemcpyAsync(out, h->corr_acc + (uint64_t)bin0 * h->lanes, (uint64_t)nbins * h->lanes * 8, cudaMemcpyDeviceToHost, st),
                           "sg_corr_fetch") ||
                  !cuda_ok(cudaStreamSynchronize(st), "sg_corr_fetch")))
        return SG_ECUDA;
    if (n_out) for (uint32_t b = 0; b < nbins; ++b) n_out[b] = h->corr_n[bin0 + b];
    return SG_OK;
}

extern "C" int sg_energy(sg_sim *h, int64_t *out)
{
    if (!h || !out) { sg_set_error("sg_energy: null argument"); return SG_EINVAL; }
    if (!on_own_device(h, "sg_energy")) return SG_EINVAL;
    if (h->model == SG_MODEL_SK) return sg_sk_energy_impl(h, out);
    cudaStream_t st = sgx_stream();
    const uint64_t lanes = h->lanes;
    if (!cuda_ok(cudaMemsetAsync(h->counts_dev, 0, lanes * 8, st), "sg_energy")) return SG_ECUDA;
    const int rc = sgk_vb_unsat(h->vb, h->g.N, h->vb_nJ, h->W, h->counts_dev, st);
    if (rc) return rc;
    std::vector<uint64_t> twoU(lanes);
    if (!cuda_ok(cudaMemcpyAsync(twoU.data(), h->counts_dev, lanes * 8, cudaMemcpyDeviceToHost, st), "sg_energy") ||
        !cuda_ok(cudaStreamSynchronize(st), "sg_energy"))
        return SG_ECUDA;
    // sum_i u_i counts every unsatisfied bond from both ends: = 2U.  E = -(M - U) + U = 2U - M.
    for (uint64_t l = 0; l < lanes; ++l) out[l] = (int64_t)twoU[l] - (int64_t)h->M;
    return SG_OK;
}

// ---- getters ------------------------------------------------------------------------------------
extern "C" uint64_t sg_sweep_count(const sg_sim *h) { return h ? h->sweep : 0; }
extern "C" uint64_t sg_num_edges(const sg_sim *h) { return h ? h->M : 0; }
extern "C" uint32_t sg_num_colours(const sg_sim *h) { return (h && h->model == SG_MODEL_VB) ? h->g.K : 0; }
extern "C" uint32_t sg_max_degree(const sg_sim *h)
{
    if (!h) return 0;
    return h->model == SG_MODEL_VB ? h->g.dmax : (uint32_t)(h->N - 1);
}

static bool ensure_scratch(sg_sim *h)
{
    if (!h->scratch) h->scratch = dev_alloc<uint64_t>(h, h->N * h->W);   // original order
    return h->scratch != nullptr;
}

extern "C" int sg_get_spins(sg_sim *h, int32_t slot, uint64_t *out)
{
    if (!h || !out) { sg_set_error("sg_get_spins: null argument"); return SG_EINVAL; }
    const uint64_t *src = current_config(h);
    if (slot >= 0) {
        if (slot >= SG_MAX_SLOTS) { sg_set_error("sg_get_spins: slot out of range"); return SG_EINVAL; }
        if (!h->slot[slot]) { sg_set_error("sg_get_spins: slot was never written"); return SG_ESLOT; }
        src = h->slot[slot];
    }
    cudaStream_t st = sgx_stream();
    if (h->model == SG_MODEL_SK) return sg_sk_get_spins_impl(h, src, out);
    if (!ensure_scratch(h)) return SG_ENOMEM;
    const int rc = sgk_permute_words(src, h->scratch, h->vb.orig, h->vb.eps, h->g.N, h->W, /*scatter=*/true, st);
    if (rc) return rc;
    if (!cuda_ok(cudaMemcpyAsync(out, h->scratch, h->N * h->W * 8, cudaMemcpyDeviceToHost, st), "sg_get_spins") ||
        !cuda_ok(cudaStreamSynchronize(st), "sg_get_spins"))
        return SG_ECUDA;
    return SG_OK;
}

extern "C" int sg_set_spins(sg_sim *h, const uint64_t *in)
{
    if (!h || !in) { sg_set_error("sg_set_spins: null argument"); return SG_EINVAL; }
    if (h->model == SG_MODEL_SK) return sg_sk_set_spins_impl(h, in);
    cudaStream_t st = sgx_stream();
    if (!ensure_scratch(h)) return SG_ENOMEM;
    if (!cuda_ok(cudaMemcpyAsync(h->scratch, in, h->N * h->W * 8, cudaMemcpyHostToDevice, st), "sg_set_spins")) return SG_ECUDA;
    const int rc = sgk_permute_words(h->scratch, h->vb.spin, h->vb.orig, h->vb.eps, h->g.N, h->W, /*scatter=*/false, st);
    if (rc) return rc;
    if (!cuda_ok(cudaStreamSynchronize(st), "sg_set_spins")) return SG_ECUDA;
    return SG_OK;
}

extern "C" int sg_set_sweep_count(sg_sim *h, uint64_t t)
{
    if (!h || t >= (1ull << 56)) { sg_set_error("sg_set_sweep_count: bad argument"); return SG_EINVAL; }
    h->sweep = t;
    return SG_OK;
}

extern "C" int sg_get_graph(sg_sim *h, uint64_t *row_ptr, uint32_t *col, uint32_t *colour)
{
    if (!h || h->model != SG_MODEL_VB) { sg_set_error("sg_get_graph: VB handle required"); return SG_EINVAL; }
    const VBHostGraph &g = h->g;
    if (row_ptr) std::memcpy(row_ptr, g.row_ptr.data(), (g.N + 1) * sizeof(uint64_t));
    if (col) std::memcpy(col, g.adj.data(), 2 * g.M * sizeof(uint32_t));
    if (colour) for (uint64_t i = 0; i < g.N; ++i) colour[i] = g.colour[i];
    return SG_OK;
}

extern "C" int sg_get_edges(sg_sim *h, uint32_t *u, uint32_t *v)
{
    if (!h || h->model != SG_MODEL_VB || !u || !v) { sg_set_error("sg_get_edges: VB handle required"); return SG_EINVAL; }
    std::memcpy(u, h->g.eu.data(), h->g.M * sizeof(uint32_t));
    std::memcpy(v, h->g.ev.data(), h->g.M * sizeof(uint32_t));
    return SG_OK;
}

extern "C" int sg_get_couplings(sg_sim *h, uint64_t *out)
{
    if (!h || !out) { sg_set_error("sg_get_couplings: null argument"); return SG_EINVAL; }
    if (h->model == SG_MODEL_SK) return sg_sk_get_couplings_impl(h, out);
    // Undo the gauge from what the device holds: a coupling entry of the site at position p towards position nb stores
    // kappa ^ eps[p] ^ eps[nb]; a tree edge stores nothing and has kappa = eps[p] ^ eps[parent].  Every edge that is
    // not a tree edge is stored at both endpoints; the two copies must agree.
    cudaStream_t st = sgx_stream();
    const VBHostGraph &g = h->g;
    const uint64_t W = h->W, N = g.N, nslices = g.hdr.size() - 1, entries = g.hdr[nslices].col_off, nJ = g.hdr[nslices].j_off;
    std::vector<uint64_t> J(nJ * W), eps(N * W);
    std::vector<uint32_t> col(entries);
    if (!cuda_ok(cudaMemcpyAsync(J.data(), h->vb.J, J.size() * 8, cudaMemcpyDeviceToHost, st), "sg_get_couplings") ||
        !cuda_ok(cudaMemcpyAsync(eps.data(), h->vb.eps, eps.size() * 8, cudaMemcpyDeviceToHost, st), "sg_get_couplings") ||
        !cuda_ok(cudaMemcpyAsync(col.data(), h->vb.col, col.size() * 4, cudaMemcpyDeviceToHost, st), "sg_get_couplings") ||
        !cuda_ok(cudaStreamSynchronize(st), "sg_get_couplings"))
        return SG_ECUDA;
    std::vector<uint8_t> seen(g.M, 0);
    auto edge_between = [&](uint32_t i, uint32_t v) -> uint32_t {
        for (uint64_t a = g.row_ptr[i]; a < g.row_ptr[i + 1]; ++a)
            if (g.adj[a] == v) return g.adj_e[a];
        return SG_NONE;
    };
    for (uint64_t s = 0; s < nslices; ++s) {
        const SGHdr &hd = g.hdr[s];
        const uint32_t n = hd.counts & 63u;
        for (uint32_t j = 0; j < n; ++j) {
            const uint32_t rp = g.rp_s[32 * s + j], xOff = rp & 255u, nX = (rp >> 17) & 31u;
            const uint64_t p = (uint64_t)hd.pos0 + j;
            for (uint32_t r = 0; r < nX; ++r) {
                const uint64_t nb = col[(uint64_t)hd.col_off + xOff + r], x = (uint64_t)hd.j_off + xOff + r;
                const uint32_t e = edge_between(g.orig[p], g.orig[nb]);
                if (e == SG_NONE) { sg_set_error("sg_get_couplings: a stored entry is not an edge of the graph"); return SG_ECUDA; }
                for (uint32_t w = 0; w < W; ++w) {
                    const uint64_t k = J[x * W + w] ^ eps[p * W + w] ^ eps[nb * W + w];
                    if (seen[e] && out[(uint64_t)e * W + w] != k) { sg_set_error("sg_get_couplings: the two stored copies of an edge differ"); return SG_ECUDA; }
                    out[(uint64_t)e * W + w] = k;
                }
                seen[e]++;
            }
        }
    }
    for (uint64_t p = 0; p < N; ++p) {
        if (!g.gauge || g.tpar[p] == SG_NONE) continue;
        const uint32_t e = g.teid[p];
        if (seen[e]) { sg_set_error("sg_get_couplings: a tree edge also has a stored coupling"); return SG_ECUDA; }
        for (uint32_t w = 0; w < W; ++w) out[(uint64_t)e * W + w] = eps[p * W + w] ^ eps[(uint64_t)g.tpar[p] * W + w];
        seen[e] = 2;
    }
    for (uint64_t e = 0; e < g.M; ++e)
        if (seen[e] != 2) { sg_set_error("sg_get_couplings: an edge is not stored exactly twice"); return SG_ECUDA; }
    return SG_OK;
}

extern "C" int sg_get_thresholds(sg_sim *h, uint64_t *out, uint64_t n)
{
    if (!h || !out) { sg_set_error("sg_get_thresholds: null argument"); return SG_EINVAL; }
    for (uint64_t k = 0; k < n; ++k) out[k] = k < h->thr_host.size() ? h->thr_host[k] : 0;
    return SG_OK;
}
