// sg_kernels.cu -- CUDA kernels (sm_100a) of the Viana-Bray path that do not walk rows (those are in sg_vb_sweep.cu):
// initial spins (a2 of SURVEY.md 8(a)), the correlation counts (a6), relabelling for the getters.
// Conventions: DESIGN.md section 3.  All arithmetic is integer / bitwise.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <string>

#include "sg_device.cuh"
#include "sg_internal.h"

static std::atomic<uint64_t> g_launches{0};
uint64_t sgk_launch_count() { return g_launches.load(); }
void sgk_count_launch() { g_launches.fetch_add(1); }

#define SG_LAUNCH_CHECK()                                                        \
    do {                                                                         \
        sgk_count_launch();                                                      \
        cudaError_t e_ = cudaGetLastError();                                     \
        if (e_ != cudaSuccess) {                                                 \
            sg_set_error(std::string("kernel launch failed: ") + cudaGetErrorString(e_)); \
            return SG_ECUDA;                                                     \
        }                                                                        \
    } while (0)

// ------------------------------------------------------------------------------------ init
// O4: sigma_p[w] = x0 | x1<<32 of P(orig[p], w, 0, tag 1), stored gauge-transformed (^ eps); N here = number of positions
__global__ void __launch_bounds__(256) k_init_spins(uint64_t *__restrict__ spin, const uint32_t *__restrict__ orig,
                                                    const uint64_t *__restrict__ eps, uint64_t n, uint32_t W, uint32_t word0, int aligned,
                                                    uint32_t k0, uint32_t k1)
{
    for (uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t p = q / W;
        const uint32_t w = (uint32_t)(q % W);
        const uint32_t site = orig ? orig[p] : (uint32_t)p;
        if (site == SG_NONE) { spin[q] = 0; continue; }   // padding position
        uint32_t x[4] = {0, 0, 0, 0};
        if (!aligned) philox4x32_10(site, word0 + w, 0u, 1u << 24, k0, k1, x);      // aligned start: every spin +1 (bit 0)
        spin[q] = ((uint64_t)x[0] | ((uint64_t)x[1] << 32)) ^ (eps ? eps[q] : 0ull);
    }
}

static unsigned grid_for(uint64_t n, unsigned per_block)
{
    const uint64_t b = (n + per_block - 1) / per_block;
    return (unsigned)std::min<uint64_t>(std::max<uint64_t>(b, 1), 1u << 20);     // grid-stride beyond 2^20 blocks
}

int sgk_init_spins(uint64_t *spin, const uint32_t *orig, const uint64_t *eps, uint64_t N, uint32_t W, uint32_t word0, bool aligned, SGSeed key,
                   cudaStream_t st)
{
    const uint64_t n = N * W;
    k_init_spins<<<grid_for(n, 256), 256, 0, st>>>(spin, orig, eps, n, W, word0, aligned ? 1 : 0, key.k0, key.k1);
    SG_LAUNCH_CHECK();
    return SG_OK;
}

// ------------------------------------------------------------------------------------ correlation
// counts[w*64+b] += #{ sites : bit b of (a ^ b)[site*W+w] set }.
// CONTIG (W a power of two <= 32): a warp reads 32 consecutive words; lane's word index is lane % W.
// otherwise: blockIdx.y = w, a warp reads word w of 32 consecutive sites (stride W).
template <bool CONTIG>
__global__ void __launch_bounds__(256)
k_xor_popcount(const uint64_t *__restrict__ a, const uint64_t *__restrict__ b, uint64_t n_sites, uint32_t W,
               unsigned long long *__restrict__ counts)
{
    constexpr int P = 6, PT = P + 5;
    uint64_t acc[PT];
    vc_clear(acc);
    const uint32_t lane = threadIdx.x & 31u;
    const uint64_t warp = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint64_t nwarps = ((uint64_t)gridDim.x * blockDim.x) >> 5;
    const uint64_t pol_stream = policy_evict_first();
    const uint64_t total = CONTIG ? n_sites * W : n_sites;
    const uint64_t nchunks = (total + 31) / 32;
    const uint32_t w_fixed = CONTIG ? 0u : blockIdx.y;
    const uint32_t G = CONTIG ? W : 1u;
    uint32_t pending = 0;
    constexpr int U = 4;                       // chunks per iteration: 2*U loads in flight per thread
    for (uint64_t ch = warp; ch < nchunks; ch += (uint64_t)U * nwarps) {
        uint64_t x[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint64_t q = (ch + (uint64_t)u * nwarps) * 32 + lane;
            x[u] = 0;
            if (q < total) {
                const uint64_t idx = CONTIG ? q : q * W + w_fixed;
                x[u] = ld_plain_u64(a + idx) ^ ld_stream_u64(b + idx, pol_stream);
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) vc_add_bit<P, PT>(acc, x[u]);
        pending += U;
        if (pending + U > (1u << P) - 1u) {
            vc_warp_flush<PT>(acc, G, w_fixed, counts);
            vc_clear(acc);
            pending = 0;
        }
    }
    if (pending) vc_warp_flush<PT>(acc, G, w_fixed, counts);
}

int sgk_xor_popcount(const uint64_t *a, const uint64_t *b, uint64_t n_sites, uint32_t W, uint64_t *counts, cudaStream_t st)
{
    const bool contig = W <= 32 && (W & (W - 1)) == 0;
    const uint64_t total = contig ? n_sites * W : n_sites;
    uint64_t blocks = (total + 32 * 8 * 16 - 1) / (32 * 8 * 16);   // >= 16 chunks per warp when large
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    if (contig) {
        k_xor_popcount<true><<<(unsigned)blocks, 256, 0, st>>>(a, b, n_sites, W, (unsigned long long *)counts);
    } else {
        dim3 grid((unsigned)std::max<uint64_t>(1, blocks / W), W);
        k_xor_popcount<false><<<grid, 256, 0, st>>>(a, b, n_sites, W, (unsigned long long *)counts);
    }
    SG_LAUNCH_CHECK();
    return SG_OK;
}

// ------------------------------------------------------------------------------------ correlation without allocation
// sg_correlation_noalloc (include/sg.h): the per-lane counters that k_xor_popcount adds to live in a file-scope device
// array instead of a buffer of the handle.  Every GPU that loads the library holds these 32 KiB until exit.  In host code
// the array's NAME is a host-side stand-in, not a device address: its address on the current device comes from
// cudaGetSymbolAddress, once per device with that device current.  All calls share the array: it is cleared at the start of
// each call, and calls that overlap on the GPU (other streams, other host threads) race.
static __device__ __align__(256) unsigned long long g_noalloc_counts[64 * SG_NOALLOC_MAX_WORDS];

int sgk_xor_popcount_noalloc(const uint64_t *a, const uint64_t *b, uint64_t n_sites, uint32_t W, uint64_t *out_host, cudaStream_t st)
{
    if (W == 0 || W > SG_NOALLOC_MAX_WORDS) {
        sg_set_error("sg_correlation_noalloc: n_words exceeds the static scratch (at most " + std::to_string(SG_NOALLOC_MAX_WORDS) + " words per site)");
        return SG_EINVAL;
    }
    constexpr int MAX_DEV = 64;
    static unsigned long long *addr[MAX_DEV] = {nullptr};     // the array's device address, per device
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEV) { sg_set_error("sg_correlation_noalloc: no usable current device"); return SG_ECUDA; }
    if (!addr[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_counts);
        if (e != cudaSuccess || !p) { sg_set_error(std::string("sg_correlation_noalloc: cudaGetSymbolAddress failed: ") + cudaGetErrorString(e)); return SG_ECUDA; }
        addr[dev] = static_cast<unsigned long long *>(p);
    }
    unsigned long long *counts = addr[dev];
    const size_t bytes = (size_t)64 * W * sizeof(unsigned long long);
    cudaError_t e = cudaMemsetAsync(counts, 0, bytes, st);      // the array keeps the last call's counts
    if (e != cudaSuccess) { sg_set_error(std::string("sg_correlation_noalloc: ") + cudaGetErrorString(e)); return SG_ECUDA; }
    const int rc = sgk_xor_popcount(a, b, n_sites, W, reinterpret_cast<uint64_t *>(counts), st);
    if (rc) return rc;
    e = cudaMemcpyAsync(out_host, counts, bytes, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { sg_set_error(std::string("sg_correlation_noalloc: ") + cudaGetErrorString(e)); return SG_ECUDA; }
    return SG_OK;
}

// The same against S stored configurations in one pass over the current one (the windowed protocol of PAPER.md:95,
// :270 counts against every stored waiting time after every sweep): 8 + 8 S bytes per site-word instead of 16 S.
// W a power of two <= 32; counts are added to S separate rows.
template <int S>
__global__ void __launch_bounds__(256, 2)
k_xor_popcount_multi(const uint64_t *__restrict__ a, const uint64_t *__restrict__ b0, const uint64_t *__restrict__ b1,
                     const uint64_t *__restrict__ b2, uint64_t total, uint32_t W, unsigned long long *__restrict__ c0,
                     unsigned long long *__restrict__ c1, unsigned long long *__restrict__ c2)
{
    // 102 registers, two CTAs per SM: measured faster (0.133 ms per three-slot pass at N = 2^24) than a variant that keeps
    // only P planes live and runs three CTAs per SM at 80 registers (0.140 ms)
    constexpr int P = 6, PT = P + 5;
    uint64_t acc[S][PT];
#pragma unroll
    for (int s = 0; s < S; ++s) vc_clear(acc[s]);
    const uint64_t *b[3] = {b0, b1, b2};
    unsigned long long *c[3] = {c0, c1, c2};
    const uint32_t lane = threadIdx.x & 31u;
    const uint64_t warp = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint64_t nwarps = ((uint64_t)gridDim.x * blockDim.x) >> 5;
    const uint64_t pol_stream = policy_evict_first();
    const uint64_t nchunks = (total + 31) / 32;
    uint32_t pending = 0;
    constexpr int U = 4;                       // chunks per iteration: (1 + S) * U loads in flight per thread
    for (uint64_t ch = warp; ch < nchunks; ch += (uint64_t)U * nwarps) {
        uint64_t x[U], y[S][U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint64_t q = (ch + (uint64_t)u * nwarps) * 32 + lane;
            x[u] = 0;
#pragma unroll
            for (int s = 0; s < S; ++s) y[s][u] = 0;
            if (q < total) {
                x[u] = ld_plain_u64(a + q);
#pragma unroll
                for (int s = 0; s < S; ++s) y[s][u] = ld_stream_u64(b[s] + q, pol_stream);
            }
        }
        // four one-bit numbers per lane into the counter: two carry-save adders into plane 0, one into plane 1,
        // then the carry ripples from plane 2
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const uint64_t d0 = x[0] ^ y[s][0], d1 = x[1] ^ y[s][1], d2 = x[2] ^ y[s][2], d3 = x[3] ^ y[s][3];
            uint64_t ones = acc[s][0];
            const uint64_t ta = maj64(ones, d0, d1);
            ones ^= d0 ^ d1;
            const uint64_t tb = maj64(ones, d2, d3);
            ones ^= d2 ^ d3;
            acc[s][0] = ones;
            const uint64_t twos = acc[s][1];
            uint64_t carry = maj64(twos, ta, tb);
            acc[s][1] = twos ^ ta ^ tb;
#pragma unroll
            for (int p = 2; p < P; ++p) {
                const uint64_t t = acc[s][p] & carry;
                acc[s][p] ^= carry;
                carry = t;
            }
        }
        pending += U;
        if (pending + U > (1u << P) - 1u) {
#pragma unroll
            for (int s = 0; s < S; ++s) { vc_warp_flush<PT>(acc[s], W, 0, c[s]); vc_clear(acc[s]); }
            pending = 0;
        }
    }
    if (pending) {
#pragma unroll
        for (int s = 0; s < S; ++s) vc_warp_flush<PT>(acc[s], W, 0, c[s]);
    }
}

// counts[s][64*W] += D(a, b[s]) for s < n (n <= 3); falls back to one pass per slot when W is not a power of two <= 32
int sgk_xor_popcount_multi(const uint64_t *a, const uint64_t *const *b, uint32_t n, uint64_t n_sites, uint32_t W, uint64_t *const *counts,
                           cudaStream_t st)
{
    const bool contig = W <= 32 && (W & (W - 1)) == 0;
    if (!contig || n == 1) {
        for (uint32_t s = 0; s < n; ++s) {
            const int rc = sgk_xor_popcount(a, b[s], n_sites, W, counts[s], st);
            if (rc) return rc;
        }
        return SG_OK;
    }
    const uint64_t total = n_sites * W;
    // a grid-stride kernel: exactly the CTAs that are resident at once (one wave), or fewer for small inputs
    static int per_sm[2] = {0, 0}, n_sm = 0;
    if (n_sm == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[0], k_xor_popcount_multi<2>, 256, 0);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[1], k_xor_popcount_multi<3>, 256, 0);
    }
    uint64_t blocks = (total + 32 * 8 * 16 - 1) / (32 * 8 * 16);
    const uint64_t wave = (uint64_t)n_sm * (uint64_t)std::max(1, per_sm[n == 2 ? 0 : 1]);
    if (blocks > wave) blocks = wave;
    if (blocks < 1) blocks = 1;
    auto cc = [&](uint32_t s) { return (unsigned long long *)counts[s < n ? s : 0]; };
    auto bb = [&](uint32_t s) { return b[s < n ? s : 0]; };
    if (n == 2) k_xor_popcount_multi<2><<<(unsigned)blocks, 256, 0, st>>>(a, bb(0), bb(1), bb(1), total, W, cc(0), cc(1), cc(1));
    else k_xor_popcount_multi<3><<<(unsigned)blocks, 256, 0, st>>>(a, bb(0), bb(1), bb(2), total, W, cc(0), cc(1), cc(2));
    SG_LAUNCH_CHECK();
    return SG_OK;
}

// ------------------------------------------------------------------------------------ relabelling helper
// n = number of words P*W (padding positions included); map = orig; eps = the gauge (position order) or nullptr
// scatter: dst[map[p]*W + w] = src[p*W + w] ^ eps[p*W + w]   (device order -> original order and gauge)
// gather : dst[p*W + w] = src[map[p]*W + w] ^ eps[p*W + w]   (original order and gauge -> device order)
__global__ void __launch_bounds__(256) k_permute_words(const uint64_t *__restrict__ src, uint64_t *__restrict__ dst,
                                                       const uint32_t *__restrict__ map, const uint64_t *__restrict__ eps,
                                                       uint64_t n, uint32_t W, int scatter)
{
    for (uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t p = q / W;
        const uint32_t w = (uint32_t)(q % W);
        const uint32_t m = map[p];
        if (m == SG_NONE) {            // padding position: nothing to export, stays 0 on import
            if (!scatter) dst[q] = 0;
            continue;
        }
        const uint64_t other = (uint64_t)m * W + w;
        const uint64_t e = eps ? eps[q] : 0ull;
        if (scatter) dst[other] = src[q] ^ e;
        else dst[q] = src[other] ^ e;
    }
}

int sgk_permute_words(const uint64_t *src, uint64_t *dst, const uint32_t *map, const uint64_t *eps, uint64_t N, uint32_t W, bool scatter,
                      cudaStream_t st)
{
    const uint64_t n = N * W;
    k_permute_words<<<grid_for(n, 256), 256, 0, st>>>(src, dst, map, eps, n, W, scatter ? 1 : 0);
    SG_LAUNCH_CHECK();
    return SG_OK;
}
