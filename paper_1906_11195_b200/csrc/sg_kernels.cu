// sg_kernels.cu -- CUDA kernels (sm_100a) of the Viana-Bray path besides the sweep (sg_vb_sweep.cu):
// initial spins and couplings (a1, a2 of SURVEY.md 8(a)), the correlation counts (a6)
// and the energy (a7).
// Conventions: DESIGN.md section 3.  All arithmetic is integer / bitwise.
#include <cuda_runtime.h>

#include <atomic>

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
// O4: sigma_p[w] = x0 | x1<<32 of P(orig[p], w, 0, tag 1); N here = number of positions
__global__ void __launch_bounds__(256) k_init_spins(uint64_t *__restrict__ spin, const uint32_t *__restrict__ orig,
                                                    uint64_t N, uint32_t W, uint32_t k0, uint32_t k1)
{
    const uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= N * W) return;
    const uint64_t p = q / W;
    const uint32_t w = (uint32_t)(q % W);
    const uint32_t site = orig ? orig[p] : (uint32_t)p;
    if (site == SG_NONE) { spin[q] = 0; return; }   // padding position
    uint32_t x[4];
    philox4x32_10(site, w, 0u, 1u << 24, k0, k1, x);
    spin[q] = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
}

// O3: kappa_e[w] = x0 | x1<<32 of P(e, w, 0, tag 2); padding entries get 0
__global__ void __launch_bounds__(256) k_init_vb_couplings(uint64_t *__restrict__ J, const uint32_t *__restrict__ eid,
                                                           uint64_t entries, uint32_t W, uint32_t k0, uint32_t k1)
{
    const uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= entries * W) return;
    // entry-major word-minor inside a 32-entry column: index = (ent32*32)*W + t, t = j*W + w
    const uint64_t col32 = q / (32ull * W);
    const uint32_t t = (uint32_t)(q % (32ull * W));
    const uint32_t j = t / W, w = t % W;
    const uint32_t e = eid[col32 * 32 + j];
    uint64_t v = 0;
    if (e != 0xFFFFFFFFu) {
        uint32_t x[4];
        philox4x32_10(e, w, 0u, 2u << 24, k0, k1, x);
        v = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
    }
    J[q] = v;
}

int sgk_init_spins(uint64_t *spin, const uint32_t *orig, uint64_t N, uint32_t W, SGSeed key, cudaStream_t st)
{
    const uint64_t n = N * W;
    k_init_spins<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(spin, orig, N, W, key.k0, key.k1);
    SG_LAUNCH_CHECK();
    return SG_OK;
}

int sgk_init_vb_couplings(uint64_t *J, const uint32_t *eid, uint64_t entries, uint32_t W, SGSeed key, cudaStream_t st)
{
    const uint64_t n = entries * W;
    if (n == 0) return SG_OK;
    k_init_vb_couplings<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(J, eid, entries, W, key.k0, key.k1);
    SG_LAUNCH_CHECK();
    return SG_OK;
}

// ------------------------------------------------------------------------------------ VB sweep
// One thread per (site, word) of one colour class.  Thread index T -> slice = T / (32 W),
// t = T % (32 W), site-in-slice j = t / W, word w = t % W.  Warps never straddle slices.
// Returns the 5 count planes of u = number of unsatisfied incident bonds for every lane.
struct Planes5 { uint64_t p0, p1, p2, p3, p4; };

__device__ __forceinline__ void csa4(uint64_t a, uint64_t b, uint64_t c, uint64_t d,
                                     uint64_t &s0, uint64_t &s1, uint64_t &s2)
{
    const uint64_t s = a ^ b ^ c;
    const uint64_t cy = (a & b) | (c & (a ^ b));
    s0 = s ^ d;
    const uint64_t c2 = s & d;
    s1 = cy ^ c2;
    s2 = cy & c2;
}

template <bool SPIN_HINT>
__device__ __forceinline__ Planes5 count_unsatisfied(const uint64_t *__restrict__ spin, const uint64_t *__restrict__ J,
                                                     const uint32_t *__restrict__ col, uint64_t ent_base /*32*slice_ptr*/,
                                                     uint32_t D, uint32_t j, uint32_t t, uint32_t w, uint32_t W,
                                                     uint64_t own, uint64_t pol_stream, uint64_t pol_keep)
{
    Planes5 P{0, 0, 0, 0, 0};
    for (uint32_t k = 0; k < D; k += 4) {
        uint32_t nb[4];
        uint64_t jw[4], sn[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (k + q < D) {
                const uint64_t ent = ent_base + 32ull * (k + q);
                nb[q] = ld_stream_u32(col + ent + j, pol_stream);
                jw[q] = ld_stream_u64(J + ent * W + t, pol_stream);
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (k + q < D) sn[q] = SPIN_HINT ? ld_keep_u64(spin + (uint64_t)(nb[q] & 0x7FFFFFFFu) * W + w, pol_keep)
                                     : ld_plain_u64(spin + (uint64_t)(nb[q] & 0x7FFFFFFFu) * W + w);
        uint64_t m[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) m[q] = (k + q < D) ? (own ^ sn[q] ^ jw[q]) : 0ull;
        uint64_t s0, s1, s2;
        csa4(m[0], m[1], m[2], m[3], s0, s1, s2);
        if (k == 0) {
            P.p0 = s0; P.p1 = s1; P.p2 = s2;
        } else {
            // P += (s2 s1 s0)
            const uint64_t c0 = P.p0 & s0;            P.p0 ^= s0;
            const uint64_t c1 = (P.p1 & s1) | (c0 & (P.p1 ^ s1));  P.p1 ^= s1 ^ c0;
            const uint64_t c2 = (P.p2 & s2) | (c1 & (P.p2 ^ s2));  P.p2 ^= s2 ^ c1;
            const uint64_t c3 = P.p3 & c2;            P.p3 ^= c2;
            P.p4 ^= c3;
        }
    }
    return P;
}

// lanes with u >= umin (bit-sliced comparison of the 5 planes against a per-thread scalar)
__device__ __forceinline__ uint64_t lanes_ge(const Planes5 &P, uint32_t umin)
{
    uint64_t gt = 0, eq = ~0ull;
    const uint64_t pl[5] = {P.p0, P.p1, P.p2, P.p3, P.p4};
#pragma unroll
    for (int b = 4; b >= 0; --b) {
        const uint64_t cb = ((umin >> b) & 1u) ? ~0ull : 0ull;
        gt |= eq & pl[b] & ~cb;
        eq &= ~(pl[b] ^ cb);
    }
    return gt | eq;
}

// ------------------------------------------------------------------------------------ per-lane counting
// Per-thread vertical counters: acc[p] holds bit p of 64 independent lane counters.
template <int P, int PT>
__device__ __forceinline__ void vc_add_bit(uint64_t (&acc)[PT], uint64_t x)
{
#pragma unroll
    for (int p = 0; p < P; ++p) {
        const uint64_t c = acc[p] & x;
        acc[p] ^= x;
        x = c;
    }
}

// acc += value given by 5 planes
template <int P, int PT>
__device__ __forceinline__ void vc_add_planes5(uint64_t (&acc)[PT], const Planes5 &v)
{
    const uint64_t in[5] = {v.p0, v.p1, v.p2, v.p3, v.p4};
    uint64_t carry = 0;
#pragma unroll
    for (int p = 0; p < P; ++p) {
        const uint64_t b = p < 5 ? in[p] : 0ull;
        const uint64_t a = acc[p];
        acc[p] = a ^ b ^ carry;
        carry = (a & b) | (carry & (a ^ b));
    }
}

// Sum the PT-plane counters of lanes that share a word index (lane % G, G a power of two <= 32)
// with an xor-shuffle tree, then add the per-lane totals to counts[(w_base + lane%G)*64 + bit].
// acc must have enough head-room planes for log2(32/G) doublings.
template <int PT>
__device__ __forceinline__ void vc_warp_flush(uint64_t (&acc)[PT], uint32_t G, uint32_t w_base,
                                              unsigned long long *__restrict__ counts)
{
    const uint32_t lane = threadIdx.x & 31u;
    for (uint32_t off = 16; off >= G; off >>= 1) {
        uint64_t carry = 0;
#pragma unroll
        for (int p = 0; p < PT; ++p) {
            const uint64_t a = acc[p];
            const uint64_t b = __shfl_xor_sync(0xFFFFFFFFu, a, off);
            acc[p] = a ^ b ^ carry;
            carry = (a & b) | (carry & (a ^ b));
        }
        if (off == 1) break;
    }
    for (uint32_t g = 0; g < G; ++g) {
        unsigned long long lo = 0, hi = 0;
#pragma unroll
        for (int p = 0; p < PT; ++p) {
            const uint64_t v = __shfl_sync(0xFFFFFFFFu, acc[p], g);
            lo += ((v >> lane) & 1ull) << p;
            hi += ((v >> (lane + 32u)) & 1ull) << p;
        }
        if (lo) atomicAdd(counts + (uint64_t)(w_base + g) * 64 + lane, lo);
        if (hi) atomicAdd(counts + (uint64_t)(w_base + g) * 64 + 32 + lane, hi);
    }
}

template <int PT>
__device__ __forceinline__ void vc_clear(uint64_t (&acc)[PT])
{
#pragma unroll
    for (int p = 0; p < PT; ++p) acc[p] = 0;
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

// ------------------------------------------------------------------------------------ VB energy
// counts[w*64+b] += sum over the class's sites of u_i (unsatisfied incident bonds of lane w*64+b).
// sum over all classes = 2 U_l, and E_l = 2 U_l - M.  One warp per slice-row of 32 threads, UNSAT_ROWS rows per
// warp; same thread -> (slice, j, w) map as the sweep.  Per-lane totals go
// to shared-memory counters first and to global memory once per CTA.
constexpr uint32_t UNSAT_ROWS = 4;
constexpr uint32_t UNSAT_SMEM_WORDS = 32;   // contiguous path: n_words <= 32

__global__ void __launch_bounds__(256, 3)
k_vb_unsat(const uint64_t *__restrict__ spin, const uint64_t *__restrict__ J, const uint32_t *__restrict__ col,
           const uint32_t *__restrict__ slice_ptr, uint64_t pos0, uint64_t n_sites, uint64_t slice0, uint64_t nslices,
           uint32_t W, unsigned long long *__restrict__ counts)
{
    constexpr int P = 3, PT = P + 5 + 5;   // UNSAT_ROWS additions of values <= 31, then 5 doublings in the warp
    __shared__ unsigned long long s_counts[64 * UNSAT_SMEM_WORDS];
    const bool contig = W <= UNSAT_SMEM_WORDS && (W & (W - 1)) == 0;
    if (contig) {
        for (uint32_t q = threadIdx.x; q < 64u * W; q += blockDim.x) s_counts[q] = 0;
        __syncthreads();
    }
    uint64_t acc[PT];
    vc_clear(acc);
    const uint32_t lane = threadIdx.x & 31u;
    const uint64_t warp = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint64_t pol_stream = policy_evict_first();
    const uint64_t pol_keep = policy_evict_normal();
    const uint32_t per_slice = 32u * W;
    const uint64_t nrows = nslices * W;           // warp-rows of 32 threads
#pragma unroll 1
    for (uint32_t it = 0; it < UNSAT_ROWS; ++it) {
        const uint64_t row = warp * UNSAT_ROWS + it;
        if (row >= nrows) break;
        const uint64_t T = row * 32 + lane;
        const uint64_t slice = T / per_slice;
        const uint32_t t = (uint32_t)(T % per_slice);
        const uint32_t j = t / W, w = t % W;
        const uint64_t local = slice * 32 + j;
        Planes5 u{0, 0, 0, 0, 0};
        if (local < n_sites) {
            const uint64_t p = pos0 + local;
            const uint32_t sp0 = __ldg(slice_ptr + slice0 + slice), sp1 = __ldg(slice_ptr + slice0 + slice + 1);
            const uint64_t own = ld_plain_u64(spin + p * W + w);
            u = count_unsatisfied<false>(spin, J, col, 32ull * sp0, sp1 - sp0, j, t, w, W, own, pol_stream, pol_keep);
        }
        if (contig) {
            vc_add_planes5<P + 5, PT>(acc, u);
        } else {
            // arbitrary W: lanes of a warp hold different words with no shuffle-friendly pattern;
            // flush every lane on its own (slow path, exact).
            const uint64_t pl[5] = {u.p0, u.p1, u.p2, u.p3, u.p4};
            for (int b = 0; b < 64; ++b) {
                unsigned long long v = 0;
#pragma unroll
                for (int q = 0; q < 5; ++q) v += ((pl[q] >> b) & 1ull) << q;
                if (v) atomicAdd(counts + (uint64_t)w * 64 + b, v);
            }
        }
    }
    if (contig) {
        vc_warp_flush<PT>(acc, W, 0, s_counts);
        __syncthreads();
        for (uint32_t q = threadIdx.x; q < 64u * W; q += blockDim.x)
            if (s_counts[q]) atomicAdd(counts + q, s_counts[q]);
    }
}

int sgk_vb_unsat_class(const VBDevice &d, const VBClass &c, uint32_t W, uint64_t *counts, cudaStream_t st)
{
    if (c.n == 0) return SG_OK;
    const uint64_t rows = c.nslices * W;
    const uint64_t blocks = (rows + 8 * UNSAT_ROWS - 1) / (8 * UNSAT_ROWS);
    k_vb_unsat<<<(unsigned)blocks, 256, 0, st>>>(d.spin, d.J, d.col, d.slice_ptr, c.pos0, c.n, c.slice0, c.nslices, W,
                                                 (unsigned long long *)counts);
    SG_LAUNCH_CHECK();
    return SG_OK;
}

// ------------------------------------------------------------------------------------ relabelling helper
// N = number of positions (padding included); map = orig
// scatter: dst[map[p]*W + w] = src[p*W + w]   (position order -> original order)
// gather : dst[p*W + w] = src[map[p]*W + w]   (original order -> position order)
__global__ void __launch_bounds__(256) k_permute_words(const uint64_t *__restrict__ src, uint64_t *__restrict__ dst,
                                                       const uint32_t *__restrict__ map, uint64_t N, uint32_t W, int scatter)
{
    const uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= N * W) return;
    const uint64_t p = q / W;
    const uint32_t w = (uint32_t)(q % W);
    const uint32_t m = map[p];
    if (m == SG_NONE) {            // padding position: nothing to export, stays 0 on import
        if (!scatter) dst[q] = 0;
        return;
    }
    const uint64_t other = (uint64_t)m * W + w;
    if (scatter) dst[other] = src[q];
    else dst[q] = src[other];
}

int sgk_permute_words(const uint64_t *src, uint64_t *dst, const uint32_t *map, uint64_t N, uint32_t W, bool scatter, cudaStream_t st)
{
    const uint64_t n = N * W;
    k_permute_words<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(src, dst, map, N, W, scatter ? 1 : 0);
    SG_LAUNCH_CHECK();
    return SG_OK;
}
