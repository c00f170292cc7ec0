// sg_vb_sweep.cu -- the hot kernel: one colour class of one Viana-Bray Metropolis sweep
// (row a3 of SURVEY.md 8(a); PAPER.md:260 "classic single spin flip Metropolis", :318-320 kernel prose).
// Specialised for n_words = 2^LOGW <= 16 with 32-bit index arithmetic; sg_kernels.cu keeps the
// general-W kernel.  Conventions: DESIGN.md section 3 (O7, Q14).
//
// Per (site, word): m_e = own ^ neighbour ^ coupling (bit = bond unsatisfied) for every incident edge,
// u = per-lane sum of the m_e in 5 bit planes (carry-save adders), one Philox draw r shared by the
// 64 lanes, kstar = #{k >= 1 : r < thr[k]}, flip the lanes with u >= ceil((d - kstar)/2).
//
// Memory behaviour (B200): couplings, neighbour indices and per-site metadata are read once per
// sweep and stream through L2 with evict_first; the spin array is gathered at random, 8 useful
// bytes per 32-byte sector.  It does not fit the part of L2 a single SM can use for data shared
// by all SMs, so only the spins of high-degree sites (gathered d times per sweep) are kept with
// evict_last: bit 31 of a neighbour index marks such a "hot" neighbour (set by the host generator).
#include <cuda_runtime.h>

#include <cstdlib>

#include "sg_device.cuh"
#include "sg_internal.h"

void sgk_count_launch();

namespace {

struct P5 { uint64_t p0, p1, p2, p3, p4; };

__device__ __forceinline__ uint64_t maj64(uint64_t a, uint64_t b, uint64_t c) { return (a & b) | (c & (a ^ b)); }

// policies are plain 64-bit descriptors; pick per access without a branch
__device__ __forceinline__ uint64_t pick(bool hot, uint64_t pol_hot, uint64_t pol_cold) { return hot ? pol_hot : pol_cold; }

template <int LOGW, int MINB>
__global__ void __launch_bounds__(256, MINB)
k_vb_sweep_w(uint64_t *__restrict__ spin, const uint64_t *__restrict__ J, const uint32_t *__restrict__ col,
             const uint32_t *__restrict__ orig, const uint32_t *__restrict__ slice_ptr,
             const uint64_t *__restrict__ thr, uint32_t pos0, uint32_t n_sites, uint32_t slice0, uint32_t nslices,
             uint32_t dhot, uint32_t sweep_lo, uint32_t sweep_hi, uint32_t k0, uint32_t k1)
{
    constexpr uint32_t W = 1u << LOGW;
    const uint32_t T = blockIdx.x * 256u + threadIdx.x;
    const uint32_t slice = T >> (5 + LOGW);
    if (slice >= nslices) return;
    const uint32_t t = T & (32u * W - 1u);
    const uint32_t j = t >> LOGW, w = t & (W - 1u);
    const uint32_t local = slice * 32u + j;
    if (local >= n_sites) return;
    const uint32_t p = pos0 + local;
    const uint64_t pol_stream = policy_evict_first();
    const uint64_t pol_hot = policy_evict_last();
    const uint64_t pol_cold = policy_evict_normal();

    const uint32_t sp0 = __ldg(slice_ptr + slice0 + slice), sp1 = __ldg(slice_ptr + slice0 + slice + 1);
    const uint32_t D = sp1 - sp0;
    const uint32_t d = D;   // slices hold sites of one degree
    const uint32_t site = ld_stream_u32(orig + p, pol_stream);
    if (site == SG_NONE) return;   // padding position
    uint64_t *own_ptr = spin + ((size_t)p << LOGW) + w;
    const uint64_t pol_own = pick(d >= dhot, pol_hot, pol_cold);
    const uint64_t own = ld_keep_u64(own_ptr, pol_own);

    const uint32_t *cp = col + (size_t)sp0 * 32u + j;            // + 32 per neighbour slot
    const uint64_t *jp = J + (((size_t)sp0 * 32u) << LOGW) + t;  // + 32 W per neighbour slot
    P5 P{0, 0, 0, 0, 0};
    for (uint32_t k = 0; k < D; k += 4) {
        uint32_t nb[4];
        uint64_t jw[4], sn[4];
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (k + q < D) {
                nb[q] = ld_stream_u32(cp + (k + q) * 32u, pol_stream);
                jw[q] = ld_stream_u64(jp + (size_t)(k + q) * (32u * W), pol_stream);
            }
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (k + q < D)
                sn[q] = ld_keep_u64(spin + ((size_t)(nb[q] & 0x7FFFFFFFu) << LOGW) + w, pick(nb[q] >> 31, pol_hot, pol_cold));
        uint64_t m[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) m[q] = (k + q < D) ? (own ^ sn[q] ^ jw[q]) : 0ull;
        // 4 one-bit numbers -> 3 planes
        const uint64_t s = m[0] ^ m[1] ^ m[2], cy = maj64(m[0], m[1], m[2]);
        const uint64_t s0 = s ^ m[3], c2 = s & m[3];
        const uint64_t s1 = cy ^ c2, s2 = cy & c2;
        if (k == 0) {
            P.p0 = s0; P.p1 = s1; P.p2 = s2;
        } else {
            const uint64_t c0 = P.p0 & s0;             P.p0 ^= s0;
            const uint64_t c1 = maj64(P.p1, s1, c0);   P.p1 ^= s1 ^ c0;
            const uint64_t c2b = maj64(P.p2, s2, c1);  P.p2 ^= s2 ^ c1;
            const uint64_t c3 = P.p3 & c2b;            P.p3 ^= c2b;
            P.p4 ^= c3;
        }
    }

    // r = x_{w&3} of P(site, w>>2, sweep, tag 0)
    uint32_t x[4];
    philox4x32_10(site, w >> 2, sweep_lo, sweep_hi, k0, k1, x);
    const uint32_t r = (W == 1) ? x[0] : ((w & 2u) ? ((w & 1u) ? x[3] : x[2]) : ((w & 1u) ? x[1] : x[0]));
    uint32_t kstar = 0;
    while (kstar < d && (uint64_t)r < __ldg(thr + kstar + 1)) ++kstar;
    const uint32_t umin = (d - kstar + 1u) >> 1;
    // lanes with u >= umin
    uint64_t gt = 0, eq = ~0ull;
    const uint64_t pl[5] = {P.p0, P.p1, P.p2, P.p3, P.p4};
#pragma unroll
    for (int b = 4; b >= 0; --b) {
        const uint64_t cb = ((umin >> b) & 1u) ? ~0ull : 0ull;
        gt |= eq & pl[b] & ~cb;
        eq &= ~(pl[b] ^ cb);
    }
    st_keep_u64(own_ptr, own ^ (gt | eq), pol_own);
}

template <int LOGW, int MINB>
int launch(const VBDevice &d, const VBClass &c, uint64_t sweep, SGSeed key, cudaStream_t st)
{
    const uint64_t threads = (c.nslices * 32ull) << LOGW;
    const unsigned grid = (unsigned)((threads + 255) / 256);
    k_vb_sweep_w<LOGW, MINB><<<grid, 256, 0, st>>>(d.spin, d.J, d.col, d.orig, d.slice_ptr, d.thr, (uint32_t)c.pos0, (uint32_t)c.n,
                                             (uint32_t)c.slice0, (uint32_t)c.nslices, d.dhot, (uint32_t)sweep,
                                             (uint32_t)(sweep >> 32) /* tag 0 */, key.k0, key.k1);
    sgk_count_launch();
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        sg_set_error(std::string("k_vb_sweep_w launch failed: ") + cudaGetErrorString(e));
        return SG_ECUDA;
    }
    return SG_OK;
}

}  // namespace

// true if the specialised kernel can run this shape (else the caller uses the general one)
bool sgk_vb_sweep_fast_ok(uint64_t N, uint64_t entries, uint32_t W)
{
    if (W > 16 || (W & (W - 1))) return false;
    return N * W < (1ull << 31) && entries * W < (1ull << 32);
}

int sgk_vb_sweep_class_fast(const VBDevice &d, const VBClass &c, uint32_t W, uint64_t sweep, SGSeed key, cudaStream_t st)
{
    if (c.n == 0) return SG_OK;
    static const int minb = [] { const char *e = std::getenv("SG_VB_MINB"); return e ? std::atoi(e) : 5; }();
    switch (W) {
    case 1:
        if (minb == 4) return launch<0, 4>(d, c, sweep, key, st);
        if (minb == 6) return launch<0, 6>(d, c, sweep, key, st);
        if (minb == 8) return launch<0, 8>(d, c, sweep, key, st);
        return launch<0, 5>(d, c, sweep, key, st);
    case 2: return launch<1, 5>(d, c, sweep, key, st);
    case 4: return launch<2, 5>(d, c, sweep, key, st);
    case 8: return launch<3, 5>(d, c, sweep, key, st);
    case 16: return launch<4, 5>(d, c, sweep, key, st);
    }
    sg_set_error("sgk_vb_sweep_class_fast: unsupported n_words");
    return SG_EINVAL;
}
