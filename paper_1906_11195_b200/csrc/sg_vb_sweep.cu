// sg_vb_sweep.cu -- the hot kernel: one colour class of one Viana-Bray Metropolis sweep
// (row a3 of SURVEY.md 8(a); PAPER.md:260 "classic single spin flip Metropolis", :318-320 kernel prose).
// Conventions: DESIGN.md section 3 (O7, Q14).
//
// One thread per (site, word), SG_BT threads per CTA.  m_e = own ^ neighbour ^ coupling (bit = bond unsatisfied) for
// every incident edge, u = per-lane sum of the m_e in 5 bit planes (carry-save adders), one Philox draw r shared by the 64
// lanes, kstar = #{k >= 1 : r < thr[k]}, flip the lanes with u >= ceil((d - kstar)/2).  No floating point.
//
// Memory behaviour (B200, profiles/r01_probes.md): couplings, neighbour indices and site labels are read once
// per sweep, coalesced, and stream through L2 (evict_first, no L1 allocation).  The neighbour spin words are
// 8-byte gathers: they cost one L1TEX wavefront each and, when they miss L2, a whole 128-byte line from HBM each,
// which is what bounds the sweep.  The host generator therefore orders the sites of a class by breadth-first index
// (sg_host.cpp), so that the gathers along tree edges stay inside a moving window of every other class's block.
#include <cuda_runtime.h>

#include <cstdlib>
#include <string>

#include "sg_device.cuh"
#include "sg_internal.h"

void sgk_count_launch();

namespace {
// threads per CTA: 128 (4 slices) measures 3 % faster than 256 and 14 % faster than 512; 64 equals 128 (profiles/r01_sweep.md)
#ifndef SG_BT
#define SG_BT 128
#endif

__device__ __forceinline__ uint64_t maj64(uint64_t a, uint64_t b, uint64_t c) { return (a & b) | (c & (a ^ b)); }

// index type: 32-bit when every index of the instance fits, else 64-bit
template <bool WIDE> struct Idx { using type = uint32_t; };
template <> struct Idx<true> { using type = uint64_t; };

// LOGW >= 0: n_words = 2^LOGW (compile time); LOGW < 0: n_words = Wrt (run time)
template <int LOGW, bool WIDE, int MINB>
__global__ void __launch_bounds__(SG_BT, (MINB * 256) / SG_BT)
k_vb_sweep(uint64_t *__restrict__ spin, const uint64_t *__restrict__ J, const uint32_t *__restrict__ col,
           const uint32_t *__restrict__ orig, const uint32_t *__restrict__ slice_ptr, const uint64_t *__restrict__ thr,
           uint32_t pos0, uint32_t slice0, uint32_t nslices, uint32_t Wrt, uint32_t sweep_lo, uint32_t sweep_hi, uint32_t k0, uint32_t k1,
           uint32_t reverse)
{
    using I = typename Idx<WIDE>::type;
    const uint32_t bid = reverse ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
    const uint32_t W = LOGW >= 0 ? (1u << (LOGW >= 0 ? LOGW : 0)) : Wrt;
    // `reverse`: walk the class from its last slice to its first (the host alternates the direction from launch to
    // launch, so that a launch starts where the previous one ended and finds those spin words still in L2)
    const I T = (I)bid * (uint32_t)SG_BT + threadIdx.x;
    const uint32_t per_slice = 32u * W;
    const uint32_t slice = LOGW >= 0 ? (uint32_t)(T >> (5 + (LOGW >= 0 ? LOGW : 0))) : (uint32_t)(T / per_slice);
    // (no thread leaves before griddep_wait(): ptxas hoists the wait above every load that follows an exit)
    const bool in_range = slice < nslices;
    const uint32_t t = LOGW >= 0 ? (uint32_t)T & (per_slice - 1u) : (uint32_t)(T % per_slice);
    const uint32_t j = LOGW >= 0 ? t >> (LOGW >= 0 ? LOGW : 0) : t / W;
    const uint32_t w = LOGW >= 0 ? t & (W - 1u) : t % W;
    const uint32_t p = pos0 + slice * 32u + j;
    const uint64_t pol_stream = policy_evict_first();

    const uint32_t site = in_range ? ld_stream_u32(orig + p, pol_stream) : SG_NONE;   // SG_NONE: padding position
    uint32_t sp0 = 0, sp1 = 0;
    if (in_range) { sp0 = __ldg(slice_ptr + slice0 + slice); sp1 = __ldg(slice_ptr + slice0 + slice + 1); }
    const uint32_t D = site != SG_NONE ? sp1 - sp0 : 0u;  // row length of the slice >= degree of this site
    uint64_t *own_ptr = spin + (I)p * W + w;

    const uint32_t *cp = col + (I)sp0 * 32u + j;          // + 32 per neighbour slot
    const uint64_t *jp = J + (I)sp0 * 32u * W + t;         // + 32 W per neighbour slot
    // neighbour indices and coupling words of slots k .. k+3 (padding: own position, coupling 0)
    auto load_chunk = [&](uint32_t k, uint32_t (&nb)[4], uint64_t (&jw)[4]) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            nb[q] = p;
            jw[q] = 0;
            if (k + q < D) {
                nb[q] = ld_stream_u32(cp + (I)(k + q) * 32u, pol_stream);
                jw[q] = ld_stream_u64(jp + (I)(k + q) * per_slice, pol_stream);
            }
        }
    };
    uint32_t nb[4];
    uint64_t jw[4];
    load_chunk(0, nb, jw);
    // r = x_{w&3} of P(site, w>>2, sweep, tag 0): the ten Philox rounds run while the row loads are in flight
    uint32_t x[4];
    philox4x32_10(site, w >> 2, sweep_lo, sweep_hi, k0, k1, x);
    const uint32_t r = (LOGW == 0) ? x[0] : ((w & 2u) ? ((w & 1u) ? x[3] : x[2]) : ((w & 1u) ? x[1] : x[0]));
    // thr[k] is non-increasing in k, so r < thr[kk] <=> kk <= kall := #{k >= 1 : r < thr[k]} (thr[k] = 0 beyond dmax)
    uint32_t kall = 0;
    while (kall < 31u && (uint64_t)r < __ldg(thr + kall + 1)) ++kall;
    // Everything above reads arrays that no kernel writes.  The launch is a programmatic dependent launch: this
    // grid's CTAs start while the previous colour class is still draining and wait here, before the first spin
    // word is read, until that grid has completed and its writes are visible.
    // (ptxas hoists the wait above every global load that no thread exit separates from it; this exit, never taken
    // because indices are positions < 2^31, depends on the row loads and so pins them before the wait)
    if ((nb[0] & nb[1] & nb[2] & nb[3]) == SG_NONE || site == SG_NONE) return;
    griddep_wait();
    griddep_launch_dependents();
    const uint64_t own = *own_ptr;

    uint64_t p0 = 0, p1 = 0, p2 = 0, p3 = 0, p4 = 0;
    uint32_t d = 0;
    for (uint32_t k = 0; k < D; k += 4) {
        uint64_t sn[4], jc[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            sn[q] = own;                                   // padding entry: own ^ own ^ 0 = satisfied
            jc[q] = jw[q];
            if (nb[q] != p) { sn[q] = spin[(I)nb[q] * W + w]; ++d; }
        }
        if (k + 4 < D) load_chunk(k + 4, nb, jw);          // next slots' streams go out under the gathers' latency
        uint64_t m[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) m[q] = own ^ sn[q] ^ jc[q];
        // 4 one-bit numbers -> 3 planes
        const uint64_t s = m[0] ^ m[1] ^ m[2], cy = maj64(m[0], m[1], m[2]);
        const uint64_t s0 = s ^ m[3], c2 = s & m[3];
        const uint64_t s1 = cy ^ c2, s2 = cy & c2;
        if (k == 0) {
            p0 = s0; p1 = s1; p2 = s2;
        } else {
            const uint64_t c0 = p0 & s0;             p0 ^= s0;
            const uint64_t c1 = maj64(p1, s1, c0);   p1 ^= s1 ^ c0;
            const uint64_t c2b = maj64(p2, s2, c1);  p2 ^= s2 ^ c1;
            const uint64_t c3 = p3 & c2b;            p3 ^= c2b;
            p4 ^= c3;
        }
    }

    // flip <=> kk = d - 2u <= kstar <=> u >= ceil((d - kstar)/2)
    const uint32_t kstar = min(kall, d);
    const uint32_t umin = (d - kstar + 1u) >> 1;
    uint64_t gt = 0, eq = ~0ull;
    const uint64_t pl[5] = {p0, p1, p2, p3, p4};
#pragma unroll
    for (int b = 4; b >= 0; --b) {
        const uint64_t cb = ((umin >> b) & 1u) ? ~0ull : 0ull;
        gt |= eq & pl[b] & ~cb;
        eq &= ~(pl[b] ^ cb);
    }
    const uint64_t flip = gt | eq;
    if (flip) *own_ptr = own ^ flip;
}

template <int LOGW, bool WIDE, int MINB>
int launch(const VBDevice &d, const VBClass &c, uint32_t W, uint64_t sweep, SGSeed key, bool reverse, cudaStream_t st)
{
    const uint64_t threads = c.nslices * 32ull * W;
    const unsigned grid = (unsigned)((threads + SG_BT - 1) / SG_BT);
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(SG_BT);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddep_wait() in the kernel
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    static const bool no_pdl = std::getenv("SG_NO_PDL") != nullptr;   // measurement knob
    cfg.numAttrs = no_pdl ? 0 : 1;
    const cudaError_t le = cudaLaunchKernelEx(&cfg, k_vb_sweep<LOGW, WIDE, MINB>, d.spin, (const uint64_t *)d.J, (const uint32_t *)d.col,
                                              (const uint32_t *)d.orig, (const uint32_t *)d.slice_ptr, (const uint64_t *)d.thr, (uint32_t)c.pos0,
                                              (uint32_t)c.slice0, (uint32_t)c.nslices, W, (uint32_t)sweep, (uint32_t)(sweep >> 32) /* tag 0 */,
                                              key.k0, key.k1, reverse ? 1u : 0u);
    sgk_count_launch();
    const cudaError_t e = le != cudaSuccess ? le : cudaGetLastError();
    if (e != cudaSuccess) {
        sg_set_error(std::string("k_vb_sweep launch failed: ") + cudaGetErrorString(e));
        return SG_ECUDA;
    }
    return SG_OK;
}

}  // namespace

int sgk_vb_sweep_class(const VBDevice &d, const VBClass &c, uint64_t P, uint64_t entries, uint32_t W, uint64_t sweep, SGSeed key,
                       bool reverse, cudaStream_t st)
{
    if (c.n == 0) return SG_OK;
    if (c.nslices * 32ull * W >= (1ull << 40)) { sg_set_error("sgk_vb_sweep_class: class too large"); return SG_EINVAL; }
    const bool narrow = P * W < (1ull << 32) && entries * W < (1ull << 32);
    // 1280 threads per SM: 48 registers, no spills (1536 spill, 1024 lose latency hiding; profiles/r01_sweep.md)
    if (narrow) {
        switch (W) {
        case 1: return launch<0, false, 5>(d, c, W, sweep, key, reverse, st);
        case 2: return launch<1, false, 5>(d, c, W, sweep, key, reverse, st);
        case 4: return launch<2, false, 5>(d, c, W, sweep, key, reverse, st);
        case 8: return launch<3, false, 5>(d, c, W, sweep, key, reverse, st);
        case 16: return launch<4, false, 5>(d, c, W, sweep, key, reverse, st);
        default: return launch<-1, false, 4>(d, c, W, sweep, key, reverse, st);
        }
    }
    return launch<-1, true, 4>(d, c, W, sweep, key, reverse, st);
}
