// sg_vb_sweep.cu -- the kernels that walk the rows of a Viana-Bray instance: the Metropolis sweep of one colour class
// (row a3 of SURVEY.md 8(a); PAPER.md:260 "classic single spin flip Metropolis", :318-320 kernel prose), the energy
// (a7) and the drawing of the coupling words (a1).  Conventions: DESIGN.md section 3 (O3, O7, Q14).
//
// One warp per (slice, group of G words); layout in sg_internal.h.  Two phases:
//   1. one lane per row ENTRY of the slice, 32 entries per step: neighbour index and (X entries) coupling word from the
//      coalesced streams, gather of the neighbour's spin word(s), x_e = spin ^ coupling (tree entries: no coupling
//      after the gauge transformation) parked in shared memory.  Every lane is busy whatever the degrees; consecutive
//      tree entries belong to consecutive sites in breadth-first order, so the lanes of a gather share 128-byte lines.
//   2. one lane per SITE: m_e = own ^ x_e (bit = bond unsatisfied), u = per-lane sum of the m_e in bit planes
//      (carry-save adders), one Philox draw r per word shared by its 64 lanes, kstar = #{k >= 1 : r < thr[k]}, flip the
//      lanes with u >= ceil((d - kstar)/2).  No floating point.
// G = 2 (even n_words): a thread owns two words of its entry / site: 16-byte accesses (LDG.128), one Philox call for the
// two words (Q6).  G = 4 (32-byte accesses, LDG.256, one Philox call for four words) is kept behind SG_VB_G=4: at
// 96 registers it is 25-30 % slower than G = 2.
//
// Memory behaviour (B200, profiles/): couplings, neighbour indices, labels and row pointers are read once per sweep,
// coalesced, and stream through L2 (evict_first, no L1 allocation).  The gathers cost one L1TEX wavefront per distinct
// 128-byte line of the warp's request, one L2 sector per distinct 32 bytes and, when they miss L2, a whole line from
// HBM.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdlib>
#include <string>

#include "sg_device.cuh"
#include "sg_internal.h"

void sgk_count_launch();

namespace {
#ifndef SG_BT
#define SG_BT 128      // threads per CTA = 4 warps = 4 (slice, word group) jobs
#endif
// resident CTAs per SM the one-word kernels are compiled for, by entry budget (it = 6, 8): 40 / 48 registers
#ifndef SG_MINB6
#define SG_MINB6 12
#endif
#ifndef SG_MINB8
#define SG_MINB8 10
#endif
constexpr int WARPS = SG_BT / 32;
// the never-taken exit in front of griddepcontrol.wait compares against this value: an AND of neighbour positions
// (all < 2^31 - 2) and SG_NONE fillers can never equal it
constexpr uint32_t PIN_IMPOSSIBLE = 0x7FFFFFFEu;

// index type: 32-bit when every index of the instance fits, else 64-bit
template <bool WIDE> struct Idx { using type = uint32_t; };
template <> struct Idx<true> { using type = uint64_t; };

// u (number of unsatisfied bonds) per lane of each of G words, as 5 bit planes
template <int G> struct Planes { uint64_t p[5][G]; };

// P = m[0] + ... + m[7] (one-bit numbers per lane): a carry-save tree, 14 three-input operations per word
template <int G>
__device__ __forceinline__ void planes_from8(Planes<G> &P, const Vec<G> (&a)[4], const Vec<G> (&b)[4])
{
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const uint64_t s1 = a[0].v[g] ^ a[1].v[g] ^ a[2].v[g], c1 = maj64(a[0].v[g], a[1].v[g], a[2].v[g]);
        const uint64_t s2 = a[3].v[g] ^ b[0].v[g] ^ b[1].v[g], c2 = maj64(a[3].v[g], b[0].v[g], b[1].v[g]);
        const uint64_t s3 = b[2].v[g] ^ b[3].v[g], c3 = b[2].v[g] & b[3].v[g];
        P.p[0][g] = s1 ^ s2 ^ s3;
        const uint64_t c4 = maj64(s1, s2, s3);
        const uint64_t t = c1 ^ c2 ^ c3, c5 = maj64(c1, c2, c3);
        P.p[1][g] = t ^ c4;
        const uint64_t c6 = t & c4;
        P.p[2][g] = c5 ^ c6;
        P.p[3][g] = c5 & c6;
        P.p[4][g] = 0;
    }
}

// P += m (a one-bit number per lane)
template <int G>
__device__ __forceinline__ void planes_add1(Planes<G> &P, const Vec<G> &m)
{
#pragma unroll
    for (int g = 0; g < G; ++g) {
        uint64_t c = m.v[g];
#pragma unroll
        for (int b = 0; b < 5; ++b) {
            const uint64_t t = P.p[b][g] & c;
            P.p[b][g] ^= c;
            c = t;
        }
    }
}

// shared-memory parking of x_e: G consecutive words per entry
template <int G> __device__ __forceinline__ void sm_store(uint64_t *s, uint32_t e, const Vec<G> &x)
{
    if constexpr (G == 1) {
        s[e] = x.v[0];
    } else {
#pragma unroll
        for (int g = 0; g < G; g += 2) *reinterpret_cast<ulonglong2 *>(s + (size_t)e * G + g) = make_ulonglong2(x.v[g], x.v[g + 1]);
    }
}
template <int G> __device__ __forceinline__ Vec<G> sm_load(const uint64_t *s, uint32_t e)
{
    Vec<G> x;
    if constexpr (G == 1) {
        x.v[0] = s[e];
    } else {
#pragma unroll
        for (int g = 0; g < G; g += 2) {
            const ulonglong2 t = *reinterpret_cast<const ulonglong2 *>(s + (size_t)e * G + g);
            x.v[g] = t.x; x.v[g + 1] = t.y;
        }
    }
    return x;
}

// ---- phase 1 ------------------------------------------------------------------------------------
// The stream part: neighbour positions of the slice's entries 32k + lane (SG_NONE beyond the run) and the coupling
// words of its X entries (the first nXs of the run).  Reads arrays that no kernel writes.
// IT / ITX: steps of 32 entries / of 32 X entries the slices of the class may need (VBClass::it, itx).
template <int G, int IT, int ITX, bool WIDE>
struct Streams {
    uint32_t nb[IT];
    Vec<G> jw[ITX];

    __device__ __forceinline__ void load(const uint32_t *__restrict__ col, const uint64_t *__restrict__ J, SGHdr h, uint32_t W, uint32_t w0, uint64_t pol)
    {
        using I = typename Idx<WIDE>::type;
        const uint32_t lane = threadIdx.x & 31u;
        const uint32_t nXs = (h.counts >> 6) & 1023u, nE = (h.counts >> 16) & 4095u;
        const uint32_t *c = col + h.col_off + lane;
        const uint64_t *jp = J + (I)(h.j_off + lane) * W + w0;
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            nb[k] = SG_NONE;
            if (32u * k + lane < nE) nb[k] = ld_stream_u32(c + 32 * k, pol);
        }
#pragma unroll
        for (int k = 0; k < ITX; ++k) {
#pragma unroll
            for (int g = 0; g < G; ++g) jw[k].v[g] = 0;
            if (32u * k + lane < nXs) jw[k] = ld_stream_vec<G>(jp + (I)(32u * k) * W, pol);
        }
    }
    // A value that can never equal PIN_IMPOSSIBLE and is known only when every stream load has returned.
    __device__ __forceinline__ uint32_t pin(uint32_t site, uint32_t rp) const
    {
        uint32_t a = nb[0];                                            // AND of positions (< 2^31 - 2) and SG_NONE fillers
#pragma unroll
        for (int k = 1; k < IT; ++k) a &= nb[k];
        uint32_t o = site | rp;
#pragma unroll
        for (int k = 0; k < ITX; ++k) o |= (uint32_t)(jw[k].v[G - 1] >> 32) | (uint32_t)jw[k].v[0];
        return a & (o | 0x7FFFFFFFu);
    }
    // the gather part: x_e = spin[neighbour] (^ coupling) into shared memory; all gathers in flight before the first store
    __device__ __forceinline__ void gather(const uint64_t *spin, uint32_t W, uint32_t w0, uint64_t *sx, uint32_t nXs) const
    {
        using I = typename Idx<WIDE>::type;
        const uint32_t lane = threadIdx.x & 31u;
        Vec<G> x[IT];
#pragma unroll
        for (int k = 0; k < IT; ++k)
            if (nb[k] != SG_NONE) {
                // X entries: one word of a random line, no reuse: kept out of L1 (.cg), which is measurably better than
                // any L1 hint (profiles/r02_sweep.md); T entries: neighbouring lanes, steps and slices share lines
                if constexpr (G == 1) {
                    if (k < ITX && 32u * k + lane < nXs) x[k].v[0] = ld_x_u64(spin + (I)nb[k] * W + w0);
                    else x[k].v[0] = ld_plain_u64(spin + (I)nb[k] * W + w0);
                } else {
                    x[k] = ld_plain_vec<G>(spin + (I)nb[k] * W + w0);
                }
            }
#pragma unroll
        for (int k = 0; k < IT; ++k)
            if (nb[k] != SG_NONE) {
                if (k < ITX) {
#pragma unroll
                    for (int g = 0; g < G; ++g) x[k].v[g] ^= jw[k].v[g];
                }
                sm_store<G>(sx, 32u * k + lane, x[k]);
            }
    }
};

// ---- phase 2 ------------------------------------------------------------------------------------
// u of the site whose row pointer is rp: its X entries sx[xOff ..], its T entries sx[tOff ..]
template <int G>
__device__ __forceinline__ void count_unsatisfied(const uint64_t *sx, uint32_t rp, const Vec<G> &own, Planes<G> &P)
{
    const uint32_t xOff = rp & 255u, tOff = (rp >> 8) & 511u, nX = (rp >> 17) & 31u, nT = rp >> 22;
    Vec<G> mT[4], mX[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
#pragma unroll
        for (int g = 0; g < G; ++g) mT[q].v[g] = mX[q].v[g] = 0;
        if ((uint32_t)q < nX) {
            mX[q] = sm_load<G>(sx, xOff + q);
#pragma unroll
            for (int g = 0; g < G; ++g) mX[q].v[g] ^= own.v[g];
        }
        if ((uint32_t)q < nT) {
            mT[q] = sm_load<G>(sx, tOff + q);
#pragma unroll
            for (int g = 0; g < G; ++g) mT[q].v[g] ^= own.v[g];
        }
    }
    planes_from8<G>(P, mT, mX);
    // long rows: one per-lane loop over the X entries beyond the fourth, then the T entries beyond the fourth
    const uint32_t eX = nX > 4u ? nX - 4u : 0u, eT = nT > 4u ? nT - 4u : 0u;
    for (uint32_t q = 0; q < eX + eT; ++q) {
        Vec<G> m = sm_load<G>(sx, q < eX ? xOff + 4u + q : tOff + 4u + (q - eX));
#pragma unroll
        for (int g = 0; g < G; ++g) m.v[g] ^= own.v[g];
        planes_add1<G>(P, m);
    }
}

// The same for a slice whose sites all have at most NS X entries and NS T entries (NS = 2 or 4; shapes 0 and 1 of
// sg_vb_shape): no loops, u <= 2 NS fits 3 / 4 planes (the planes above stay zero).
template <int G, int NS>
__device__ __forceinline__ void count_unsatisfied_short(const uint64_t *sx, uint32_t rp, const Vec<G> &own, Planes<G> &P)
{
    const uint32_t xOff = rp & 255u, tOff = (rp >> 8) & 511u, nX = (rp >> 17) & 31u, nT = rp >> 22;
    Vec<G> mT[4], mX[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
#pragma unroll
        for (int g = 0; g < G; ++g) mT[q].v[g] = mX[q].v[g] = 0;
        if (q < NS && (uint32_t)q < nX) {
            mX[q] = sm_load<G>(sx, xOff + q);
#pragma unroll
            for (int g = 0; g < G; ++g) mX[q].v[g] ^= own.v[g];
        }
        if (q < NS && (uint32_t)q < nT) {
            mT[q] = sm_load<G>(sx, tOff + q);
#pragma unroll
            for (int g = 0; g < G; ++g) mT[q].v[g] ^= own.v[g];
        }
    }
    if constexpr (NS == 4) {
        planes_from8<G>(P, mT, mX);
    } else {
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const uint64_t a = mX[0].v[g], b = mX[1].v[g], c = mT[0].v[g], d = mT[1].v[g];
            const uint64_t s = a ^ b ^ c, c1 = maj64(a, b, c), c2 = s & d;
            P.p[0][g] = s ^ d;
            P.p[1][g] = c1 ^ c2;
            P.p[2][g] = c1 & c2;
            P.p[3][g] = 0;
            P.p[4][g] = 0;
        }
    }
}

// lanes with u >= umin, for u < 2^NP and umin <= 2^(NP-1): the carry out of u + (2^NP - umin) over the NP planes, one
// majority per plane: carry' = maj(plane, carry, k_b) with k_b = bit b of 2^NP - umin spread over the word
// (umin = 0: every lane)
template <int G, int NP>
__device__ __forceinline__ uint64_t lanes_ge(const Planes<G> &P, int g, uint32_t umin)
{
    const uint32_t K = (1u << NP) - umin;
    uint32_t clo = 0, chi = 0;
#pragma unroll
    for (int b = 0; b < NP; ++b) {
        const uint32_t kb = (uint32_t)((int32_t)(K << (31 - b)) >> 31);
        const uint32_t plo = (uint32_t)P.p[b][g], phi = (uint32_t)(P.p[b][g] >> 32);
        clo = (plo & clo) | (kb & (plo ^ clo));
        chi = (phi & chi) | (kb & (phi ^ chi));
    }
    const uint64_t carry = (uint64_t)chi << 32 | clo;
    return umin == 0 ? ~0ull : carry;
}

struct SweepArgs {
    uint64_t *spin;
    const uint64_t *J;
    const uint32_t *col, *orig_s, *rp_s;
    const SGHdr *hdr;
    uint64_t thr[32];                 // thr[k], k = 0..31 (0 beyond dmax): read from the constant bank
    uint32_t slice0, nslices;         // of the colour class
    uint32_t W, NG, word0;            // words per site, word groups (W / G), first word of the instance (multiple of 4)
    uint32_t sweep_lo, sweep_hi;
    uint32_t rk[20];                  // Philox round keys (k0 + r*0x9E3779B9, k1 + r*0xBB67AE85), r = 0..9
    uint32_t reverse;
};

// W1: one word per site, known at compile time (no index multiplications)
template <int G, int IT, int ITX, bool WIDE, bool W1, int MINB>
__global__ void __launch_bounds__(SG_BT, MINB) k_vb_sweep(const __grid_constant__ SweepArgs a)
{
    using I = typename Idx<WIDE>::type;
    const uint32_t W = W1 ? 1u : a.W, NG = W1 ? 1u : a.NG;
    __shared__ __align__(16) uint64_t s_x[WARPS][32 * IT * G];
    uint64_t *sx = s_x[threadIdx.x >> 5];
    // `reverse`: walk the class from its last slice to its first (the host alternates the direction from launch to
    // launch, so that a launch starts where the previous one ended and finds those spin words still in L2)
    const uint32_t bid = a.reverse ? gridDim.x - 1u - blockIdx.x : blockIdx.x;
    const uint32_t job = bid * WARPS + (threadIdx.x >> 5);
    const uint32_t slice = NG == 1 ? job : job / NG;
    const uint32_t w0 = NG == 1 ? 0u : (job % NG) * G;
    const uint32_t lane = threadIdx.x & 31u;
    const uint64_t pol = policy_evict_first();
    if (slice >= a.nslices) return;                           // whole warps only
    const uint32_t gs = a.slice0 + slice;
    const uint4 t = __ldg(reinterpret_cast<const uint4 *>(a.hdr) + gs);
    const SGHdr h{t.x, t.y, t.z, t.w};
    const uint32_t site = ld_stream_u32(a.orig_s + (gs * 32u + lane), pol);   // SG_NONE: no site in this lane
    const uint32_t rp = ld_stream_u32(a.rp_s + (gs * 32u + lane), pol);
    Streams<G, IT, ITX, WIDE> st;
    st.load(a.col, a.J, h, W, w0, pol);

    // r = x_{w&3} of P(site, w>>2, sweep, tag 0): the ten Philox rounds run while the stream loads are in flight
    uint32_t x[4];
    philox4x32_10_keys(site, (a.word0 + w0) >> 2, a.sweep_lo, a.sweep_hi, a.rk, x);
    // thr[k] is non-increasing in k, so r < thr[kk] <=> kk <= kall := #{k >= 1 : r < thr[k]} (thr[k] = 0 beyond dmax)
    uint32_t kall[G];
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const uint32_t r = G == 4 ? x[g] : (G == 2 ? ((w0 & 2u) ? x[2 + g] : x[g])
                                                   : ((w0 & 2u) ? ((w0 & 1u) ? x[3] : x[2]) : ((w0 & 1u) ? x[1] : x[0])));
        uint32_t k = 0;
        while (k < 31u && (uint64_t)r < a.thr[k + 1]) ++k;
        kall[g] = k;
    }
    // Everything above reads arrays that no kernel writes.  The launch is a programmatic dependent launch: this
    // grid's CTAs start while the previous colour class is still draining and wait here, before the first spin
    // word is read, until that grid has completed and its writes are visible.
    // (ptxas hoists the wait above every global load that no thread exit separates from it; this exit is never
    // taken -- see PIN_IMPOSSIBLE -- and depends on every stream load, which pins them all in front of the wait;
    // tests/test_host_logic.py checks the order in the SASS)
    if (st.pin(site, rp) == PIN_IMPOSSIBLE) return;
    griddep_wait();
    griddep_launch_dependents();

    uint64_t *own_ptr = a.spin + (I)(h.pos0 + lane) * W + w0;
    Vec<G> own;
#pragma unroll
    for (int g = 0; g < G; ++g) own.v[g] = 0;
    if (site != SG_NONE) own = ld_plain_vec<G>(own_ptr);
    st.gather(a.spin, W, w0, sx, (h.counts >> 6) & 1023u);
    __syncwarp();

    // flip <=> kk = d - 2u <= kstar <=> u >= ceil((d - kstar)/2); the slice's shape (warp-uniform) picks the count
    Planes<G> P;
    const uint32_t d = ((rp >> 17) & 31u) + (rp >> 22), shape = h.counts >> 28;
    uint64_t any = 0;
    if (shape == 0) {
        count_unsatisfied_short<G, 2>(sx, rp, own, P);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const uint64_t flip = lanes_ge<G, 3>(P, g, (d - min(kall[g], d) + 1u) >> 1);
            own.v[g] ^= flip;
            any |= flip;
        }
    } else if (shape == 1) {
        count_unsatisfied_short<G, 4>(sx, rp, own, P);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const uint64_t flip = lanes_ge<G, 4>(P, g, (d - min(kall[g], d) + 1u) >> 1);
            own.v[g] ^= flip;
            any |= flip;
        }
    } else {
        count_unsatisfied<G>(sx, rp, own, P);
#pragma unroll
        for (int g = 0; g < G; ++g) {
            const uint64_t flip = lanes_ge<G, 5>(P, g, (d - min(kall[g], d) + 1u) >> 1);
            own.v[g] ^= flip;
            any |= flip;
        }
    }
    if (site != SG_NONE && any) st_plain_vec<G>(own_ptr, own);
}

// ------------------------------------------------------------------------------------ energy
// counts[w*64+b] += sum over all sites of u_i (unsatisfied incident bonds of lane w*64+b) = 2 U_l; E_l = 2 U_l - M.
// One launch over every slice of the instance; grid.y = word; a warp takes UNSAT_ROWS consecutive slices and keeps its
// per-lane totals in vertical counters, then shared memory, then one atomicAdd per lane and CTA.
#ifndef SG_UNSAT_MINB
#define SG_UNSAT_MINB 8
#endif
#ifndef SG_UNSAT_ROWS
#define SG_UNSAT_ROWS 16
#endif
constexpr uint32_t UNSAT_ROWS = SG_UNSAT_ROWS;
constexpr int UNSAT_IT = 8, UNSAT_ITX = 6;      // the largest budgets of SG_VB_BUDGETS_G1: serves every class

template <bool WIDE, int IT, int ITX, int MINB>
__global__ void __launch_bounds__(SG_BT, MINB)
k_vb_unsat(const uint64_t *__restrict__ spin, const uint64_t *__restrict__ J, const uint32_t *__restrict__ col,
           const uint32_t *__restrict__ rp_s, const SGHdr *__restrict__ hdr, uint32_t nslices, uint32_t W,
           unsigned long long *__restrict__ counts)
{
    using I = typename Idx<WIDE>::type;
    constexpr int LR = UNSAT_ROWS <= 2 ? 1 : UNSAT_ROWS <= 4 ? 2 : UNSAT_ROWS <= 8 ? 3 : 4;
    constexpr int PT = 5 + LR + 5;     // u <= 31, UNSAT_ROWS additions, 5 doublings in the warp
    __shared__ __align__(16) uint64_t s_x[WARPS][32 * IT];
    __shared__ unsigned long long s_counts[64];
    uint64_t *sx = s_x[threadIdx.x >> 5];
    if (threadIdx.x < 64) s_counts[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t w = blockIdx.y;
    const uint32_t warp = blockIdx.x * WARPS + (threadIdx.x >> 5), lane = threadIdx.x & 31u;
    const uint64_t pol = policy_evict_first();
    uint64_t acc[PT];
    vc_clear(acc);
#pragma unroll 1
    for (uint32_t it = 0; it < UNSAT_ROWS; ++it) {
        const uint32_t slice = warp * UNSAT_ROWS + it;
        if (slice >= nslices) break;                           // warp-uniform
        const uint4 t = __ldg(reinterpret_cast<const uint4 *>(hdr) + slice);
        const SGHdr h{t.x, t.y, t.z, t.w};
        const uint32_t rp = ld_stream_u32(rp_s + slice * 32u + lane, pol);
        Streams<1, IT, ITX, WIDE> st;
        st.load(col, J, h, W, w, pol);
        Vec<1> own;
        own.v[0] = 0;
        if (lane < (h.counts & 63u)) own = ld_plain_vec<1>(spin + (I)(h.pos0 + lane) * W + w);
        st.gather(spin, W, w, sx, (h.counts >> 6) & 1023u);
        __syncwarp();
        Planes<1> P;
        count_unsatisfied<1>(sx, rp, own, P);
        __syncwarp();
        const uint64_t pl[5] = {P.p[0][0], P.p[1][0], P.p[2][0], P.p[3][0], P.p[4][0]};
        vc_add_planes<5 + LR, PT, 5>(acc, pl);
    }
    vc_warp_flush<PT>(acc, 1, 0, s_counts);
    __syncthreads();
    if (threadIdx.x < 64 && s_counts[threadIdx.x]) atomicAdd(counts + (uint64_t)w * 64 + threadIdx.x, s_counts[threadIdx.x]);
}

// ------------------------------------------------------------------------------------ couplings
// O3 + gauge: the coupling entry x of the site at position p towards position nb, edge e = jeid[x], gets
// J[x*W + w] = kappa_e[w] ^ eps[p*W + w] ^ eps[nb*W + w], kappa_e[w] = x0 | x1<<32 of P(e, word0 + w, 0, tag 2).
// One thread per site, every X entry and every word in turn (runs once per sg_create).
__global__ void __launch_bounds__(SG_BT)
k_init_vb_couplings(uint64_t *__restrict__ J, const uint64_t *__restrict__ eps, const uint32_t *__restrict__ col,
                    const uint32_t *__restrict__ jeid, const uint32_t *__restrict__ rp_s, const SGHdr *__restrict__ hdr,
                    uint32_t nslices, uint32_t W, uint32_t word0, uint32_t k0, uint32_t k1)
{
    const uint32_t slice = blockIdx.x * WARPS + (threadIdx.x >> 5), lane = threadIdx.x & 31u;
    if (slice >= nslices) return;
    const SGHdr h = hdr[slice];
    if (lane >= (h.counts & 63u)) return;
    const uint32_t rp = rp_s[slice * 32u + lane];
    const uint32_t xOff = rp & 255u, nX = (rp >> 17) & 31u;
    const uint64_t p = (uint64_t)h.pos0 + lane;
    for (uint32_t r = 0; r < nX; ++r) {
        const uint64_t nb = col[(uint64_t)h.col_off + xOff + r];
        const uint64_t xi = (uint64_t)h.j_off + xOff + r;
        const uint32_t e = jeid[xi];
        for (uint32_t w = 0; w < W; ++w) {
            uint32_t x[4];
            philox4x32_10(e, word0 + w, 0u, 2u << 24, k0, k1, x);
            J[xi * W + w] = ((uint64_t)x[0] | ((uint64_t)x[1] << 32)) ^ eps[p * W + w] ^ eps[nb * W + w];
        }
    }
}

template <int G, int IT, int ITX, bool WIDE, bool W1, int MINB>
int launch(const VBDevice &d, const VBClass &c, uint32_t W, uint32_t word0, uint64_t sweep, SGSeed key, bool reverse, cudaStream_t st)
{
    SweepArgs a;
    a.spin = d.spin; a.J = d.J; a.col = d.col; a.orig_s = d.orig_s; a.rp_s = d.rp_s; a.hdr = d.hdr;
    for (int k = 0; k < 32; ++k) a.thr[k] = d.thr_host[k];
    a.slice0 = (uint32_t)c.slice0; a.nslices = (uint32_t)c.nslices;
    a.W = W; a.NG = W / G; a.word0 = word0;
    a.sweep_lo = (uint32_t)sweep; a.sweep_hi = (uint32_t)(sweep >> 32) /* tag 0 */;
    for (uint32_t r = 0; r < 10; ++r) { a.rk[2 * r] = key.k0 + r * 0x9E3779B9u; a.rk[2 * r + 1] = key.k1 + r * 0xBB67AE85u; }
    a.reverse = reverse ? 1u : 0u;
    const uint64_t jobs = c.nslices * a.NG;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)((jobs + WARPS - 1) / WARPS));
    cfg.blockDim = dim3(SG_BT);
    // Shared-memory carve-out: a preference of 28 % makes the driver configure 100 KiB of shared memory -- the smallest
    // size that holds the 12 CTAs (7 KiB each with the system's 1 KiB) the register file admits -- and leaves 156 KiB L1.
    // The gathers keep thousands of lines in flight per SM and L1 is where they land: the driver's own default is
    // 3.5 % slower, 44 % (132 KiB) 5 % slower, 100 % (228 KiB) 2.5 x slower; 14-24 % (64 KiB, 9 CTAs) is 5 % slower
    // too (profiles/r02_sweep.md).  SG_VB_CARVEOUT=<percent>: measurement knob.
    const char *carve_env = std::getenv("SG_VB_CARVEOUT");      // read at every launch, like the other knobs: tests switch them
    const int carve_pct = carve_env ? std::atoi(carve_env) : 28;
    static int carved = -1;                 // per instantiation: the preference that is in force
    if (carved != carve_pct) {
        cudaFuncSetAttribute(k_vb_sweep<G, IT, ITX, WIDE, W1, MINB>, cudaFuncAttributePreferredSharedMemoryCarveout, carve_pct);
        carved = carve_pct;
    }
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddep_wait() in the kernel
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    const bool no_pdl = std::getenv("SG_NO_PDL") != nullptr;   // measurement knob
    cfg.numAttrs = no_pdl ? 0 : 1;
    const cudaError_t le = cudaLaunchKernelEx(&cfg, k_vb_sweep<G, IT, ITX, WIDE, W1, MINB>, a);
    sgk_count_launch();
    const cudaError_t e = le != cudaSuccess ? le : cudaGetLastError();
    if (e != cudaSuccess) {
        sg_set_error(std::string("k_vb_sweep launch failed: ") + cudaGetErrorString(e));
        return SG_ECUDA;
    }
    return SG_OK;
}

// one word per thread: the class's budget picks the instantiation (SG_VB_BUDGETS_G1)
template <bool WIDE, bool W1>
int launch_g1(const VBDevice &d, const VBClass &c, uint32_t W, uint32_t word0, uint64_t sweep, SGSeed key, bool reverse, cudaStream_t st)
{
    if (c.it <= 6 && c.itx <= 4) return launch<1, 6, 4, WIDE, W1, SG_MINB6>(d, c, W, word0, sweep, key, reverse, st);
    if (c.it <= 8 && c.itx <= 6) return launch<1, 8, 6, WIDE, W1, SG_MINB8>(d, c, W, word0, sweep, key, reverse, st);
    sg_set_error("k_vb_sweep: the slice budget of the class exceeds the kernels'");
    return SG_EINVAL;
}

// test knob (read at every launch, so that one process can exercise both paths): 64-bit index arithmetic on any instance
bool force_wide() { return std::getenv("SG_FORCE_WIDE") != nullptr; }

}  // namespace

int sgk_vb_sweep_class(const VBDevice &d, const VBClass &c, uint64_t N, uint64_t nJ, uint32_t W, uint32_t word0, uint64_t sweep, SGSeed key,
                       bool reverse, cudaStream_t st)
{
    if (c.n == 0) return SG_OK;
    const bool wide = force_wide() || N * W >= (1ull << 32) || nJ * W >= (1ull << 32);
    const uint32_t G = sg_vb_group(W);
    if (c.nslices * (uint64_t)(W / G) >= (1ull << 31)) { sg_set_error("sgk_vb_sweep_class: class too large"); return SG_EINVAL; }
    if (G != 1 && (c.it > 4 || c.itx > (G == 2 ? 3u : 2u))) { sg_set_error("k_vb_sweep: the slice budget of the class exceeds the kernels'"); return SG_EINVAL; }
    if (!wide) {
        switch (G) {
        case 1: return W == 1 ? launch_g1<false, true>(d, c, W, word0, sweep, key, reverse, st) : launch_g1<false, false>(d, c, W, word0, sweep, key, reverse, st);
        case 2: return launch<2, 4, 3, false, false, 6>(d, c, W, word0, sweep, key, reverse, st);
        default: return launch<4, 4, 2, false, false, 4>(d, c, W, word0, sweep, key, reverse, st);
        }
    }
    switch (G) {
    case 1: return launch_g1<true, false>(d, c, W, word0, sweep, key, reverse, st);
    case 2: return launch<2, 4, 3, true, false, 6>(d, c, W, word0, sweep, key, reverse, st);
    default: return launch<4, 4, 2, true, false, 4>(d, c, W, word0, sweep, key, reverse, st);
    }
}

int sgk_vb_unsat(const VBDevice &d, uint64_t N, uint64_t nJ, uint32_t W, uint64_t *counts, cudaStream_t st)
{
    const uint64_t nslices = d.nslices;
    if (nslices == 0) return SG_OK;
    if (d.it_max > (uint32_t)UNSAT_IT || d.itx_max > (uint32_t)UNSAT_ITX) { sg_set_error("k_vb_unsat: the slice budget of the instance exceeds the kernel's"); return SG_EINVAL; }
    const bool wide = force_wide() || N * W >= (1ull << 32) || nJ * W >= (1ull << 32);
    const uint64_t warps = (nslices + UNSAT_ROWS - 1) / UNSAT_ROWS;
    dim3 grid((unsigned)((warps + WARPS - 1) / WARPS), W);
    // the instantiation for the instance's largest per-class budget
    const bool small = d.it_max <= 6 && d.itx_max <= 4;
    auto go = [&](auto kern) {
        static bool carved = false;     // per instantiation (the lambda is instantiated once per kernel)
        if (!carved) { cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 28); carved = true; }
        kern<<<grid, SG_BT, 0, st>>>(d.spin, d.J, d.col, d.rp_s, d.hdr, (uint32_t)nslices, W, (unsigned long long *)counts);
    };
    if (wide) { if (small) go(k_vb_unsat<true, 6, 4, SG_UNSAT_MINB>); else go(k_vb_unsat<true, UNSAT_IT, UNSAT_ITX, 7>); }
    else { if (small) go(k_vb_unsat<false, 6, 4, SG_UNSAT_MINB>); else go(k_vb_unsat<false, UNSAT_IT, UNSAT_ITX, 7>); }
    sgk_count_launch();
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { sg_set_error(std::string("k_vb_unsat launch failed: ") + cudaGetErrorString(e)); return SG_ECUDA; }
    return SG_OK;
}

int sgk_init_vb_couplings(const VBDevice &d, const uint32_t *jeid, uint32_t W, uint32_t word0, SGSeed key, cudaStream_t st)
{
    const uint64_t nslices = d.nslices;
    if (nslices == 0) return SG_OK;
    k_init_vb_couplings<<<(unsigned)((nslices + WARPS - 1) / WARPS), SG_BT, 0, st>>>(d.J, d.eps, d.col, jeid, d.rp_s, d.hdr, (uint32_t)nslices, W,
                                                                                     word0, key.k0, key.k1);
    sgk_count_launch();
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { sg_set_error(std::string("k_init_vb_couplings launch failed: ") + cudaGetErrorString(e)); return SG_ECUDA; }
    return SG_OK;
}
