// sg_vb_sweep.cu -- the kernels that walk the rows of a Viana-Bray instance: the Metropolis sweep of one colour class
// (row a3 of SURVEY.md 8(a); PAPER.md:260 "classic single spin flip Metropolis", :318-320 kernel prose), the energy
// (a7) and the drawing of the coupling words (a1).  Conventions: DESIGN.md section 3 (O3, O7, Q14).
//
// One warp per (slice, group of G words); layout in sg_internal.h.  Two phases:
//   1. one lane per row ENTRY of the slice: neighbour index and coupling word from the coalesced streams, gather of
//      the neighbour's spin word(s), x_e = spin ^ coupling (tree entries: no coupling after the gauge transformation)
//      parked in shared memory.  Every lane is busy whatever the degrees are; consecutive entries belong to
//      consecutive sites in breadth-first order, so the lanes of a gather share 128-byte lines and 32-byte sectors.
//   2. one lane per SITE: m_e = own ^ x_e (bit = bond unsatisfied), u = per-lane sum of the m_e in 5 bit planes
//      (carry-save adders), one Philox draw r per word shared by its 64 lanes, kstar = #{k >= 1 : r < thr[k]}, flip the
//      lanes with u >= ceil((d - kstar)/2).  No floating point.
// G = 4: a thread owns four words of its entry / site: one 32-byte sector per access (LDG.256) and one Philox call for
// the four words (Q6).
//
// Memory behaviour (B200, profiles/): couplings, neighbour indices, labels and row pointers are read once per sweep,
// coalesced, and stream through L2 (evict_first, no L1 allocation).  The gathers are what bounds the sweep: each costs
// one L1TEX wavefront per distinct 128-byte line of the warp's request, one L2 sector per distinct 32 bytes and, when
// it misses L2, a whole line from HBM.
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
#ifndef SG_MINB1
#define SG_MINB1 10    // resident CTAs per SM the one-word kernel is compiled for
#endif
constexpr int WARPS = SG_BT / 32;
// the never-taken exit in front of griddepcontrol.wait compares against this value: an AND of neighbour positions
// (all < 2^31 - 2) and SG_NONE fillers can never equal it
constexpr uint32_t PIN_IMPOSSIBLE = 0x7FFFFFFEu;

// compile-time entry budget of a slice (>= sg_vb_slice_cap of the words it serves) and iterations of 32 entries
template <int G> struct Cap { static constexpr int value = G == 4 ? 64 : 128; static constexpr int iters = value / 32; };

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
// The stream part: neighbour positions of the slice's T and X entries 32k + lane (SG_NONE beyond the run) and the
// coupling words of the X entries.  Reads arrays that no kernel writes.
template <int G, bool WIDE>
struct Streams {
    static constexpr int IT = Cap<G>::iters;
    uint32_t nbT[IT], nbX[IT];
    Vec<G> jw[IT];

    __device__ __forceinline__ void load(const uint32_t *__restrict__ col, const uint64_t *__restrict__ J, SGHdr h, uint32_t W, uint32_t w0, uint64_t pol)
    {
        using I = typename Idx<WIDE>::type;
        const uint32_t lane = threadIdx.x & 31u;
        const uint32_t nTs = (h.counts >> 6) & 1023u, nXs = h.counts >> 16;
        const uint32_t *ct = col + h.col_off + lane, *cx = ct + nTs;
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            nbT[k] = SG_NONE;
            if (32u * k < nTs)                                 // warp-uniform: most slices need two iterations
                if (32u * k + lane < nTs) nbT[k] = ld_stream_u32(ct + 32 * k, pol);
        }
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            nbX[k] = SG_NONE;
#pragma unroll
            for (int g = 0; g < G; ++g) jw[k].v[g] = 0;
            if (32u * k < nXs && 32u * k + lane < nXs) {
                nbX[k] = ld_stream_u32(cx + 32 * k, pol);
                jw[k] = ld_stream_vec<G>(J + (I)(h.j_off + 32u * k + lane) * W + w0, pol);
            }
        }
    }
    // A value that can never equal PIN_IMPOSSIBLE and is known only when the last stream loads have returned: the
    // last index and coupling loads of both runs (loads return in order per thread) and the two per-site loads.
    __device__ __forceinline__ uint32_t pin(uint32_t site, uint32_t rp) const
    {
        uint32_t a = nbT[IT - 1] & nbX[IT - 1] & nbT[0] & nbX[0];     // a position (< 2^31 - 2) or SG_NONE
        a &= (uint32_t)(jw[IT - 1].v[G - 1] >> 32) | (uint32_t)(jw[0].v[0] >> 32) | site | rp | 0x7FFFFFFFu;
        return a;
    }
    // the gather part: x_e = spin[neighbour] (^ coupling) into shared memory; all gathers in flight before the first store
    __device__ __forceinline__ void gather(const uint64_t *spin, uint32_t W, uint32_t w0, uint64_t *sT, uint64_t *sX) const
    {
        using I = typename Idx<WIDE>::type;
        const uint32_t lane = threadIdx.x & 31u;
        Vec<G> xT[IT], xX[IT];
#pragma unroll
        for (int k = 0; k < IT; ++k)
            if (nbT[k] != SG_NONE) xT[k] = ld_plain_vec<G>(spin + (I)nbT[k] * W + w0);
#pragma unroll
        for (int k = 0; k < IT; ++k)
            if (nbX[k] != SG_NONE) xX[k] = ld_plain_vec<G>(spin + (I)nbX[k] * W + w0);
#pragma unroll
        for (int k = 0; k < IT; ++k)
            if (nbT[k] != SG_NONE) sm_store<G>(sT, 32u * k + lane, xT[k]);
#pragma unroll
        for (int k = 0; k < IT; ++k)
            if (nbX[k] != SG_NONE) {
#pragma unroll
                for (int g = 0; g < G; ++g) xX[k].v[g] ^= jw[k].v[g];
                sm_store<G>(sX, 32u * k + lane, xX[k]);
            }
    }
};

// ---- phase 2 ------------------------------------------------------------------------------------
// u of the site whose row pointer is rp: its T entries sT[tOff ..], its X entries sX[xOff ..]
template <int G>
__device__ __forceinline__ void count_unsatisfied(const uint64_t *sT, const uint64_t *sX, uint32_t rp, const Vec<G> &own, Planes<G> &P)
{
    const uint32_t tOff = rp & 1023u, xOff = (rp >> 10) & 1023u, nT = (rp >> 20) & 31u, nX = rp >> 25;
    Vec<G> mT[4], mX[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
#pragma unroll
        for (int g = 0; g < G; ++g) mT[q].v[g] = mX[q].v[g] = 0;
        if ((uint32_t)q < nT) {
            mT[q] = sm_load<G>(sT, tOff + q);
#pragma unroll
            for (int g = 0; g < G; ++g) mT[q].v[g] ^= own.v[g];
        }
        if ((uint32_t)q < nX) {
            mX[q] = sm_load<G>(sX, xOff + q);
#pragma unroll
            for (int g = 0; g < G; ++g) mX[q].v[g] ^= own.v[g];
        }
    }
    planes_from8<G>(P, mT, mX);
    for (uint32_t q = 4; q < nT; ++q) {           // long rows: per-lane loops, shared memory only
        Vec<G> m = sm_load<G>(sT, tOff + q);
#pragma unroll
        for (int g = 0; g < G; ++g) m.v[g] ^= own.v[g];
        planes_add1<G>(P, m);
    }
    for (uint32_t q = 4; q < nX; ++q) {
        Vec<G> m = sm_load<G>(sX, xOff + q);
#pragma unroll
        for (int g = 0; g < G; ++g) m.v[g] ^= own.v[g];
        planes_add1<G>(P, m);
    }
}

// lanes with u >= umin, umin <= 16: the carry out of u + (32 - umin) over the 5 planes, one majority per plane:
// carry' = maj(plane, carry, k_b) with k_b = bit b of 32 - umin spread over the word (umin = 0: every lane)
template <int G>
__device__ __forceinline__ uint64_t lanes_ge(const Planes<G> &P, int g, uint32_t umin)
{
    const uint32_t K = 32u - umin;
    uint64_t carry = 0;
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        const uint64_t kb = 0ull - (uint64_t)((K >> b) & 1u);
        carry = maj64(P.p[b][g], carry, kb);
    }
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
template <int G, bool WIDE, bool W1, int MINB>
__global__ void __launch_bounds__(SG_BT, MINB) k_vb_sweep(const __grid_constant__ SweepArgs a)
{
    using I = typename Idx<WIDE>::type;
    const uint32_t W = W1 ? 1u : a.W, NG = W1 ? 1u : a.NG;
    constexpr int CAPK = Cap<G>::value;
    __shared__ __align__(16) uint64_t s_x[WARPS][2 * CAPK * G];
    uint64_t *sT = s_x[threadIdx.x >> 5], *sX = sT + CAPK * G;
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
    Streams<G, WIDE> st;
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
    st.gather(a.spin, W, w0, sT, sX);
    __syncwarp();

    Planes<G> P;
    count_unsatisfied<G>(sT, sX, rp, own, P);
    // flip <=> kk = d - 2u <= kstar <=> u >= ceil((d - kstar)/2)
    const uint32_t d = ((rp >> 20) & 31u) + (rp >> 25);
    uint64_t any = 0;
#pragma unroll
    for (int g = 0; g < G; ++g) {
        const uint32_t kstar = min(kall[g], d);
        const uint64_t flip = lanes_ge<G>(P, g, (d - kstar + 1u) >> 1);
        own.v[g] ^= flip;
        any |= flip;
    }
    if (site != SG_NONE && any) st_plain_vec<G>(own_ptr, own);
}

// ------------------------------------------------------------------------------------ energy
// counts[w*64+b] += sum over all sites of u_i (unsatisfied incident bonds of lane w*64+b) = 2 U_l; E_l = 2 U_l - M.
// One launch over every slice of the instance; grid.y = word; a warp takes UNSAT_ROWS consecutive slices and keeps its
// per-lane totals in vertical counters, then shared memory, then one atomicAdd per lane and CTA.
constexpr uint32_t UNSAT_ROWS = 4;

template <bool WIDE>
__global__ void __launch_bounds__(SG_BT, 8)
k_vb_unsat(const uint64_t *__restrict__ spin, const uint64_t *__restrict__ J, const uint32_t *__restrict__ col,
           const uint32_t *__restrict__ rp_s, const SGHdr *__restrict__ hdr, uint32_t nslices, uint32_t W,
           unsigned long long *__restrict__ counts)
{
    using I = typename Idx<WIDE>::type;
    constexpr int CAPK = Cap<1>::value;
    constexpr int PT = 5 + 2 + 5;      // u <= 31, UNSAT_ROWS additions, 5 doublings in the warp
    __shared__ __align__(16) uint64_t s_x[WARPS][2 * CAPK];
    __shared__ unsigned long long s_counts[64];
    uint64_t *sT = s_x[threadIdx.x >> 5], *sX = sT + CAPK;
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
        Streams<1, WIDE> st;
        st.load(col, J, h, W, w, pol);
        Vec<1> own;
        own.v[0] = 0;
        if (lane < (h.counts & 63u)) own = ld_plain_vec<1>(spin + (I)(h.pos0 + lane) * W + w);
        st.gather(spin, W, w, sT, sX);
        __syncwarp();
        Planes<1> P;
        count_unsatisfied<1>(sT, sX, rp, own, P);
        __syncwarp();
        const uint64_t pl[5] = {P.p[0][0], P.p[1][0], P.p[2][0], P.p[3][0], P.p[4][0]};
        vc_add_planes<5 + 2, PT, 5>(acc, pl);
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
    const uint32_t xOff = (rp >> 10) & 1023u, nX = rp >> 25, nTs = (h.counts >> 6) & 1023u;
    const uint64_t p = (uint64_t)h.pos0 + lane;
    for (uint32_t r = 0; r < nX; ++r) {
        const uint64_t nb = col[(uint64_t)h.col_off + nTs + xOff + r];
        const uint64_t xi = (uint64_t)h.j_off + xOff + r;
        const uint32_t e = jeid[xi];
        for (uint32_t w = 0; w < W; ++w) {
            uint32_t x[4];
            philox4x32_10(e, word0 + w, 0u, 2u << 24, k0, k1, x);
            J[xi * W + w] = ((uint64_t)x[0] | ((uint64_t)x[1] << 32)) ^ eps[p * W + w] ^ eps[nb * W + w];
        }
    }
}

template <int G, bool WIDE, bool W1, int MINB>
int launch(const VBDevice &d, const VBClass &c, uint32_t W, uint32_t word0, uint64_t sweep, SGSeed key, bool reverse, cudaStream_t st)
{
    if (d.cap > (uint32_t)Cap<G>::value) { sg_set_error("k_vb_sweep: the slice budget of the instance exceeds the kernel's"); return SG_EINVAL; }
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
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddep_wait() in the kernel
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    static const bool no_pdl = std::getenv("SG_NO_PDL") != nullptr;   // measurement knob
    cfg.numAttrs = no_pdl ? 0 : 1;
    const cudaError_t le = cudaLaunchKernelEx(&cfg, k_vb_sweep<G, WIDE, W1, MINB>, a);
    sgk_count_launch();
    const cudaError_t e = le != cudaSuccess ? le : cudaGetLastError();
    if (e != cudaSuccess) {
        sg_set_error(std::string("k_vb_sweep launch failed: ") + cudaGetErrorString(e));
        return SG_ECUDA;
    }
    return SG_OK;
}

// test knob (read at every launch, so that one process can exercise both paths): 64-bit index arithmetic on any instance
bool force_wide() { return std::getenv("SG_FORCE_WIDE") != nullptr; }

}  // namespace

int sgk_vb_sweep_class(const VBDevice &d, const VBClass &c, uint64_t N, uint64_t nJ, uint32_t W, uint32_t word0, uint64_t sweep, SGSeed key,
                       bool reverse, cudaStream_t st)
{
    if (c.n == 0) return SG_OK;
    const bool wide = force_wide() || N * W >= (1ull << 32) || nJ * W >= (1ull << 32);
    const uint32_t G = (W % 4 == 0) ? 4 : (W % 2 == 0) ? 2 : 1;
    if (c.nslices * (uint64_t)(W / G) >= (1ull << 31)) { sg_set_error("sgk_vb_sweep_class: class too large"); return SG_EINVAL; }
    if (!wide) {
        switch (G) {
        case 1: return W == 1 ? launch<1, false, true, SG_MINB1>(d, c, W, word0, sweep, key, reverse, st)
                              : launch<1, false, false, SG_MINB1>(d, c, W, word0, sweep, key, reverse, st);
        case 2: return launch<2, false, false, 6>(d, c, W, word0, sweep, key, reverse, st);
        default: return launch<4, false, false, 4>(d, c, W, word0, sweep, key, reverse, st);
        }
    }
    switch (G) {
    case 1: return launch<1, true, false, SG_MINB1>(d, c, W, word0, sweep, key, reverse, st);
    case 2: return launch<2, true, false, 6>(d, c, W, word0, sweep, key, reverse, st);
    default: return launch<4, true, false, 4>(d, c, W, word0, sweep, key, reverse, st);
    }
}

int sgk_vb_unsat(const VBDevice &d, uint64_t N, uint64_t nJ, uint32_t W, uint64_t *counts, cudaStream_t st)
{
    const uint64_t nslices = d.nslices;
    if (nslices == 0) return SG_OK;
    if (d.cap > (uint32_t)Cap<1>::value) { sg_set_error("k_vb_unsat: the slice budget of the instance exceeds the kernel's"); return SG_EINVAL; }
    const bool wide = force_wide() || N * W >= (1ull << 32) || nJ * W >= (1ull << 32);
    const uint64_t warps = (nslices + UNSAT_ROWS - 1) / UNSAT_ROWS;
    dim3 grid((unsigned)((warps + WARPS - 1) / WARPS), W);
    if (wide)
        k_vb_unsat<true><<<grid, SG_BT, 0, st>>>(d.spin, d.J, d.col, d.rp_s, d.hdr, (uint32_t)nslices, W, (unsigned long long *)counts);
    else
        k_vb_unsat<false><<<grid, SG_BT, 0, st>>>(d.spin, d.J, d.col, d.rp_s, d.hdr, (uint32_t)nslices, W, (unsigned long long *)counts);
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
