// sg_device.cuh -- device helpers: Philox4x32-10 (O1), cache-hinted and vector loads/stores,
// programmatic-dependent-launch controls, bit-sliced per-lane counters.
#pragma once
#include <cstdint>

// Philox4x32-10: 10 rounds of
//   (c0,c1,c2,c3) <- (hi(B*c2)^c1^k0, lo(B*c2), hi(A*c0)^c3^k1, lo(A*c0)),  A=0xD2511F53, B=0xCD9E8D57
// with (k0,k1) += (0x9E3779B9, 0xBB67AE85) between rounds.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t ha = __umulhi(0xD2511F53u, c0), la = 0xD2511F53u * c0;
        const uint32_t hb = __umulhi(0xCD9E8D57u, c2), lb = 0xCD9E8D57u * c2;
        c0 = hb ^ c1 ^ k0;
        c2 = ha ^ c3 ^ k1;
        c1 = lb;
        c3 = la;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// the same with the ten round keys precomputed (rk[2r] = k0 + r*0x9E3779B9, rk[2r+1] = k1 + r*0xBB67AE85): the key
// schedule then costs no instruction (the keys are operands from the constant bank)
__device__ __forceinline__ void philox4x32_10_keys(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const uint32_t (&rk)[20],
                                                   uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t ha = __umulhi(0xD2511F53u, c0), la = 0xD2511F53u * c0;
        const uint32_t hb = __umulhi(0xCD9E8D57u, c2), lb = 0xCD9E8D57u * c2;
        c0 = hb ^ c1 ^ rk[2 * r];
        c2 = ha ^ c3 ^ rk[2 * r + 1];
        c1 = lb;
        c3 = la;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// G consecutive 64-bit words (G = 1, 2, 4): one site's words of one word group
template <int G> struct Vec { uint64_t v[G]; };

// L2 eviction policy for data that is touched once per sweep (couplings, indices, labels): evict_first, so that
// it displaces as little as possible of the spin words that the gathers re-read (profiles/r01_probes.md).
__device__ __forceinline__ uint64_t policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint32_t ld_stream_u32(const uint32_t *ptr, uint64_t pol)
{
    uint32_t v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.b32 %0, [%1], %2;" : "=r"(v) : "l"(ptr), "l"(pol));
    return v;
}
__device__ __forceinline__ uint32_t ld_stream_u16(const uint16_t *ptr, uint64_t pol)
{
    uint16_t v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.b16 %0, [%1], %2;" : "=h"(v) : "l"(ptr), "l"(pol));
    return v;
}
__device__ __forceinline__ uint64_t ld_stream_u64(const uint64_t *ptr, uint64_t pol)
{
    uint64_t v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.b64 %0, [%1], %2;" : "=l"(v) : "l"(ptr), "l"(pol));
    return v;
}
__device__ __forceinline__ uint64_t ld_plain_u64(const uint64_t *ptr)
{
    uint64_t v;
    asm volatile("ld.global.b64 %0, [%1];" : "=l"(v) : "l"(ptr));
    return v;
}
// a spin word that is read once in this launch (gather along a non-tree edge): cached in L2 only
__device__ __forceinline__ uint64_t ld_x_u64(const uint64_t *ptr)
{
    uint64_t v;
    asm volatile("ld.global.cg.b64 %0, [%1];" : "=l"(v) : "l"(ptr));
    return v;
}
// vector forms: 8, 16 or 32 bytes per access (LDG.64 / LDG.128 / LDG.256 on sm_100a); ptr aligned to 8*G bytes
template <int G> __device__ __forceinline__ Vec<G> ld_stream_vec(const uint64_t *ptr, uint64_t pol);
template <> __device__ __forceinline__ Vec<1> ld_stream_vec<1>(const uint64_t *ptr, uint64_t pol)
{
    Vec<1> r;
    r.v[0] = ld_stream_u64(ptr, pol);
    return r;
}
template <> __device__ __forceinline__ Vec<2> ld_stream_vec<2>(const uint64_t *ptr, uint64_t pol)
{
    Vec<2> r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v2.u64 {%0,%1}, [%2], %3;"
                 : "=l"(r.v[0]), "=l"(r.v[1]) : "l"(ptr), "l"(pol));
    return r;
}
template <> __device__ __forceinline__ Vec<4> ld_stream_vec<4>(const uint64_t *ptr, uint64_t pol)
{
    Vec<4> r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.u64 {%0,%1,%2,%3}, [%4], %5;"
                 : "=l"(r.v[0]), "=l"(r.v[1]), "=l"(r.v[2]), "=l"(r.v[3]) : "l"(ptr), "l"(pol));
    return r;
}
// spin words: written by other launches, so no .nc and the default policy
template <int G> __device__ __forceinline__ Vec<G> ld_plain_vec(const uint64_t *ptr);
template <> __device__ __forceinline__ Vec<1> ld_plain_vec<1>(const uint64_t *ptr)
{
    Vec<1> r;
    r.v[0] = ld_plain_u64(ptr);
    return r;
}
template <> __device__ __forceinline__ Vec<2> ld_plain_vec<2>(const uint64_t *ptr)
{
    Vec<2> r;
    asm volatile("ld.global.v2.u64 {%0,%1}, [%2];" : "=l"(r.v[0]), "=l"(r.v[1]) : "l"(ptr));
    return r;
}
template <> __device__ __forceinline__ Vec<4> ld_plain_vec<4>(const uint64_t *ptr)
{
    Vec<4> r;
    asm volatile("ld.global.v4.u64 {%0,%1,%2,%3}, [%4];" : "=l"(r.v[0]), "=l"(r.v[1]), "=l"(r.v[2]), "=l"(r.v[3]) : "l"(ptr));
    return r;
}
template <int G> __device__ __forceinline__ void st_plain_vec(uint64_t *ptr, const Vec<G> &x);
template <> __device__ __forceinline__ void st_plain_vec<1>(uint64_t *ptr, const Vec<1> &x)
{
    asm volatile("st.global.b64 [%0], %1;" ::"l"(ptr), "l"(x.v[0]) : "memory");
}
template <> __device__ __forceinline__ void st_plain_vec<2>(uint64_t *ptr, const Vec<2> &x)
{
    asm volatile("st.global.v2.u64 [%0], {%1,%2};" ::"l"(ptr), "l"(x.v[0]), "l"(x.v[1]) : "memory");
}
template <> __device__ __forceinline__ void st_plain_vec<4>(uint64_t *ptr, const Vec<4> &x)
{
    asm volatile("st.global.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(ptr), "l"(x.v[0]), "l"(x.v[1]), "l"(x.v[2]), "l"(x.v[3]) : "memory");
}

// Programmatic dependent launch (sm_90+): wait until the grid this one depends on has completed and its memory
// operations are visible; allow the grid that depends on this one to start launching.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ uint64_t maj64(uint64_t a, uint64_t b, uint64_t c) { return (a & b) | (c & (a ^ b)); }

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

// acc += the number whose bits are the NP planes in[0..NP)
template <int P, int PT, int NP>
__device__ __forceinline__ void vc_add_planes(uint64_t (&acc)[PT], const uint64_t (&in)[NP])
{
    uint64_t carry = 0;
#pragma unroll
    for (int p = 0; p < P; ++p) {
        const uint64_t b = p < NP ? in[p] : 0ull;
        const uint64_t a = acc[p];
        acc[p] = a ^ b ^ carry;
        carry = maj64(a, b, carry);
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
            carry = maj64(a, b, carry);
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
