// sg_device.cuh -- device helpers: Philox4x32-10 (O1) and cache-hinted loads/stores.
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

// L2 eviction policies.  Couplings, indices and per-site labels are touched once per sweep and stream through
// (evict_first, no L1 allocation), so that they displace as little as possible of the spin words that the gathers
// re-read; the spin words themselves use the default policy (evict_last / L1::no_allocate on them measured no gain,
// profiles/r01_sweep.md).
__device__ __forceinline__ uint64_t policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_normal()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t ld_stream_u64(const uint64_t *ptr, uint64_t pol)
{
    uint64_t v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.b64 %0, [%1], %2;" : "=l"(v) : "l"(ptr), "l"(pol));
    return v;
}
__device__ __forceinline__ uint32_t ld_stream_u32(const uint32_t *ptr, uint64_t pol)
{
    uint32_t v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.b32 %0, [%1], %2;" : "=r"(v) : "l"(ptr), "l"(pol));
    return v;
}
// spin words: written by other classes' launches, so no .nc; keep in L2
__device__ __forceinline__ uint64_t ld_keep_u64(const uint64_t *ptr, uint64_t pol)
{
    uint64_t v;
    asm volatile("ld.global.L1::no_allocate.L2::cache_hint.b64 %0, [%1], %2;" : "=l"(v) : "l"(ptr), "l"(pol));
    return v;
}
__device__ __forceinline__ uint64_t ld_plain_u64(const uint64_t *ptr)
{
    uint64_t v;
    asm volatile("ld.global.b64 %0, [%1];" : "=l"(v) : "l"(ptr));
    return v;
}

// Programmatic dependent launch (sm_90+): wait until the grid this one depends on has completed and its memory
// operations are visible; allow the grid that depends on this one to start launching.
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void griddep_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
