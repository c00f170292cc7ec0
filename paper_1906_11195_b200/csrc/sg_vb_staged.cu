// sg_vb_staged.cu -- the hot kernel for n_words = 1: one colour class of one Viana-Bray Metropolis
// sweep (row a3 of SURVEY.md 8(a)), as a persistent, warp-specialised kernel.
//
// The paper's kernel (P100) reads its coupling vector coalesced and gathers the neighbour spins
// uncoalesced, hiding the latency by occupancy alone.  Here the coalesced part never
// touches a register before it is needed: a producer warp streams each tile's neighbour indices,
// coupling words, own spin words and site labels from HBM into a shared-memory ring with
// cp.async.bulk (the TMA copy engine, completion on an mbarrier, L2 evict_first), several tiles
// ahead of the 8 consumer warps.  A consumer thread (one site) reads its row from shared memory,
// issues its <= 8 random 8-byte gathers of neighbour spin words at once (the only exposed DRAM
// round trip), counts unsatisfied bonds per lane with carry-save adders, draws its Philox uniform
// and writes the updated word.  Conventions: DESIGN.md section 3 (O7, Q14).
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdlib>

#include "sg_device.cuh"
#include "sg_internal.h"

void sgk_count_launch();

namespace {

constexpr uint32_t CONSUMER_WARPS = SG_TILE_SLICES;            // one warp per slice of the tile
constexpr uint32_t ST_THREADS = 32u * (CONSUMER_WARPS + 1u);   // + producer warp
constexpr uint32_t NSTAGE = 3;
constexpr uint32_t TILE_ENT = 32u * SG_TILE_ENT32;             // 1280 entries
constexpr uint32_t TILE_POS = 32u * SG_TILE_SLICES;            // 256 positions
// stage layout (bytes)
constexpr uint32_t OFF_J = 0;                                  // TILE_ENT * 8
constexpr uint32_t OFF_G = OFF_J + TILE_ENT * 8u;              // TILE_ENT * 8: gathered neighbour spin words
constexpr uint32_t OFF_OWN = OFF_G + TILE_ENT * 8u;            // TILE_POS * 8
constexpr uint32_t OFF_COL = OFF_OWN + TILE_POS * 8u;          // TILE_ENT * 4
constexpr uint32_t OFF_ORIG = OFF_COL + TILE_ENT * 4u;         // TILE_POS * 4
constexpr uint32_t OFF_DESC = OFF_ORIG + TILE_POS * 4u;        // 16
constexpr uint32_t STAGE_BYTES = OFF_DESC + 16u;
constexpr uint32_t OFF_BARS = NSTAGE * STAGE_BYTES;              // 2 * NSTAGE mbarriers
constexpr uint32_t OFF_THR = OFF_BARS + 2u * NSTAGE * 8u + 8u;   // 32 thresholds (8-byte aligned)
constexpr uint32_t SMEM_BYTES = OFF_THR + 32u * 8u;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" ::"r"(bar), "r"(parity) : "memory");
}
// global -> shared bulk copy (TMA engine); bytes and both addresses are multiples of 16
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy) : "memory");
}

// 8-byte asynchronous gather global -> shared (LDGSTS): no register is held while it is in flight
__device__ __forceinline__ void cp_async_8(uint32_t dst, const void *src, uint64_t policy)
{
    asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "l"(policy) : "memory");
}

__device__ __forceinline__ uint64_t maj64(uint64_t a, uint64_t b, uint64_t c) { return (a & b) | (c & (a ^ b)); }

__global__ void __launch_bounds__(ST_THREADS, 3)
k_vb_sweep_staged(uint64_t *__restrict__ spin, const uint64_t *__restrict__ J, const uint32_t *__restrict__ col,
                  const uint32_t *__restrict__ orig, const VBTile *__restrict__ tiles, uint32_t ntiles,
                  const uint64_t *__restrict__ thr, uint32_t dhot, uint32_t sweep_lo, uint32_t sweep_hi, uint32_t k0, uint32_t k1)
{
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t bar_full = smem_base + NSTAGE * STAGE_BYTES;     // NSTAGE x 8 bytes
    const uint32_t bar_empty = bar_full + NSTAGE * 8u;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    uint64_t *s_thr = reinterpret_cast<uint64_t *>(smem + OFF_THR);
    if (threadIdx.x < 32) s_thr[threadIdx.x] = thr[threadIdx.x];

    if (threadIdx.x == 0) {
        for (uint32_t s = 0; s < NSTAGE; ++s) {
            mbar_init(bar_full + 8u * s, 1u);
            mbar_init(bar_empty + 8u * s, CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (warp == CONSUMER_WARPS) {
        // ------------------------------------------------------------------ producer warp
        // The 32 lanes fetch 32 tile descriptors at a time (one coalesced 512-byte read), so that the
        // serial issue loop of lane 0 never waits on a dependent global load.
        const uint64_t pol_stream = policy_evict_first();
        const uint64_t pol_spin = policy_evict_normal();
        uint32_t it = 0;
        for (uint32_t tile0 = blockIdx.x; tile0 < ntiles; tile0 += 32u * gridDim.x) {
            const uint64_t mytile = (uint64_t)tile0 + (uint64_t)lane * gridDim.x;
            VBTile mine{0, 0, 0};
            if (mytile < ntiles) mine = tiles[mytile];
            for (uint32_t q = 0; q < 32u && (uint64_t)tile0 + (uint64_t)q * gridDim.x < ntiles; ++q, ++it) {
                VBTile td;
                td.ent32 = __shfl_sync(0xFFFFFFFFu, mine.ent32, q);
                td.pos0 = __shfl_sync(0xFFFFFFFFu, mine.pos0, q);
                td.packed = __shfl_sync(0xFFFFFFFFu, mine.packed, q);
                if (lane == 0) {
                    const uint32_t s = it % NSTAGE, round = it / NSTAGE;
                    mbar_wait(bar_empty + 8u * s, (round & 1u) ^ 1u);        // passes at once in round 0
                    const uint32_t ns = (uint32_t)(td.packed & 15u);
                    uint32_t cols = 0;
                    for (uint32_t z = 0; z < ns; ++z) cols += (uint32_t)(td.packed >> (4u + 5u * z)) & 31u;
                    const uint32_t stage = smem_base + s * STAGE_BYTES;
                    // descriptor for the consumers (ordered before the barrier's release)
                    *reinterpret_cast<uint4 *>(smem + s * STAGE_BYTES + OFF_DESC) =
                        make_uint4(td.ent32, td.pos0, (uint32_t)td.packed, (uint32_t)(td.packed >> 32));
                    const uint32_t bar = bar_full + 8u * s;
                    mbar_arrive_expect_tx(bar, cols * 32u * 12u + ns * 32u * 12u);
                    if (cols) {
                        bulk_g2s(stage + OFF_J, J + (size_t)td.ent32 * 32u, cols * 256u, bar, pol_stream);
                        bulk_g2s(stage + OFF_COL, col + (size_t)td.ent32 * 32u, cols * 128u, bar, pol_stream);
                    }
                    bulk_g2s(stage + OFF_OWN, spin + td.pos0, ns * 256u, bar, pol_spin);
                    bulk_g2s(stage + OFF_ORIG, orig + td.pos0, ns * 128u, bar, pol_stream);
                }
                __syncwarp();
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- consumers
    // Software pipeline per warp: while tile i is being computed, the gathers of tile i+1 are in flight
    // as cp.async copies into the stage's G buffer (no registers held), and the producer is loading i+2.
    const uint64_t pol_hot = policy_evict_last();
    const uint64_t pol_cold = policy_evict_normal();
    const uint32_t ntiles_mine = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1u) / gridDim.x : 0u;

    // tile `it` has landed in its stage: issue this thread's gathers (spin word of every neighbour) -> G
    auto issue_gathers = [&](uint32_t it) {
        const uint32_t s = it % NSTAGE, round = it / NSTAGE;
        const unsigned char *st = smem + s * STAGE_BYTES;
        mbar_wait(bar_full + 8u * s, round & 1u);
        const uint4 dd = *reinterpret_cast<const uint4 *>(st + OFF_DESC);
        const uint64_t packed = (uint64_t)dd.z | ((uint64_t)dd.w << 32);
        if (warp < (dd.z & 15u)) {
            const uint32_t D = (uint32_t)(packed >> (4u + 5u * warp)) & 31u;
            uint32_t off = 0;
            for (uint32_t q = 0; q < warp; ++q) off += (uint32_t)(packed >> (4u + 5u * q)) & 31u;
            const uint32_t *s_col = reinterpret_cast<const uint32_t *>(st + OFF_COL) + off * 32u + lane;
            const uint32_t g_dst = smem_base + s * STAGE_BYTES + OFF_G + (off * 32u + lane) * 8u;
            for (uint32_t k = 0; k < D; ++k) {
                const uint32_t nb = s_col[k * 32u];
                cp_async_8(g_dst + k * 256u, spin + (nb & 0x7FFFFFFFu), (nb >> 31) ? pol_hot : pol_cold);
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    if (ntiles_mine) issue_gathers(0);
    for (uint32_t it = 0; it < ntiles_mine; ++it) {
        if (it + 1 < ntiles_mine) {
            issue_gathers(it + 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        const uint32_t s = it % NSTAGE;
        const unsigned char *st = smem + s * STAGE_BYTES;
        const uint4 dd = *reinterpret_cast<const uint4 *>(st + OFF_DESC);
        const uint64_t packed = (uint64_t)dd.z | ((uint64_t)dd.w << 32);
        const bool active = warp < (dd.z & 15u);
        uint32_t D = 0, off = 0;                      // my slice's row length and first column in the tile
        uint64_t own = 0;
        uint32_t site = SG_NONE;
        if (active) {
            D = (uint32_t)(packed >> (4u + 5u * warp)) & 31u;
            for (uint32_t q = 0; q < warp; ++q) off += (uint32_t)(packed >> (4u + 5u * q)) & 31u;
            own = reinterpret_cast<const uint64_t *>(st + OFF_OWN)[warp * 32u + lane];
            site = reinterpret_cast<const uint32_t *>(st + OFF_ORIG)[warp * 32u + lane];
        }
        const uint64_t *s_J = reinterpret_cast<const uint64_t *>(st + OFF_J) + off * 32u + lane;
        const uint64_t *s_G = reinterpret_cast<const uint64_t *>(st + OFF_G) + off * 32u + lane;
        uint64_t p0 = 0, p1 = 0, p2 = 0, p3 = 0, p4 = 0;
        for (uint32_t k = 0; k < D; k += 4) {
            uint64_t x[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) x[q] = (k + q < D) ? (own ^ s_J[(k + q) * 32u] ^ s_G[(k + q) * 32u]) : 0ull;
            // 4 one-bit numbers -> 3 planes
            const uint64_t sx = x[0] ^ x[1] ^ x[2], cy = maj64(x[0], x[1], x[2]);
            const uint64_t t0 = sx ^ x[3], c2 = sx & x[3];
            const uint64_t t1 = cy ^ c2, t2 = cy & c2;
            if (k == 0) {
                p0 = t0; p1 = t1; p2 = t2;
            } else {
                const uint64_t d0 = p0 & t0;             p0 ^= t0;
                const uint64_t d1 = maj64(p1, t1, d0);   p1 ^= t1 ^ d0;
                const uint64_t d2 = maj64(p2, t2, d1);   p2 ^= t2 ^ d1;
                const uint64_t d3 = p3 & d2;             p3 ^= d2;
                p4 ^= d3;
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8u * s);       // stage fully read by this warp
        if (site == SG_NONE) continue;                        // padding position or idle warp

        uint32_t xr[4];
        philox4x32_10(site, 0u, sweep_lo, sweep_hi, k0, k1, xr);
        const uint32_t r = xr[0];
        uint32_t kstar = 0;
        while (kstar < D && (uint64_t)r < s_thr[kstar + 1]) ++kstar;
        const uint32_t umin = (D - kstar + 1u) >> 1;
        uint64_t gt = 0, eq = ~0ull;
        const uint64_t pl[5] = {p0, p1, p2, p3, p4};
#pragma unroll
        for (int b = 4; b >= 0; --b) {
            const uint64_t cbit = ((umin >> b) & 1u) ? ~0ull : 0ull;
            gt |= eq & pl[b] & ~cbit;
            eq &= ~(pl[b] ^ cbit);
        }
        st_keep_u64(spin + dd.y + warp * 32u + lane, own ^ (gt | eq), D >= dhot ? pol_hot : pol_cold);
    }
}

}  // namespace

bool sgk_vb_sweep_staged_ok(uint64_t P, uint64_t entries, uint32_t W)
{
    return W == 1 && P < (1ull << 31) && entries < (1ull << 32);
}

int sgk_vb_sweep_class_staged(const VBDevice &d, const VBClass &c, uint64_t sweep, SGSeed key, cudaStream_t st)
{
    if (c.ntiles == 0) return SG_OK;
    static bool attr_done = false;
    static int ctas_per_sm = 3, sms = 148;
    if (!attr_done) {
        if (cudaFuncSetAttribute(k_vb_sweep_staged, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess) {
            sg_set_error("k_vb_sweep_staged: cannot reserve shared memory");
            return SG_ECUDA;
        }
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas_per_sm, k_vb_sweep_staged, (int)ST_THREADS, SMEM_BYTES);
        if (ctas_per_sm < 1) ctas_per_sm = 1;
        attr_done = true;
    }
    const unsigned grid = (unsigned)std::min<uint64_t>(c.ntiles, (uint64_t)sms * ctas_per_sm);
    k_vb_sweep_staged<<<grid, ST_THREADS, SMEM_BYTES, st>>>(d.spin, d.J, d.col, d.orig, d.tiles + c.tile0, (uint32_t)c.ntiles, d.thr, d.dhot,
                                                            (uint32_t)sweep, (uint32_t)(sweep >> 32) /* tag 0 */, key.k0, key.k1);
    sgk_count_launch();
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        sg_set_error(std::string("k_vb_sweep_staged launch failed: ") + cudaGetErrorString(e));
        return SG_ECUDA;
    }
    return SG_OK;
}
