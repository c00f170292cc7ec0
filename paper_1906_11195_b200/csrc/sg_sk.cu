// sg_sk.cu -- Sherrington-Kirkpatrick path (row a4 of SURVEY.md 8(a)).
//   H = -sum_{i<j} J_ij s_i s_j with binary couplings J_ij = J'_ij / sqrt(N), J' = +-1     PAPER.md:43 (Eq. 1), :233
//   "N single spin updates, performed in a fixed order" per iteration
//   multispin coding "to compute the force acting on a given spin (... the bottleneck)"
// Conventions: DESIGN.md section 3 (O3, O6, O8).
//
// Layout (lane = one disorder sample = one bit of the multispin word):
//   rows  [lane][i][NW32]  u32   bit j%32 of word j/32 = 1 <=> J'_ij = -1 (diagonal and padding bits 0)
//   H     [lane][Npad]     int16 integer local field H_i = sum_{j != i} J'_ij s_j, |H| <= N-1 <= 32767
//   sbits [lane][NW32]     u32   bit = 1 <=> s = -1   (the SK configuration; snapshots use the same layout)
// Clones (sg_options): lanes c*64W .. (c+1)*64W-1 are clone c; a clone shares the coupling rows of
// lane (l mod 64W) and draws spins and uniforms as the virtual word word0 + w + c*2^20 (Q25).
// One CTA owns one lane for a whole sg_sweep(n) call: fields, spins and the sweep's uniforms live in
// shared memory; sites are visited in order in batches of 32.  Warp 0 decides a batch speculatively
// (all 32 sites against the current fields, first acceptance by ballot + ffs, repair the 31 other
// fields of the batch from the prefetched diagonal block, repeat), then the whole CTA adds
// 2 J'_ij s_i to every other field for each accepted flip i of the batch, reading row i once.
#include <cuda_runtime.h>

#include <cstdlib>

#include <algorithm>

#include "sg_device.cuh"
#include "sg_sim.h"

void sgk_count_launch();

#define SK_LAUNCH_CHECK()                                                                      \
    do {                                                                                       \
        sgk_count_launch();                                                                    \
        cudaError_t e_ = cudaGetLastError();                                                   \
        if (e_ != cudaSuccess) {                                                               \
            sg_set_error(std::string("kernel launch failed: ") + cudaGetErrorString(e_));      \
            return SG_ECUDA;                                                                   \
        }                                                                                      \
    } while (0)

namespace {

constexpr int SK_THREADS = 288;      // warp 0 decides, the other eight apply
constexpr uint32_t SK_CLONE_STRIDE = 1u << 20;
constexpr int SK_PRE = 8;                // uint4 a worker thread stages per batch: 256 threads * 8 * 16 B = 32 KiB = the block at N = 8192

__host__ __device__ inline uint32_t sk_nw32(uint64_t N) { return (uint32_t)((N + 31) / 32); }
// padded row length of the transposed field array in shared memory: 2 * odd, so that the 32 lanes of
// the deciding warp (stride nw32p int16) hit 32 different banks
__host__ __device__ inline uint32_t sk_nw32p(uint32_t nw32) { uint32_t h = (nw32 + 1) / 2; if (!(h & 1)) ++h; return 2 * h; }

// O3 (SK): kappa_ij[w] = x0 | x1<<32 of P(c0 = j, c1 = w, sweep field = i, tag 2) for i < j.
// One warp per (i, word wq of j's, w): lane = j % 32 draws its coupling word, 64 ballots transpose
// the 32 x 64 bit block into one u32 per lane.
__global__ void __launch_bounds__(256) k_sk_init_rows(uint32_t *__restrict__ rows, uint64_t N, uint32_t NW32, uint32_t W, uint32_t word0,
                                                      uint32_t k0, uint32_t k1)
{
    const uint64_t warp = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t lane = threadIdx.x & 31u;
    const uint64_t total = N * NW32 * W;
    if (warp >= total) return;
    const uint32_t w = (uint32_t)(warp % W);
    const uint32_t wq = (uint32_t)((warp / W) % NW32);
    const uint64_t i = warp / ((uint64_t)W * NW32);
    const uint64_t j = 32ull * wq + lane;
    uint64_t kappa = 0;
    if (j < N && j != i) {
        const uint32_t lo = (uint32_t)(i < j ? i : j), hi = (uint32_t)(i < j ? j : i);
        uint32_t x[4];
        philox4x32_10(hi, word0 + w, lo, 2u << 24, k0, k1, x);
        kappa = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
    }
    uint32_t mine0 = 0, mine1 = 0;
#pragma unroll
    for (int b = 0; b < 32; ++b) {
        const uint32_t v0 = __ballot_sync(0xFFFFFFFFu, (kappa >> b) & 1ull);
        const uint32_t v1 = __ballot_sync(0xFFFFFFFFu, (kappa >> (b + 32)) & 1ull);
        if (lane == (uint32_t)b) { mine0 = v0; mine1 = v1; }
    }
    const uint64_t lane_g0 = 64ull * w + lane;
    rows[(lane_g0 * N + i) * NW32 + wq] = mine0;
    rows[((lane_g0 + 32) * N + i) * NW32 + wq] = mine1;
}

// H_i = sum_{j != i} J'_ij s_j = (N - 1) - 2 * #{ j != i : kappa_ij xor sigma_j = 1 }
__global__ void __launch_bounds__(256) k_sk_init_fields(const uint32_t *__restrict__ rows, const uint32_t *__restrict__ sbits,
                                                        int16_t *__restrict__ H, uint64_t N, uint32_t NW32, uint32_t lanes_w)
{
    const uint64_t lane_g = blockIdx.y;
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t *row = rows + ((lane_g % lanes_w) * N + i) * NW32;
    const uint32_t *sp = sbits + lane_g * NW32;
    uint32_t neg = 0;
    for (uint32_t wq = 0; wq < NW32; ++wq) {
        uint32_t x = row[wq] ^ sp[wq];
        if (wq == NW32 - 1 && (N & 31)) x &= (1u << (N & 31)) - 1u;   // padding bits
        if (wq == (uint32_t)(i >> 5)) x &= ~(1u << (i & 31));          // j = i
        neg += __popc(x);
    }
    H[lane_g * (32ull * NW32) + i] = (int16_t)((int)(N - 1) - 2 * (int)neg);
}

// O4 for the lane-major layout: bit (64w+b) of site i of clone c = bit b of x0|x1<<32 of P(i, word0 + w + c*2^20, 0, tag 1);
// aligned start: every bit 0.  One warp per (32 sites, w, c): lane = site, 64 ballots transpose.
__global__ void __launch_bounds__(256) k_sk_init_spins(uint32_t *__restrict__ sbits, uint64_t N, uint32_t NW32, uint32_t W, uint32_t clones,
                                                       uint32_t word0, int aligned, uint32_t k0, uint32_t k1)
{
    const uint64_t warp = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t lane = threadIdx.x & 31u;
    if (warp >= (uint64_t)NW32 * W * clones) return;
    const uint32_t w = (uint32_t)(warp % W), c = (uint32_t)((warp / W) % clones), wq = (uint32_t)(warp / ((uint64_t)W * clones));
    const uint64_t i = 32ull * wq + lane;
    uint64_t sigma = 0;
    if (i < N && !aligned) {
        uint32_t x[4];
        philox4x32_10((uint32_t)i, word0 + w + c * SK_CLONE_STRIDE, 0u, 1u << 24, k0, k1, x);
        sigma = (uint64_t)x[0] | ((uint64_t)x[1] << 32);
    }
    uint32_t mine0 = 0, mine1 = 0;
#pragma unroll
    for (int b = 0; b < 32; ++b) {
        const uint32_t v0 = __ballot_sync(0xFFFFFFFFu, (sigma >> b) & 1ull);
        const uint32_t v1 = __ballot_sync(0xFFFFFFFFu, (sigma >> (b + 32)) & 1ull);
        if (lane == (uint32_t)b) { mine0 = v0; mine1 = v1; }
    }
    const uint64_t l0 = 64ull * ((uint64_t)c * W + w) + lane;
    sbits[l0 * NW32 + wq] = mine0;
    sbits[(l0 + 32) * NW32 + wq] = mine1;
}

// named barriers of the sweep kernel (producer / consumer between the deciding warp and the others)
__device__ __forceinline__ void sk_bar_sync(uint32_t id) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(SK_THREADS) : "memory"); }
__device__ __forceinline__ void sk_bar_arrive(uint32_t id) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(SK_THREADS) : "memory"); }

// ---------------------------------------------------------------------------------------- the sweep
// dynamic shared memory: int16 Hs[32 * nw32p] (transposed: field of site j at (j%32)*nw32p + j/32),
//                        u32 rs[32 * NW32] (this sweep's uniforms), u32 sp[NW32] (spin bits), u32 ctl[4]
__global__ void __launch_bounds__(SK_THREADS)
k_sk_sweep(const uint32_t *__restrict__ rows, int16_t *__restrict__ Hg, uint32_t *__restrict__ sbits,
           const uint64_t *__restrict__ thr, uint32_t N, uint32_t NW32, uint32_t mz /* thr[m] = 0 for m >= mz */,
           uint32_t lanes_w, uint32_t word0, uint64_t sweep0, uint32_t nsweeps, uint32_t k0, uint32_t k1, uint32_t stage_off /* 0: rows not staged */)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const uint32_t nw32p = sk_nw32p(NW32);
    int16_t *Hs = reinterpret_cast<int16_t *>(smem_raw);
    uint32_t *rs = reinterpret_cast<uint32_t *>(smem_raw + ((32u * nw32p * 2u + 15u) & ~15u));
    uint32_t *sp = rs + 32u * NW32;
    volatile uint32_t *ctl = sp + NW32;
    const bool staged = stage_off != 0;
    uint4 *rowbuf = reinterpret_cast<uint4 *>(smem_raw + stage_off);      // two buffers of 32 * NW32 words (8 * NW32 uint4)

    const uint32_t lane_g = blockIdx.x;
    const uint32_t w = word0 + ((lane_g % lanes_w) >> 6) + (lane_g / lanes_w) * SK_CLONE_STRIDE;   // virtual word of the uniforms
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t *myrows = rows + (uint64_t)(lane_g % lanes_w) * N * NW32;
    int16_t *myH = Hg + (uint64_t)lane_g * 32u * NW32;
    uint32_t *mysp = sbits + (uint64_t)lane_g * NW32;

    for (uint32_t j = tid; j < 32u * NW32; j += SK_THREADS) Hs[(j & 31u) * nw32p + (j >> 5)] = j < N ? myH[j] : (int16_t)0;
    for (uint32_t q = tid; q < NW32; q += SK_THREADS) sp[q] = mysp[q];

    for (uint32_t s = 0; s < nsweeps; ++s) {
        const uint64_t t = sweep0 + s;
        // O8: r = x_{w&3} of P(i, w>>2, t, tag 0), shared by the 64 lanes of word w
        for (uint32_t i = tid; i < N; i += SK_THREADS) {
            uint32_t x[4];
            philox4x32_10(i, w >> 2, (uint32_t)t, (uint32_t)(t >> 32), k0, k1, x);
            rs[i] = (w & 2u) ? ((w & 1u) ? x[3] : x[2]) : ((w & 1u) ? x[1] : x[0]);
        }
        // Two roles, one batch apart.  Warp 0 (the decider) visits the 32 sites of batch b in order, then adds the batch's
        // flips to the 32 fields of batch b + 1 (the only fields its next decision reads) and publishes the flips; warps
        // 1-7 (the workers) add them to every other field while the decider is already at batch b + 1.
        //   full[b & 1]: the decider has published batch b          (decider arrives, workers wait)
        //   done[b & 1]: the workers have applied batch b           (workers arrive, decider waits before it touches the
        //                fields of batch b + 2, which the workers of batch b also write)
        // decider: lane l prefetches, of row 32 b + l, word b (the 32 x 32 diagonal block) and word b + 1 (towards the next batch)
        uint32_t diag = 0, nxt = 0;
        if (warp == 0 && lane < N) {
            diag = myrows[(uint64_t)lane * NW32 + 0];
            if (NW32 > 1) nxt = myrows[(uint64_t)lane * NW32 + 1];
        }
        __syncthreads();                                              // uniforms of this sweep are in place
        if (warp == 0) {
            for (uint32_t b = 0; b < NW32; ++b) {
                const uint32_t i = 32u * b + lane;
                const bool valid = i < N;
                int h = Hs[lane * nw32p + b];
                uint32_t spw = sp[b];
                const uint32_t r = valid ? rs[i] : 0u;
                uint32_t todo = 0xFFFFFFFFu, F = 0;
                while (true) {
                    const int m = ((spw >> lane) & 1u) ? -h : h;      // s_i * H_i
                    bool acc = false;
                    if (valid) {
                        if (m <= 0) acc = true;
                        else if ((uint32_t)m < mz) acc = (uint64_t)r < __ldg(thr + m);
                    }
                    const uint32_t bal = __ballot_sync(0xFFFFFFFFu, acc) & todo;
                    if (!bal) break;
                    const uint32_t k = __ffs(bal) - 1u;               // first accepted site, in order
                    F |= 1u << k;
                    spw ^= 1u << k;
                    const int snew2 = ((spw >> k) & 1u) ? -2 : 2;     // 2 * s_k(new)
                    const uint32_t rw = __shfl_sync(0xFFFFFFFFu, diag, k);
                    if (lane != k) h += ((rw >> lane) & 1u) ? -snew2 : snew2;   // H_j += 2 J'_kj s_k
                    todo = (k == 31u) ? 0u : (0xFFFFFFFFu << (k + 1u));
                }
                Hs[lane * nw32p + b] = (int16_t)h;
                if (b >= 1) sk_bar_sync(3u + ((b - 1u) & 1u));        // done[b - 1]: nobody else writes batch b + 1's fields now
                if (b + 1 < NW32) {
                    int hn = Hs[lane * nw32p + b + 1];
                    uint32_t Fl = F;
                    while (Fl) {
                        const uint32_t k = __ffs(Fl) - 1u;
                        Fl &= Fl - 1u;
                        const int snew2 = ((spw >> k) & 1u) ? -2 : 2;
                        const uint32_t rw = __shfl_sync(0xFFFFFFFFu, nxt, k);
                        hn += ((rw >> lane) & 1u) ? -snew2 : snew2;
                    }
                    Hs[lane * nw32p + b + 1] = (int16_t)hn;
                }
                if (lane == 0) { sp[b] = spw; ctl[b & 1u] = F; }
                __threadfence_block();
                sk_bar_arrive(1u + (b & 1u));                         // full[b]
                if (b + 1 < NW32) {                                   // prefetch for the next batch
                    const uint32_t inext = 32u * (b + 1) + lane;
                    diag = 0; nxt = 0;
                    if (inext < N) {
                        diag = myrows[(uint64_t)inext * NW32 + (b + 1)];
                        if (b + 2 < NW32) nxt = myrows[(uint64_t)inext * NW32 + (b + 2)];
                    }
                }
            }
            sk_bar_sync(3u + ((NW32 - 1u) & 1u));                     // done[last]
        } else {
            const uint32_t wtid = tid - 32u;
            constexpr uint32_t NWK = SK_THREADS - 32u;                // worker threads
            const uint32_t blk4 = 8u * NW32;                          // uint4 per staged block (32 full rows: N % 128 == 0)
            if (staged) {                                             // batch 0's rows; the full[0] barrier below publishes them
                const uint4 *g4 = reinterpret_cast<const uint4 *>(myrows);
                for (uint32_t q = wtid; q < blk4; q += NWK) rowbuf[q] = __ldg(g4 + q);
            }
            for (uint32_t b = 0; b < NW32; ++b) {
                sk_bar_sync(1u + (b & 1u));                           // full[b]: also, every worker is past batch b - 1
                const uint32_t F = ctl[b & 1u];
                // the next batch's rows: loads issued now, stored to the other buffer after this batch's work
                uint4 pre[SK_PRE];
                const bool more = staged && b + 1 < NW32;
                if (more) {
                    const uint4 *g4 = reinterpret_cast<const uint4 *>(myrows + (uint64_t)32u * (b + 1) * NW32);
#pragma unroll
                    for (int u = 0; u < SK_PRE; ++u)
                        if (wtid + u * NWK < blk4) pre[u] = __ldg(g4 + wtid + u * NWK);
                }
                const uint32_t *grow = myrows + (uint64_t)32u * b * NW32;                                    // rows of this batch, global
                const uint32_t *srow = reinterpret_cast<const uint32_t *>(rowbuf + (b & 1u) * blk4);          // ... and staged
                if (F) {
                    const uint32_t spw = sp[b];
                    // each thread owns half-words of the row: item it -> word it>>1, bits 16*(it&1) .. +15
                    for (uint32_t it = wtid; it < 2u * NW32; it += SK_THREADS - 32u) {
                        const uint32_t wq = it >> 1, half = it & 1u;
                        if (wq == b || wq == b + 1u) continue;        // done by the decider
                        int16_t *hp = Hs + (16u * half) * nw32p + wq;
                        uint32_t Fl = F;
                        while (Fl) {
                            // up to four flips at a time: their row words are read together (independent loads), then added
                            uint32_t kk[4], rw[4];
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                kk[u] = 32u;
                                rw[u] = 0;
                                if (Fl) {
                                    kk[u] = __ffs(Fl) - 1u;
                                    Fl &= Fl - 1u;
                                    rw[u] = (staged ? srow[kk[u] * NW32 + wq] : __ldg(grow + kk[u] * NW32 + wq)) >> (16u * half);
                                }
                            }
                            int d[16];
#pragma unroll
                            for (int q = 0; q < 16; ++q) d[q] = 0;
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                if (kk[u] < 32u) {
                                    const int snew2 = ((spw >> kk[u]) & 1u) ? -2 : 2;
#pragma unroll
                                    for (int q = 0; q < 16; ++q) d[q] += ((rw[u] >> q) & 1u) ? -snew2 : snew2;
                                }
                            }
#pragma unroll
                            for (int q = 0; q < 16; ++q) hp[q * nw32p] += (int16_t)d[q];
                        }
                    }
                }
                if (more) {
#pragma unroll
                    for (int u = 0; u < SK_PRE; ++u)
                        if (wtid + u * NWK < blk4) rowbuf[((b + 1u) & 1u) * blk4 + wtid + u * NWK] = pre[u];
                }
                __threadfence_block();
                sk_bar_arrive(3u + (b & 1u));                         // done[b]
            }
        }
        __syncthreads();                                              // end of the sweep: every field is up to date
    }
    __syncthreads();
    for (uint32_t j = tid; j < N; j += SK_THREADS) myH[j] = Hs[(j & 31u) * nw32p + (j >> 5)];
    for (uint32_t q = tid; q < NW32; q += SK_THREADS) mysp[q] = sp[q];
}

// E'_lane = -sum_{i<j} J'_ij s_i s_j = -1/2 sum_i s_i H_i
__global__ void __launch_bounds__(256) k_sk_energy(const int16_t *__restrict__ H, const uint32_t *__restrict__ sbits,
                                                   uint32_t N, uint32_t NW32, long long *__restrict__ out)
{
    __shared__ long long part[8];
    const uint32_t lane_g = blockIdx.x;
    long long acc = 0;
    for (uint32_t i = threadIdx.x; i < N; i += blockDim.x) {
        const int h = H[(uint64_t)lane_g * 32u * NW32 + i];
        const uint32_t bit = (sbits[(uint64_t)lane_g * NW32 + (i >> 5)] >> (i & 31u)) & 1u;
        acc += bit ? -h : h;
    }
    for (int off = 16; off; off >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, off);
    if ((threadIdx.x & 31u) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        long long tot = 0;
        for (uint32_t q = 0; q < blockDim.x / 32; ++q) tot += part[q];
        out[lane_g] = -tot / 2;
    }
}

// D_lane = popcount(sbits_now[lane] ^ sbits_slot[lane])
__global__ void __launch_bounds__(256) k_sk_correlation(const uint32_t *__restrict__ a, const uint32_t *__restrict__ b,
                                                        uint32_t NW32, unsigned long long *__restrict__ out, int accumulate)
{
    __shared__ uint32_t part[8];
    const uint32_t lane_g = blockIdx.x;
    uint32_t acc = 0;
    for (uint32_t q = threadIdx.x; q < NW32; q += blockDim.x)
        acc += __popc(a[(uint64_t)lane_g * NW32 + q] ^ b[(uint64_t)lane_g * NW32 + q]);
    for (int off = 16; off; off >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, off);
    if ((threadIdx.x & 31u) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t tot = 0;
        for (uint32_t q = 0; q < blockDim.x / 32; ++q) tot += part[q];
        out[lane_g] = accumulate ? out[lane_g] + tot : tot;
    }
}

// The 32 coupling rows of a batch are one contiguous block of 128 * NW32 bytes; for N <= 8192 (and N a multiple of 128, so
// that the block is a whole number of 16-byte units) two such blocks fit in shared memory: the workers copy the next
// batch's block in while they apply the current batch (SG_SK_STAGE=0 switches that off: a measurement knob).
bool sk_staged(uint32_t NW32)
{
    static const bool off = std::getenv("SG_SK_STAGE") && std::getenv("SG_SK_STAGE")[0] == '0';
    return !off && NW32 % 4u == 0 && NW32 <= 256u;
}
size_t sk_smem_base(uint32_t NW32)
{
    const uint32_t nw32p = sk_nw32p(NW32);
    return (((32u * nw32p * 2u + 15u) & ~15u) + 4u * (32u * NW32 + NW32 + 4u) + 15u) & ~(size_t)15u;
}
size_t sk_smem_bytes(uint32_t NW32) { return sk_smem_base(NW32) + (sk_staged(NW32) ? 2u * 128u * NW32 : 0u); }

}  // namespace

int sg_sk_create_impl(sg_sim *h)
{
    cudaStream_t st = sgx_stream();
    const uint64_t N = h->N;
    const uint32_t W = h->W, NW32 = sk_nw32(N);
    const uint64_t lanes = h->lanes, lanes_w = 64ull * W;
    h->M = N * (N - 1) / 2;
    h->spin_words = lanes * NW32 / 2;   // u32 words, lanes even -> whole u64 count
    SKDevice &d = h->sk;
    d.rows = dev_alloc<uint32_t>(h, lanes_w * N * NW32);
    d.H = dev_alloc<int16_t>(h, lanes * 32ull * NW32);
    d.spin = dev_alloc<uint64_t>(h, h->spin_words);
    d.thr = dev_alloc<uint64_t>(h, N);
    if (!d.rows || !d.H || !d.spin || !d.thr) return SG_ENOMEM;
    h->thr_host = sg_sk_thresholds(h->T, N);
    uint32_t mz = (uint32_t)N;
    for (uint64_t m = 1; m < N; ++m)
        if (h->thr_host[m] == 0) { mz = (uint32_t)m; break; }
    d.nthr_nz = mz;
    if (!upload(d.thr, h->thr_host, st)) return SG_ECUDA;
    const size_t smem = sk_smem_bytes(NW32);
    if (smem > 227 * 1024) { sg_set_error("SK: N too large for the shared-memory field array"); return SG_EINVAL; }
    {
        const uint64_t warps = N * NW32 * W;
        k_sk_init_rows<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, st>>>(d.rows, N, NW32, W, h->word0, h->key.k0, h->key.k1);
        SK_LAUNCH_CHECK();
    }
    {
        const uint64_t warps = (uint64_t)NW32 * W * h->clones;
        k_sk_init_spins<<<(unsigned)((warps * 32 + 255) / 256), 256, 0, st>>>((uint32_t *)d.spin, N, NW32, W, h->clones, h->word0,
                                                                              h->aligned ? 1 : 0, h->key.k0, h->key.k1);
        SK_LAUNCH_CHECK();
    }
    {
        dim3 grid((unsigned)((N + 255) / 256), (unsigned)lanes);
        k_sk_init_fields<<<grid, 256, 0, st>>>(d.rows, (const uint32_t *)d.spin, d.H, N, NW32, (uint32_t)lanes_w);
        SK_LAUNCH_CHECK();
    }
    if (!cuda_ok(cudaStreamSynchronize(st), "sg_create (SK)")) return SG_ECUDA;
    return SG_OK;
}

int sg_sk_sweep_impl(sg_sim *h, uint64_t n)
{
    cudaStream_t st = sgx_stream();
    const uint32_t NW32 = sk_nw32(h->N);
    const size_t smem = sk_smem_bytes(NW32);
    // the limit is a property of the function, not of the handle: set it to this handle's need before every launch
    // (another handle with a smaller N may have lowered it since)
    if (!cuda_ok(cudaFuncSetAttribute(k_sk_sweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem), "SK smem attribute")) return SG_ECUDA;
    while (n) {
        const uint32_t chunk = (uint32_t)std::min<uint64_t>(n, 1u << 20);
        k_sk_sweep<<<(unsigned)h->lanes, SK_THREADS, smem, st>>>(h->sk.rows, h->sk.H, (uint32_t *)h->sk.spin, h->sk.thr, (uint32_t)h->N, NW32,
                                                                 h->sk.nthr_nz, 64u * h->W, h->word0, h->sweep, chunk, h->key.k0, h->key.k1,
                                                                 sk_staged(NW32) ? (uint32_t)sk_smem_base(NW32) : 0u);
        SK_LAUNCH_CHECK();
        h->sweep += chunk;
        n -= chunk;
    }
    return SG_OK;
}

int sg_sk_energy_impl(sg_sim *h, int64_t *out)
{
    cudaStream_t st = sgx_stream();
    const uint64_t lanes = h->lanes;
    k_sk_energy<<<(unsigned)lanes, 256, 0, st>>>(h->sk.H, (const uint32_t *)h->sk.spin, (uint32_t)h->N, sk_nw32(h->N),
                                                 (long long *)h->counts_dev);
    SK_LAUNCH_CHECK();
    if (!cuda_ok(cudaMemcpyAsync(out, h->counts_dev, lanes * 8, cudaMemcpyDeviceToHost, st), "sg_energy") ||
        !cuda_ok(cudaStreamSynchronize(st), "sg_energy"))
        return SG_ECUDA;
    return SG_OK;
}

int sg_sk_correlation_impl(sg_sim *h, const uint64_t *slot_dev, uint64_t *out)
{
    cudaStream_t st = sgx_stream();
    const uint64_t lanes = h->lanes;
    k_sk_correlation<<<(unsigned)lanes, 256, 0, st>>>((const uint32_t *)h->sk.spin, (const uint32_t *)slot_dev, sk_nw32(h->N),
                                                      (unsigned long long *)h->counts_dev, 0);
    SK_LAUNCH_CHECK();
    if (!cuda_ok(cudaMemcpyAsync(out, h->counts_dev, lanes * 8, cudaMemcpyDeviceToHost, st), "sg_correlation") ||
        !cuda_ok(cudaStreamSynchronize(st), "sg_correlation"))
        return SG_ECUDA;
    return SG_OK;
}

// acc[lane] += D_lane(current, slot): the windowed protocol's accumulation, asynchronous
int sg_sk_corr_accumulate_impl(sg_sim *h, const uint64_t *slot_dev, uint64_t *acc_dev)
{
    cudaStream_t st = sgx_stream();
    k_sk_correlation<<<(unsigned)h->lanes, 256, 0, st>>>((const uint32_t *)h->sk.spin, (const uint32_t *)slot_dev, sk_nw32(h->N),
                                                         (unsigned long long *)acc_dev, 1);
    SK_LAUNCH_CHECK();
    return SG_OK;
}

// lane-major bit arrays <-> site-major multispin words (host side; debug getters only)
int sg_sk_get_spins_impl(sg_sim *h, const uint64_t *src_dev, uint64_t *out)
{
    cudaStream_t st = sgx_stream();
    const uint32_t NW32 = sk_nw32(h->N), W = h->W * h->clones;      // lane groups per site, clone-major
    const uint64_t lanes = h->lanes;
    std::vector<uint32_t> bits(lanes * NW32);
    if (!cuda_ok(cudaMemcpyAsync(bits.data(), src_dev, bits.size() * 4, cudaMemcpyDeviceToHost, st), "sg_get_spins") ||
        !cuda_ok(cudaStreamSynchronize(st), "sg_get_spins"))
        return SG_ECUDA;
    std::fill(out, out + h->N * W, 0ull);
    for (uint64_t l = 0; l < lanes; ++l)
        for (uint64_t i = 0; i < h->N; ++i)
            if ((bits[l * NW32 + (i >> 5)] >> (i & 31)) & 1u) out[i * W + (l >> 6)] |= 1ull << (l & 63);
    return SG_OK;
}

int sg_sk_set_spins_impl(sg_sim *h, const uint64_t *in)
{
    cudaStream_t st = sgx_stream();
    const uint32_t NW32 = sk_nw32(h->N), W = h->W * h->clones;
    const uint64_t lanes = h->lanes;
    std::vector<uint32_t> bits(lanes * NW32, 0u);
    for (uint64_t l = 0; l < lanes; ++l)
        for (uint64_t i = 0; i < h->N; ++i)
            if ((in[i * W + (l >> 6)] >> (l & 63)) & 1ull) bits[l * NW32 + (i >> 5)] |= 1u << (i & 31);
    if (!cuda_ok(cudaMemcpyAsync(h->sk.spin, bits.data(), bits.size() * 4, cudaMemcpyHostToDevice, st), "sg_set_spins")) return SG_ECUDA;
    dim3 grid((unsigned)((h->N + 255) / 256), (unsigned)lanes);
    k_sk_init_fields<<<grid, 256, 0, st>>>(h->sk.rows, (const uint32_t *)h->sk.spin, h->sk.H, h->N, NW32, 64u * h->W);
    SK_LAUNCH_CHECK();
    if (!cuda_ok(cudaStreamSynchronize(st), "sg_set_spins")) return SG_ECUDA;
    return SG_OK;
}

int sg_sk_get_couplings_impl(sg_sim *h, uint64_t *out)
{
    cudaStream_t st = sgx_stream();
    const uint64_t N = h->N;
    const uint32_t NW32 = sk_nw32(N), W = h->W;
    const uint64_t lanes = 64ull * W;
    std::vector<uint32_t> rows(lanes * N * NW32);
    if (!cuda_ok(cudaMemcpyAsync(rows.data(), h->sk.rows, rows.size() * 4, cudaMemcpyDeviceToHost, st), "sg_get_couplings") ||
        !cuda_ok(cudaStreamSynchronize(st), "sg_get_couplings"))
        return SG_ECUDA;
    std::fill(out, out + h->M * W, 0ull);
    for (uint64_t l = 0; l < lanes; ++l) {
        uint64_t pair = 0;
        for (uint64_t i = 0; i < N; ++i)
            for (uint64_t j = i + 1; j < N; ++j, ++pair) {
                const uint32_t up = (rows[(l * N + i) * NW32 + (j >> 5)] >> (j & 31)) & 1u;
                const uint32_t lo = (rows[(l * N + j) * NW32 + (i >> 5)] >> (i & 31)) & 1u;
                if (up != lo) { sg_set_error("SK coupling rows are not symmetric"); return SG_ECUDA; }
                if (up) out[pair * W + (l >> 6)] |= 1ull << (l & 63);
            }
    }
    return SG_OK;
}
