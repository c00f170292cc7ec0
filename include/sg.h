/*
 * sg.h -- C-ABI of the B200-native multispin Monte Carlo library (libsg.so).
 *
 * The calls follow the paper's statement of the problem (arXiv:1906.11195):
 *   an instance (graph + couplings + random start)
 *   Metropolis sweeps, "update of the whole graph as unit of time", PAPER.md:260 (VB), :233 (SK)
 *   stored configurations and the two-time correlation C(t,t')
 *   the energy, PAPER.md:43 (Eq. 1), :73 (Eq. 3), :324
 * and BASELINE.json's north_star call list.  All conventions (bit meanings, Philox counter
 * layout, thresholds, colouring, schedule) are in DESIGN.md section 3.
 *
 * Everything runs on the current CUDA device, on torch's current CUDA stream; device
 * memory comes from torch's caching allocator (the process must have imported torch so
 * that libc10_cuda is loaded).  There is no CPU fallback: without a CUDA device sg_create
 * fails.  No function aborts or throws; failures return a negative code (or NULL) and set
 * a thread-local message readable with sg_last_error().
 *
 * Pointer arguments marked HOST are caller-owned host memory.  No device pointer crosses
 * this interface.  A handle must be used by one thread at a time.
 */
#ifndef SG_H
#define SG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sg_sim sg_sim; /* opaque; owns every device and host buffer of one simulation */

enum { SG_MODEL_VB = 0, SG_MODEL_SK = 1, SG_MODEL_RRBG = 2, SG_MODEL_RRG = 3 };
enum { SG_OK = 0, SG_EINVAL = -1, SG_ENOMEM = -2, SG_ECUDA = -3, SG_ESLOT = -4 };
#define SG_MAX_SLOTS 64

/*
 * sg_create -- build one simulation: n_words*64 independent samples ("lanes") that share the
 * interaction graph and differ in couplings and initial spins.
 *   model   SG_MODEL_VB: Viana-Bray +-J model (Eq. 3) on an Erdos-Renyi graph G(N, M),
 *                        M = floor(c*N/2 + 0.5), self-loops and multi-edges rejected (O2);
 *           SG_MODEL_SK: Sherrington-Kirkpatrick model (Eq. 1) with binary couplings
 *                        +-1/sqrt(N); c is ignored.
 *           SG_MODEL_RRBG: the Viana-Bray Hamiltonian on the paper's own graph ensemble, a random regular
 *                        bipartite graph of degree 4: halves {0..N/2-1} and {N/2..N-1},
 *                        four clash-free random permutations of one half onto the other (O2b), hence
 *                        exactly two colour classes; N even and >= 8; c is ignored.
 *           SG_MODEL_RRG: the same Hamiltonian on a random regular graph of degree 4 that is not bipartite (the ensemble of the
 *                        main text; Fig. S3, shows that bipartition is irrelevant): the first
 *                        simple graph of the pairing model (O2c); first-fit colour classes; 8 <= N < 2^30; c ignored.
 *   N       number of sites, 2 <= N < 2^31 - 2 (SK: N <= 32768 so that int16 local fields are exact).
 *   c       mean degree (VB), c >= 0 and M <= N(N-1)/2.
 *   T       temperature, 0 <= T <= +inf (T = 0 and T = inf are legal).
 *   seed    Philox key.  (model, N, c, T, seed, n_words) determine every bit of every output.
 *   n_words 64-bit words per site, 1 <= n_words <= 65535; lane l = 64*w + b is bit b of word w.
 * Spins start uniformly random, sweep counter = 0.
 * The handle belongs to the CUDA device that is current at this call; sg_sweep, sg_snapshot, sg_correlation, sg_energy
 * and sg_corr_accumulate return SG_EINVAL when another device is current.  Work is enqueued on torch's current stream.
 * Returns NULL on failure (bad argument, no CUDA device, out of memory).
 */
sg_sim *sg_create(int model, uint64_t N, double c, double T, uint64_t seed, uint32_t n_words);

/*
 * sg_create_opt -- sg_create with options (NULL = all defaults = sg_create).
 *   word0          the handle simulates words word0 .. word0+n_words-1 of the instance (model, N, c, T, seed): every
 *                  Philox counter that takes a word index takes word0 + w, so that a job can split the words of one
 *                  instance over several handles / GPUs and reproduce the single-handle run bit for bit (words share only
 *                  the graph; Q16, Q24).  Must be a multiple of 4; word0 + n_words <= 2^20.
 *   n_clones       SK only, 1 or 2: "two clones (i.e. replicas with the same couplings)" simulated side by side
 *                  (PAPER.md:233, :244).  Clone c of word w shares that word's couplings and draws its initial spins and
 *                  Metropolis uniforms as the virtual word w + c*2^20 (Q25).  The handle then has
 *                  64*n_words*n_clones lanes, clone-major: lane = c*64*n_words + 64*w + b; every per-lane output and
 *                  sg_get_spins / sg_set_spins (n_words*n_clones words per site) follow that order.
 *   aligned_start  1: every spin starts at +1 ("the initial configuration has all the spins aligned", PAPER.md:231;
 *                  DESIGN.md Q26) instead of the random start.
 */
typedef struct sg_options {
    uint32_t word0;
    uint32_t n_clones;        /* 0 is read as 1 */
    uint32_t aligned_start;
    uint32_t reserved;        /* must be 0 */
} sg_options;
sg_sim *sg_create_opt(int model, uint64_t N, double c, double T, uint64_t seed, uint32_t n_words, const sg_options *opt);
/* Number of lanes of the handle: 64 * n_words * n_clones. */
uint64_t sg_num_lanes(const sg_sim *h);

/* Release everything the handle owns (synchronises the stream first).  NULL is allowed. */
void sg_destroy(sg_sim *h);

/*
 * sg_sweep -- advance n full Metropolis sweeps (one sweep = every site of every lane proposed once:
 * VB colour class by colour class, SK sites 0..N-1 in order; O7/O8).  Asynchronous:
 * kernels are enqueued on the current stream.  n = 0 is a no-op.
 */
int sg_sweep(sg_sim *h, uint64_t n);

/*
 * sg_snapshot -- slot <- current configuration (device-to-device copy on the stream; the slot is
 * allocated on first use).  slot < SG_MAX_SLOTS, else SG_EINVAL.  Asynchronous.
 */
int sg_snapshot(sg_sim *h, uint32_t slot);

/*
 * sg_correlation -- out_counts[l] = D_l = #{ i : s_i(now) != s_i(slot) } for every lane l,
 * so that C(tw, tw+t) = 1 - 2*D_l/N.  Exact integers.
 *   out_counts  HOST, sg_num_lanes() = 64*n_words(*n_clones) uint64.
 * Synchronises the stream.  SG_ESLOT if the slot was never written.
 */
int sg_correlation(sg_sim *h, uint32_t slot, uint64_t *out_counts);

/*
 * sg_correlation_noalloc -- sg_correlation for callers that cannot allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): the same counts D_l, exact integers, with the
 * kernel's per-lane counters in a static device array of the library instead of a buffer of the handle.  The call makes no
 * cudaMalloc / cudaFree and calls no allocating routine.
 *   h           a handle of a graph model (VB, RRBG, RRG) with n_words <= sg_noalloc_max_words() = 64; beyond that
 *               SG_EINVAL with a message that names the limit (the array is 64 * 64 counters = 32 KiB, held by every GPU
 *               that loads the library until exit);
 *   slot        written by sg_snapshot before (SG_ESLOT otherwise; sg_snapshot allocates a slot on its first use, so
 *               write every slot at set-up);
 *   out_counts  HOST, 64*n_words uint64.
 * All handles and all calls share the one array; it is cleared at the start of every call.  Calls that overlap on the GPU
 * (different streams or host threads) race: serialise them.  Synchronises the stream.
 */
int sg_correlation_noalloc(sg_sim *h, uint32_t slot, uint64_t *out_counts);
uint32_t sg_noalloc_max_words(void);

/*
 * sg_energy -- per-lane energy of the current configuration, exact integers.
 *   VB: out[l] = E_l  = -sum_{(ij) in E} J_ij s_i s_j
 *   SK: out[l] = E'_l = -sum_{i<j} J'_ij s_i s_j with J' = +-1; energy = E'_l / sqrt(N)
 *   out  HOST, sg_num_lanes() int64.
 * Synchronises the stream.
 */
int sg_energy(sg_sim *h, int64_t *out);

/*
 * Windowed measurement (PAPER.md:95 "averaged over the time window", :270 minor-third intervals of tw + t; :233 tritone
 * lumps for SK): the paper averages C(tw, tw+t) over every sweep of a logarithmic time window, for several stored tw at
 * once.  These calls keep that bookkeeping on the device: bins of exact per-lane sums of D, nothing crosses PCIe and
 * nothing synchronises until the fetch.
 *   sg_corr_configure   allocate nbins accumulators (sg_num_lanes() uint64 each) and zero them, and their hit counts.
 *   sg_corr_accumulate  for k < n: acc[bins[k]][l] += D_l(now, slot slots[k]) and hits[bins[k]] += 1.  Asynchronous.  The
 *                       current configuration is read once per group of three slots (8 + 8S bytes per site-word instead
 *                       of 16 S).  slots, bins: HOST, n uint32; the bins of one call must be distinct; SG_ESLOT if a slot
 *                       was never written.
 *   sg_corr_fetch       out[b*lanes + l] = acc[bin0 + b][l] (HOST, nbins*lanes uint64), n_out[b] = hits (HOST, may be
 *                       NULL).  Synchronises the stream.  The caller's window average is C = 1 - 2*acc / (hits * N).
 */
int sg_corr_configure(sg_sim *h, uint32_t nbins);
int sg_corr_accumulate(sg_sim *h, uint32_t n, const uint32_t *slots, const uint32_t *bins);
int sg_corr_fetch(sg_sim *h, uint32_t bin0, uint32_t nbins, uint64_t *out, uint64_t *n_out);

/*
 * Site-sharded sweeps over several GPUs ("each half of the lattice is split among the GPUs; every GPU
 * holds a full copy of the spins; the updated spins are exchanged at each iteration, overlapped with the update").  VB
 * models only.  A colour class is a sequence of units (the slices of the device layout); every rank holds the whole
 * instance, updates its own units of the class, and the ranks exchange the spin words those units own before the next
 * class starts.  The library provides the pieces; the exchange itself is a collective of the caller
 * (paper_1906_11195_b200.workloads.sweep_site_sharded drives torch.distributed with them):
 *   sg_class_units       number of units of colour class k.
 *   sg_sweep_part        update units unit0 .. unit0+n-1 of class k at the current sweep index.  Asynchronous; the sweep
 *                        counter does not move.  Updating every unit of every class in class order, then sg_end_sweep, is
 *                        exactly sg_sweep(1).
 *   sg_end_sweep         sweep counter += 1.
 *   sg_part_range        the contiguous range [first, first + count) of 64-bit words of the device spin array that those
 *                        units own (device order: position-major, word-minor, gauge-transformed -- identical on every
 *                        rank because the layout is a function of (model, N, c, seed, n_words) only).
 *   sg_spin_device_pointer  the ONE device pointer that crosses this interface: the spin array (sg_num_sites()*n_words
 *                        uint64), so that a device-to-device collective (NCCL over NVLink) can exchange the ranges in
 *                        place.  sg_export_part / sg_import_part do the same through HOST buffers.
 */
int sg_class_units(sg_sim *h, uint32_t k, uint64_t *n_units);
int sg_sweep_part(sg_sim *h, uint32_t k, uint64_t unit0, uint64_t n_units);
int sg_end_sweep(sg_sim *h);
int sg_part_range(sg_sim *h, uint32_t k, uint64_t unit0, uint64_t n_units, uint64_t *first_word, uint64_t *n_words);
int sg_spin_device_pointer(sg_sim *h, void **ptr);
int sg_export_part(sg_sim *h, uint64_t first_word, uint64_t n_words, uint64_t *out /* HOST */);
int sg_import_part(sg_sim *h, uint64_t first_word, uint64_t n_words, const uint64_t *in /* HOST */);

/* Message of the last failure on this thread ("" if none). */
const char *sg_last_error(void);

/* ---- debug / test getters (synchronise; not on the timed path) ------------------------------ */

/* Number of sweeps done so far. */
uint64_t sg_sweep_count(const sg_sim *h);
/* Number of edges M (VB) or N(N-1)/2 (SK). */
uint64_t sg_num_edges(const sg_sim *h);
/* Number of colour classes K (VB; 0 for SK) and maximum degree (VB; N-1 for SK). */
uint32_t sg_num_colours(const sg_sim *h);
uint32_t sg_max_degree(const sg_sim *h);

/*
 * Spin words in ORIGINAL site order, word-minor: out[i*n_words + w], bit 1 <=> s = -1.
 *   slot  -1 = current configuration, else a snapshot slot (SG_ESLOT if never written).
 *   out   HOST, N*n_words uint64.
 */
int sg_get_spins(sg_sim *h, int32_t slot, uint64_t *out);

/*
 * Overwrite the current configuration / the sweep counter (tests: a sweep is a pure function of
 * (configuration, sweep index), Q15).  in: HOST, N*n_words uint64, original site order.
 */
int sg_set_spins(sg_sim *h, const uint64_t *in);
int sg_set_sweep_count(sg_sim *h, uint64_t t);

/*
 * VB graph in original labels: row_ptr HOST N+1 uint64, col HOST 2M uint32 (neighbours of i at
 * col[row_ptr[i] .. row_ptr[i+1]), in increasing edge id), colour HOST N uint32.  Any may be NULL.
 */
int sg_get_graph(sg_sim *h, uint64_t *row_ptr, uint32_t *col, uint32_t *colour);
/* VB edge list in generation order: u, v HOST M uint32 each. */
int sg_get_edges(sg_sim *h, uint32_t *u, uint32_t *v);
/*
 * Coupling words as stored on the device, bit 1 <=> J = -1.
 *   VB: out[e*n_words + w], edge order of generation (read back from the site-major device array).
 *   SK: out[pair(i,j)*n_words + w], i<j row-major upper triangle.
 *   out HOST, M*n_words uint64.
 */
int sg_get_couplings(sg_sim *h, uint64_t *out);
/* Acceptance thresholds thr[0..n) as 64-bit integers (index 0 unused = 0). out HOST n uint64. */
int sg_get_thresholds(sg_sim *h, uint64_t *out, uint64_t n);

/* ---- host-only entry points (no GPU needed; tests of the host generator and host Philox) -------- */

/* Philox4x32-10 block as the host generator evaluates it (O1). out HOST 4 uint32. */
void sg_host_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t *out);

/*
 * The VB instance exactly as sg_create lays it out for the device, built on
 * the host only.  Sites are relabelled to positions p = 0..N-1: class-major (colour 0, 1, ...), inside a class in
 * breadth-first order (BFS over the whole graph, roots in label order, rows in edge order): the locality-improving
 * relabelling.
 * Gauge: the BFS forest's edges ("tree entries", T) carry no coupling word: with eps_root = 0 and
 * eps_child = eps_parent ^ kappa_(tree edge) the device stores sigma ^ eps and kappa_ij ^ eps_i ^ eps_j, which leaves
 * every bond state sigma_i ^ sigma_j ^ kappa_ij, hence every output, unchanged.  The other entries ("X") keep a word.
 * Slices: every class is cut greedily, in position order, into runs of at most 32 sites with at most 32*it entries of
 * which at most 32*itx are X entries; (it, itx) is chosen per class, from the class's degrees, among the budgets the
 * kernels are compiled for: for odd n_words (6,4) if its cut needs at most 30 % more slices than that of (8,6), else
 * (8,6); (4,3) for even n_words (a thread then owns two words of its entry or site).  Inside a class every window of 4096 sites is
 * stably sorted by (demand, shape): demand 0 = a neighbour in a class of fewer than N/32 sites, 1 = fewer than N/8,
 * 2 = neither; shape 0 = at most 2 X and 2 T entries, 1 = at most 4 and 4, 2 = longer rows.  hdr[g] = 4 uint32: first
 * position, first index in col, first coupling entry, and n | nXs << 6 | nE << 16 | shape << 28 (sites, X entries, all entries, largest
 * shape of the slice); one sentinel follows the last slice.  col holds, slice after slice, ONE run of nE neighbour positions: the
 * X entries in site order (per site by ascending position), then the T entries in site order (per site: parent first,
 * then the children by ascending position); the coupling entries follow the X order, jeid gives the edge id of each.
 * orig_s[32g + j] = label of the j-th site of slice g (0xFFFFFFFF for j >= n); rp_s[32g + j] =
 * xOff | tOff << 8 | nX << 17 | nT << 22: where the site's X / T entries start inside the slice's run (nXs <= tOff <= nE),
 * and how many there are.  No output depends on any of this: the Philox counter
 * uses the original label (Q15).
 */
typedef struct sg_host_graph sg_host_graph;
/* model: SG_MODEL_VB, SG_MODEL_RRBG or SG_MODEL_RRG; NULL on bad arguments */
sg_host_graph *sg_host_graph_create(int model, uint64_t N, double c, uint64_t seed, uint32_t n_words);
void sg_host_graph_destroy(sg_host_graph *g);
/* info HOST 9 uint64: M, K (colours), dmax, entries (length of col = 2M), nslices, N, nJ (coupling entries), it_max (largest per-class it), gauge (1/0) */
int sg_host_graph_info(const sg_host_graph *g, uint64_t *info);
/*
 * Copies out whichever arrays are non-NULL (all HOST): u,v M uint32; colour N uint32; orig N uint32
 * (position -> label); hdr 4*(nslices+1) uint32; orig_s, rp_s 32*nslices uint32; col entries uint32; jeid nJ uint32;
 * tpar, teid N uint32 (parent position / tree edge id, 0xFFFFFFFF for roots); bfs_pos N uint32 (positions in
 * breadth-first order); class_pos0, class_n, class_slice0, class_nslices, class_it, class_itx K uint64 each.
 */
int sg_host_graph_get(const sg_host_graph *g, uint32_t *u, uint32_t *v, uint32_t *colour, uint32_t *orig,
                      uint32_t *hdr, uint32_t *orig_s, uint32_t *rp_s, uint32_t *col, uint32_t *jeid,
                      uint32_t *tpar, uint32_t *teid, uint32_t *bfs_pos,
                      uint64_t *class_pos0, uint64_t *class_n, uint64_t *class_slice0, uint64_t *class_nslices,
                      uint64_t *class_it, uint64_t *class_itx);

/*
 * Number of kernels this library has launched (process-wide, all handles) since load.
 * bench.py reports the difference over its timed region as "gpu_launches".
 */
uint64_t sg_kernel_launches(void);

#ifdef __cplusplus
}
#endif
#endif /* SG_H */
