/*
 * sw.h -- C ABI of libsw_b200: one Swendsen-Wang (SW) multi-cluster Monte Carlo step on one
 * NVIDIA B200 (sm_100a), after arXiv 1403.7560 (Komura & Okabe), section 2.
 *
 * One SW step is
 *   (1) active-bond generation between aligned nearest neighbours,
 *   (2) cluster labelling = connected components of the active-bond graph,
 *   (3) a new random value per cluster (Ising, Potts) or a reflection of the whole cluster with
 *       probability 1/2 (XY, Wolff embedding) applied to every site,
 * followed, on request, by the observables of PAPER.md:142-157 (Eq. 1-5).
 * Lattices: periodic 2D square and 3D simple cubic.  Models: Ising (Eq. 1), q-state
 * Potts (Eq. 2), classical XY with continuous fp32 angles (Eq. 3).  J = 1, beta = 1/T.
 *
 * Every step of the path runs in hand-written CUDA kernels; there is NO CPU fallback: without a
 * usable CUDA device every call that needs one returns SW_ECUDA.
 *
 * Conventions (DESIGN.md section 3 lists every reading of the paper):
 *   site index   i = x + L*y (+ L*L*z), x fastest; each site owns its +x, +y (, +z) bonds;
 *   bond byte    bit k = the bond from site i to its +e_k neighbour is active;
 *   label        minimum linear site index of the site's cluster (what label equivalence with
 *                atomicMin from label = index converges to);
 *   randoms      Philox4x32-10, key = (seed low, seed high), counter = (index, t low, t high,
 *                domain), t = 0-based index of the step being executed (reading 6, spec
 *                version 2).  XY, clock: domain 0, index = site, word k decides bond k of the site, the
 *                top bit of word 3 is the draw of the cluster rooted at the site.  Ising, Potts: domain
 *                5, index = group G = site / 32; the group's words W_G[n] = word n % 4 of the call with
 *                counter word 3 = 5 + 256 (n / 4).  Bit b = site % 32 of W_G[1 + s dim + k] is binary digit
 *                31 - s of the 32-bit uniform integer u(site, k); bond k is active iff the neighbours are
 *                equal and u < floor(p 2^32).  Bit b of W_G[0]: Ising cluster draw; W_G[128 + b]: Potts
 *                draw word (new state (w q) >> 32).  Domain 2: start configuration; domain 3: XY
 *                direction / clock mirror of step t.
 *
 * Pointers: `sw_ctx *` is an opaque HOST pointer owned by the library.  All `host_*` arguments
 * are HOST pointers owned by the caller.  `device_workspace` (sw_create_in) is a DEVICE pointer
 * owned by the caller, which must outlive the context.  Nothing else crosses the boundary.
 *
 * Errors: every call returns an int status (SW_OK = 0, negative on error), never throws and never
 * aborts.  sw_last_error() returns a thread-local description of the last failure.  CUDA errors
 * are sticky in the context: after one, every later call on that context returns SW_ECUDA.
 *
 * Threading: one context = one CUDA stream; calls on one context are not re-entrant.
 */
#ifndef SW_B200_H
#define SW_B200_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sw_ctx sw_ctx;

enum { SW_ISING = 0, SW_POTTS = 1, SW_XY = 2, SW_CLOCK = 3 };
enum { SW_OK = 0, SW_EINVAL = -1, SW_ENOMEM = -2, SW_ECUDA = -3, SW_ESTATE = -4 };

/* ---- the four calls of the hot path ------------------------------------------------------- */

/* Create a context for a dim-dimensional (2 or 3) periodic lattice of linear size L with a seeded
 * random start configuration (device_function_spinset) and step counter t = 0.
 *   L      multiple of 32 ("nx ... multiple of 32"), L >= 32, L^dim <= 2^31;
 *   model  SW_ISING | SW_POTTS | SW_XY | SW_CLOCK;  q: number of Potts states, 2..255, with
 *          L^dim * 2^ceil(log2 q) <= 2^32 (a label word holds a site address and a state), or number
 *          of clock states, 2..512; ignored otherwise;
 *   beta   J/T with J = 1, finite, >= 0;  seed: Philox key.
 * Device memory comes from cudaMalloc and the context owns a new non-blocking stream.
 * On failure *out = NULL. */
int sw_create(sw_ctx **out, int dim, int L, int model, int q, double beta, uint64_t seed);

/* Same, but the context lives in caller-provided DEVICE memory (e.g. a torch tensor from the
 * caching allocator) of at least sw_workspace_bytes() bytes, 256-byte aligned, and launches on
 * the caller's CUDA stream (`cuda_stream` is a cudaStream_t passed as void *; NULL = the legacy
 * default stream).  The caller keeps ownership of both. */
int sw_create_in(sw_ctx **out, int dim, int L, int model, int q, double beta, uint64_t seed,
                 void *device_workspace, size_t workspace_bytes, void *cuda_stream);
/* Bytes sw_create_in needs; 0 if the arguments are invalid. */
size_t sw_workspace_bytes(int dim, int L, int model, int q);

/* n >= 0 SW steps, asynchronous on the context's stream (no host sync). */
int sw_step(sw_ctx *c, int n);

/* Instantaneous, extensive observables of the CURRENT configuration.
 * Synchronises the stream.  Any output pointer may be NULL.
 *   Ising: E = -sum_<ij> s_i s_j (Eq. 1), M = sum_i s_i (Eq. 4, signed), M2 = M^2, M4 = M^4.
 *   Potts: E = number of unequal nearest-neighbour pairs (Eq. 2), M2 = (q sum_k n_k^2 - N^2)/(q-1)
 *          (Eq. 5), M = sqrt(M2), M4 = M2^2.
 *   XY:    E = -sum_<ij> cos(theta_i - theta_j) (Eq. 3), M = |sum_i (cos, sin)|, M2, M4 likewise.
 *   Clock: as XY with theta = 2 pi p / q, from exact integer histograms.
 * Averages, the specific heat and the moment ratio (Eq. 6) are the caller's job.  Spins injected
 * with sw_set_spins must lie in the model's range (Ising +-1, Potts 0..q-1): the sums are taken
 * from byte-equality counts. */
int sw_observables(sw_ctx *c, double *host_E, double *host_M, double *host_M2, double *host_M4);

/* n SW steps with the observables of the configuration after EVERY step (the paper's measurement
 * loop): the per-step sums stay on the device and are
 * copied out once at the end, so there is no host round trip per step.  host_E .. host_M4 are HOST
 * arrays of n doubles each (any may be NULL) with the same meaning as in sw_observables.  Needs
 * n x (5 + q) x 8 bytes (clock: 5 + 2q) of library-owned device memory, allocated on first use, kept
 * with the context and grown when a larger n is asked for (SW_ENOMEM if that fails). */
int sw_run_series(sw_ctx *c, int n, double *host_E, double *host_M, double *host_M2, double *host_M4);

/* Destroy the context (synchronises its stream first).  NULL is a no-op. */
int sw_destroy(sw_ctx *c);

const char *sw_last_error(void);

/* ---- state accessors (parity tests, checkpoint/restore, end-to-end host buffers) ---------- */

/* Number of sites N = L^dim and index t of the next step. */
size_t sw_num_sites(const sw_ctx *c);
uint64_t sw_step_index(const sw_ctx *c);

/* Copy the configuration to / from a HOST buffer of exactly N elements: int8 (Ising, +-1),
 * uint8 (Potts, 0..q-1), float32 (XY angle in [0, 2 pi]) or uint16 (clock state 0..q-1).  sw_set_spins also sets the step
 * counter (state = (spins, seed, t), because the generator is counter-based).  Both synchronise.
 * Values outside the model's range are not checked. */
int sw_get_spins(sw_ctx *c, void *host_dst, size_t bytes);
int sw_set_spins(sw_ctx *c, const void *host_src, size_t bytes, uint64_t step);

/* Bond bytes (N) and cluster labels (N x uint32, label = minimum linear site index of the cluster)
 * of the LAST executed step; SW_ESTATE if no step ran since create / sw_set_spins.
 * The step itself keeps bonds on chip and labels as packed parent pointers in a tiled order, so
 *   - bond bytes exist only if recording was switched on BEFORE the step with
 *     sw_set_record_bonds(c, 1) (default off; the same kernels then also store one byte per site);
 *     otherwise sw_get_bonds returns SW_ESTATE;
 *   - sw_get_labels converts on request (an extra kernel and N x 4 bytes of scratch device memory
 *     that live only for the call; SW_ENOMEM if that allocation fails). */
int sw_set_record_bonds(sw_ctx *c, int enable);
int sw_get_bonds(sw_ctx *c, uint8_t *host_dst, size_t bytes);
int sw_get_labels(sw_ctx *c, uint32_t *host_dst, size_t bytes);

/* Cluster statistics of the LAST executed step's labelling (on request; scratch device memory of
 * N x 4 bytes for the call): number of clusters and sum over clusters of the squared cluster size.
 * For Ising and Potts <sum_c n_c^2> = <M^2> (the improved estimator of the Fortuin-Kasteleyn
 * representation; Potts with Eq. (5)'s normalisation).  Either pointer may be NULL. */
int sw_get_cluster_stats(sw_ctx *c, uint64_t *host_n_clusters, uint64_t *host_sum_nc2);

/* The same two sums for callers that must not allocate device memory (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc): no cudaMalloc / cudaFree, no allocating
 * library routine, no host synchronisation, no context.
 *   device_labels  DEVICE pointer, n uint32 canonical labels as sw_get_labels returns them: the label of
 *                  a site is the index (< n) of one site of its cluster, the same for all its sites
 *                  (a label >= n is skipped); read only, owned by the caller;
 *   n              number of sites, 1 .. SW_STATIC_MAX_SITES; anything else returns SW_EINVAL with the
 *                  limit in sw_last_error() and launches nothing;
 *   device_out     DEVICE pointer to two uint64, 8-byte aligned, owned by the caller: [0] = number of
 *                  clusters, [1] = sum_c n_c^2; written asynchronously on the stream;
 *   cuda_stream    cudaStream_t passed as void * (NULL = the legacy default stream) of the CURRENT device.
 * The per-site size counters (scratch) live in a static device array of SW_STATIC_MAX_SITES uint32
 * (4 MiB) inside the library, which every GPU that loads the library holds until the process exits.
 * All calls share that array and it keeps the last call's counters: every call clears the part it
 * uses first, and two calls that overlap on the GPU (different streams or threads) race -- order them
 * on one stream or with events. */
#define SW_STATIC_MAX_SITES (1u << 20)
int sw_cluster_stats_static(const uint32_t *device_labels, size_t n, uint64_t *device_out, void *cuda_stream);

/* Exact integer sums of the current configuration.  Ising: *host_E = -sum s_i s_j,
 * host_M_or_nk[0] = sum s_i (n >= 1).  Potts: *host_E = #unequal pairs, host_M_or_nk[k] = n_k for
 * k < min(n, q).  SW_EINVAL for XY. */
int sw_get_counts(sw_ctx *c, int64_t *host_E, int64_t *host_M_or_nk, int n);

/* Clock model (SW_CLOCK: the q-state clock discretisation of XY the paper's program runs, PAPER.md:88,
 * 159, 210; spins are uint16 states p = 0..q-1, theta = 2 pi p / q).  Exact integer histograms of the
 * current configuration: host_D[d] = number of nearest-neighbour pairs (i, i + e_k) with
 * (p_i - p_j) mod q = d, host_n[p] = number of sites in state p (q entries each, either may be NULL);
 * and the mirror index m (the paper's ispr) of the LAST step: the step reflects a cluster as
 * p -> (m - p) mod q. */
int sw_get_clock_hist(sw_ctx *c, int64_t *host_D, int64_t *host_n, int q);
int sw_get_clock_mirror(sw_ctx *c, int *host_m);

/* XY: direction r = (rx, ry) and reflection constant c = (2 phi + pi) mod 2 pi of the LAST step. */
int sw_get_xy_dir(sw_ctx *c, float *host_rx, float *host_ry, float *host_c);
/* XY test hook: use the angle phi for every following step instead of the Philox draw. */
int sw_force_xy_phi(sw_ctx *c, int enable, double phi);

/* Labelling counters of the LAST step (north_star: "labelling-iteration counts"); filled only
 * when the context was switched to counting mode with sw_set_counting(c, 1), which makes the
 * kernels slower.  out[0] = tile-face bond slots examined, out[1] = active ones (unions attempted),
 * out[2] = unions that linked two roots, out[3] = union retries (lost atomicCAS), out[4] = total
 * find hops in the merge, out[5] = max find hops of one union, out[6] = rounds of the root-chase
 * loop in the flip kernel summed over threads (a round advances up to 4 sites by one parent), out[7] =
 * the largest such sum of one thread (a thread owns sw_info(c, SW_INFO_FLIP_SITES_PER_THREAD) sites).
 * Lattices that run in one CTA (SW_INFO_ONE_CTA) have no merge and no chase kernel: all zero. */
int sw_set_counting(sw_ctx *c, int enable);
int sw_get_label_stats(sw_ctx *c, uint64_t *host_out, int n);

/* How a context runs: launch geometry chosen at create time (reported by bench.py). */
enum { SW_INFO_TILE_X = 0, SW_INFO_TILE_Y = 1, SW_INFO_TILE_Z = 2, SW_INFO_ROWS_PER_THREAD = 3,
       SW_INFO_FLIP_SITES_PER_THREAD = 4, SW_INFO_ONE_CTA = 5, SW_INFO_LAUNCHES_PER_STEP = 6,
       SW_INFO_OBSERVABLES_COPY_BYTES = 7 };
/* Returns the value, or -1 for a NULL context / unknown item.  SW_INFO_ONE_CTA = 1: lattices of at most
 * 32768 Ising / Potts sites run all n steps of sw_step(n) in ONE launch of one CTA (sw_small.cuh);
 * SW_INFO_LAUNCHES_PER_STEP is then 0 (one launch per call) and 3 otherwise.
 * SW_INFO_OBSERVABLES_COPY_BYTES: device-to-host bytes of one sw_observables call. */
long long sw_info(const sw_ctx *c, int item);

/* Per-kernel device times.  With timing enabled, sw_step brackets each of the three kernels of a
 * step (k_bond_label, k_merge, k_flip; one-CTA lattices: the whole launch in slot 0) with CUDA events on
 * the context's stream and synchronises after every step (a measurement mode, slower than the asynchronous default).
 * sw_get_kernel_times returns the accumulated milliseconds per kernel (host_ms[0..2]) and the number
 * of steps accumulated (*host_steps) since timing was enabled, then clears the accumulators. */
int sw_set_kernel_timing(sw_ctx *c, int enable);
int sw_get_kernel_times(sw_ctx *c, double *host_ms, int n, uint64_t *host_steps);

/* Philox4x32-10 exactly as the kernels compute it, evaluated on the device for `count` (counter,
 * key) pairs: host_ctr = count x 4 words, host_key = count x 2 words, host_out = count x 4 words.
 * Lets the tests pin the GPU generator to the known-answer vectors. */
int sw_philox_selftest(const uint32_t *host_ctr, const uint32_t *host_key, uint32_t *host_out, int count);

/* Micro-benchmarks behind the bounds DESIGN.md section 6 quotes (test / bench only; allocate and free
 * their own device memory, run on the legacy default stream, time `reps` launches with CUDA events after
 * one warm-up launch and return the mean milliseconds per launch in *host_ms):
 *   SW_MICRO_PHILOX_SITE   one Philox4x32-10 call and three threshold compares per site, one result byte
 *                          per site written (the per-site keying of XY / clock);
 *   SW_MICRO_PHILOX_GROUP  the transposed-digit decisions of one group of 32 sites per thread (10 calls,
 *                          13 digits x 3 directions; the Ising / Potts keying), three mask words written;
 *   SW_MICRO_GATHER        n dependent-free random 4-byte reads from a table of `table_words` words
 *                          (k_merge / k_flip chase pattern), one word written per read.
 * n = number of sites (PHILOX_*) or reads (GATHER). */
enum { SW_MICRO_PHILOX_SITE = 0, SW_MICRO_PHILOX_GROUP = 1, SW_MICRO_GATHER = 2 };
int sw_micro_bench(int kind, size_t n, size_t table_words, int reps, double *host_ms);

#ifdef __cplusplus
}
#endif
#endif
