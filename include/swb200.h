/*
 * swb200.h -- C-ABI of libswb200.so: Swendsen-Wang and Wolff cluster updates of the 2D nearest-neighbour
 * Ising / q-state Potts model on a periodic L x L square lattice, hand-written CUDA for sm_100a (B200).
 *
 * Method: M. Weigel, "Connected component identification and cluster update on GPU", arXiv:1105.5804.
 * "P:NN" = line NN of the paper text; "S:8x" = SURVEY.md section 8(x); DESIGN.md lists every
 * reading of the paper taken here.
 *
 * Conventions (S:8b, S:8c):
 *   - site i = y*L + x, x,y in [0,L); east(i) = (x+1 mod L, y); north(i) = (x, y+1 mod L)   (P:66 periodic
 *     square lattice; Fig. 1: site 0 bottom-left).
 *   - q = 2: Ising convention, spins int8 in {+1,-1} (state k=0 -> +1, k=1 -> -1), bond probability
 *     p = 1 - exp(-2 beta) (BASELINE.json configs), beta_c = ln(1+sqrt 2)/2.
 *     3 <= q <= 8: Potts delta convention (Eq. 1), spins uint8 in [0,q), p = 1 - exp(-beta).  J = 1.
 *   - random numbers: stateless Philox4x32-10, key = (seed low 32, seed high 32), counter
 *     (c0, t low 32, t high 32, domain) with domains INIT=0, BOND=1, FLIP=2, WSEED=3; t is the step counter,
 *     starting at 0 and increased by one per SW sweep or Wolff step (S:8c.2).  The paper's per-thread LCGs
 *      make results depend on the thread layout and are replaced (reading 5).
 *   - labels are canonical: labels[i] = the minimum site index of i's cluster (BASELINE.json north_star (3)).
 *   - packed bonds: byte b holds sites 4b..4b+3; site j uses bit 2(j&3) (east bond) and 2(j&3)+1 (north bond).
 *
 * Memory: every `d_` pointer is DEVICE memory owned by the caller (e.g. a torch tensor), 16-byte aligned, alive
 * for as long as it is bound.  The handle owns only host state and never frees caller memory.  `h_` pointers
 * are HOST memory.  `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  All
 * kernels are enqueued on that stream; a function is asynchronous unless it says "synchronises".
 *
 * Errors: every function returns SW_OK (0) or a negative code; nothing throws, aborts or prints.
 */
#ifndef SWB200_H
#define SWB200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    SW_OK      = 0,
    SW_EINVAL  = -1,  /* bad argument: L<4, L%4!=0, L>32768 (L>16384 for q>2), q outside [2,8], beta not finite or <0, NULL or
                         misaligned pointer, workspace too small, n<0                                      */
    SW_ESTATE  = -2,  /* handle not bound (sw_bind not called), or d_bonds needed but bound as NULL        */
    SW_ECUDA   = -3,  /* a CUDA runtime call or kernel launch failed; text via sw_strerror / sw_last_cuda_error */
    SW_ENOMEM  = -4,  /* host allocation failed                                                          */
    SW_ELIMIT  = -5   /* sw_cluster_stats_static: the lattice has more than SW_STATIC_MAX_SITES sites        */
};

typedef struct sw_handle sw_handle;   /* opaque; host-side state only */

/* Observables (S:8a a6, a9).  Spin part: Eq. 1.  Cluster part refers to the labelling performed by the
 * LAST sw_sweep / wolff_step / sw_label on this handle (reading 13); zero if none happened yet. */
typedef struct {
    int64_t  sat_bonds;        /* number of the 2N bonds whose end spins are equal                            */
    int64_t  energy;           /* q=2: -sum_<ij> s_i s_j = -(2 sat - 2N);  q>2: -sat  (Eq. 1 with J=1)    */
    int64_t  magnetisation;    /* q=2: sum_i s_i;  q>2: q * max_k n_k - N                                     */
    int64_t  state_count[8];   /* n_k = number of sites in state k, k < q                                     */
    int64_t  n_clusters;       /* #{ i : labels[i] == i }                                                     */
    int64_t  n_active_bonds;   /* bonds activated in the last sweep / step (0 after sw_label)                 */
    int64_t  max_cluster;      /* size of the largest cluster                                                 */
    uint64_t sum_sq_cluster;   /* sum over clusters of size^2 (FK estimator of N^2 <m^2>)                     */
    uint64_t counter;          /* step counter t after the last sweep / step                                  */
} sw_obs;

/* What the paper's own pipeline needed (sw_label_paper). */
typedef struct {
    int32_t selflabel_passes_max;   /* self-labelling passes of the slowest tile (n_B, Eq. 11)                   */
    int32_t relax_iterations;       /* label-relaxation iterations until nothing changed (n_relax, Eq. 13); 0 for sewing */
    int32_t sewing_levels;          /* levels of the hierarchical sewing (log2(L/B)); 0 for relaxation               */
    int32_t reserved;
    double  ms_local, ms_consolidate, ms_flatten;   /* CUDA-event times of the three phases                         */
    double  ms_wrap;                /* the part of ms_consolidate spent closing the 2L bonds that wrap around the lattice (sewing
                                       only, else 0).  The paper says only "in an additional step"; here it is ONE thread,
                                       like the last sewing level -- this repository's choice, reported so that ratios can be
                                       quoted with and without it                                                     */
} sw_paper_stats;

/* Cluster statistics of a canonical labelling (S:8a a9; BASELINE.json config 4 "cluster-size histogram"). */
typedef struct {
    int64_t  n_clusters;
    int64_t  max_cluster;
    uint64_t sum_sq_cluster;
    int64_t  hist32[32];       /* hist32[b] = number of clusters with 2^b <= size < 2^(b+1)                   */
} sw_cstats;

/* Create a handle for an L x L lattice of q-state spins at inverse temperature beta with RNG seed `seed`
 * (BASELINE.json north_star "sw_create(L,q,beta,seed)").  The bond threshold is T = floor((1-exp(-K beta)) 2^32)
 * in IEEE double on the host, K = 2 for q=2, K = 1 otherwise (S:8c.4); a bond between equal spins is activated
 * iff its 32-bit draw is < T (P:53 step 1, Eq. 7).  Requires 4 <= L <= 32768 (L <= 16384 if q > 2), L % 4 == 0,
 * 2 <= q <= 8, beta finite and >= 0.  The step counter starts at 0.  No device memory is allocated. */
int sw_create(sw_handle** out, int32_t L, int32_t q, double beta, uint64_t seed);
int sw_destroy(sw_handle* h);

/* The same update on the periodic L x L x L SIMPLE CUBIC lattice (S:8f row 2; "hypercubic lattices": a site
 * looks after "three out of six neighbours").  Site i = z L^2 + y L + x; it owns its bonds to the east (x+1), north (y+1)
 * and up (z+1) neighbour; N = L^3.  Bond draws (reading 19): n(i,d) = [s_i == s_nbr(i,d)] and
 * [PHILOX(seed; i, t, BOND3 = 4)[d] < T], d = 0 east, 1 north, 2 up -- one call per site.  Threshold, initialisation, flip
 * and label convention are the square lattice's (the 2N of sw_obs / sw_series_read becomes 3N).  Requires 4 <= L <= 1024
 * (N <= 2^30), L % 4 == 0, 2 <= q <= 8.  A cubic handle supports sw_bind (d_bonds: N bytes or NULL, workspace
 * sw_workspace_bytes3d), sw_init_spins, sw_sweep, sw_sweep_host, sw_activate (one byte per site: bit 0 east, 1 north, 2 up),
 * sw_label (bonds: one byte per site), sw_observables(_ex), sw_cluster_stats, sw_series_read, the threshold / counter / profile
 * calls; wolff_step, sw_wolff_frontier and sw_label_paper return SW_EINVAL.  sw_profile_read phases: 0 = k3_local, 1 = k3_faces, 2 = k3_final. */
int sw_create3d(sw_handle** out, int32_t L, int32_t q, double beta, uint64_t seed);
size_t sw_workspace_bytes3d(int32_t L, int32_t q);

/* Bytes of device workspace sw_bind needs for an L x L lattice (int32 strip-edge root arrays, int32 cluster-size scratch,
 * accumulators).  0 if L or q is invalid. */
size_t sw_workspace_bytes(int32_t L, int32_t q);

/* Bind caller-owned device buffers: d_spins N bytes (int8 for q=2, uint8 for q>2), d_labels N int32,
 * d_bonds N/4 bytes of packed bonds or NULL (only sw_activate and sw_label(d_bonds=NULL) need it),
 * d_work >= sw_workspace_bytes(L,q) bytes.  Zeroes the accumulators in d_work on `stream`: later calls on this
 * handle must be ordered after that memset -- use the same stream, or synchronise `stream` before the first call on
 * another one.  (An argument the proposed signature of S:8b does not have; DESIGN.md section 1 lists the deviations.)
 * The CUDA device the buffers live on is read from d_spins (cudaPointerGetAttributes; SW_EINVAL if it is not device memory);
 * every later call on the handle makes that device current for its own duration and restores the caller's, so a process
 * with several GPUs need not cudaSetDevice around the library. */
int sw_bind(sw_handle* h, void* d_spins, int32_t* d_labels, uint8_t* d_bonds, void* d_work, size_t work_bytes,
            void* stream);

/* Threshold override (percolation, BASELINE.json config 4; tests) and step-counter access (checkpoint /
 * resume: the whole state is (spins, t), S:5). */
int sw_set_threshold(sw_handle* h, uint32_t T);
int sw_get_threshold(const sw_handle* h, uint32_t* T);
int sw_set_counter(sw_handle* h, uint64_t t);
int sw_get_counter(const sw_handle* h, uint64_t* t);

/* Initialise d_spins (S:8c.8): mode 0 = cold (all k=0, i.e. +1 for q=2); mode 1 = random,
 * k_i = (PHILOX(seed; i>>2, 0, 0, INIT)[i&3] * q) >> 32.  Does not change the counter. */
int sw_init_spins(sw_handle* h, int mode, void* stream);

/* n Swendsen-Wang sweeps (P:51-55 steps 1-3), asynchronous; t += n.  Each sweep at counter t:
 *   1. bond activation (S:8c.3-4): n(i,d) = [s_i == s_nbr(i,d)] and [PHILOX(seed; i>>1, t, BOND)[2(i&1)+d] < T]
 *   2. labelling: d_labels[i] = min site index of i's connected component in the activated-bond graph
 *   3. flip: every cluster with root r takes state k_r = (PHILOX(seed; r, t, FLIP)[0] * q) >> 32 (P:55 step 3)
 * After return (and stream completion) d_spins holds the new configuration and d_labels the canonical labels of
 * the last sweep's bond graph. */
int sw_sweep(sw_handle* h, int64_t n, void* stream);

/* Write the packed bonds of step t (the current counter, not advanced) for the current spins into the bound
 * d_bonds ("bond array"; S:8a a1).  SW_ESTATE if d_bonds was bound as NULL. */
int sw_activate(sw_handle* h, void* stream);

/* Connected-component labelling of an arbitrary packed bond array on the L x L torus
 * (BASELINE.json north_star "sw_label(bonds->labels)"; P:54 step 2; config 4 percolation):
 * d_labels_out[i] = min site index of i's component.  d_bonds_in == NULL uses the bound d_bonds,
 * d_labels_out == NULL the bound d_labels.  Does not touch spins or the counter. */
int sw_label(sw_handle* h, const uint8_t* d_bonds_in, int32_t* d_labels_out, void* stream);

/* Cluster statistics of canonical labels (d_labels_in == NULL: the bound d_labels).  Synchronises `stream`. */
int sw_cluster_stats(sw_handle* h, const int32_t* d_labels_in, sw_cstats* h_out, void* stream);

/* Cluster statistics WITHOUT a workspace, for callers that cannot obtain device memory at the moment they need the numbers.
 * sw_cluster_stats needs a bound handle, i.e. a d_work of sw_workspace_bytes() that somebody had to allocate (4 bytes per site
 * of cluster-size scratch plus the strip arrays).  Some users of this library cannot do that: a measurement hook that runs
 * inside a simulation whose device memory is entirely handed out to a pool of fixed size (a raw cudaMalloc there fails, or
 * steals pages the pool expects to get back); a latency-critical loop, where cudaMalloc / cudaFree synchronise the whole
 * device; a plug-in that is handed two device pointers and nothing else.  For them the per-root size array and the
 * accumulators live in ONE array compiled into the library (`static __device__`, SW_STATIC_MAX_SITES int32 + 4 KiB,
 * about 4 MiB): every GPU that loads libswb200.so holds that much from the moment the library's module is loaded on it
 * until the process exits, whether or not this function is ever called.
 *   L        : L x L square lattice, 4 <= L, L % 4 == 0, L * L <= SW_STATIC_MAX_SITES (L <= 1024); a larger lattice is refused
 *              with SW_ELIMIT and nothing is launched (use sw_cluster_stats with a workspace).
 *   d_labels : DEVICE, N = L * L int32, 16-byte aligned, canonical labels (every value the index of a site, e.g. what
 *              sw_sweep / sw_label wrote); read only.
 *   d_out    : DEVICE, one sw_cstats, 8-byte aligned, on the same GPU as d_labels; overwritten.  Valid once `stream` has
 *              reached the end of the call's work; the call itself is asynchronous and copies nothing to the host.
 * The call allocates nothing: no cudaMalloc / cudaFree, no allocating library routine, no host heap.  It needs no handle.
 * The GPU d_labels lives on is made current for the duration of the call.  The FIRST call on each GPU also looks up the
 * device address of the array on that GPU (cudaGetSymbolAddress, once per device; the result is cached); make that first call
 * at set-up time, before any stream capture begins.
 * The array is shared by every call in the process and keeps whatever the previous call left, so each call first clears the
 * part it uses, on `stream`.  Two calls whose work overlaps on one GPU (different streams, or different host threads on different
 * streams) race on it and both results are garbage: order them on one stream or with events.  Calls on different GPUs do not
 * interact (each GPU has its own copy).
 * Errors: SW_EINVAL (NULL / misaligned pointer, bad L, a pointer that is not device memory, d_out on another GPU), SW_ELIMIT
 * (lattice larger than the array), SW_ECUDA (a runtime call or launch failed). */
#define SW_STATIC_MAX_SITES (1 << 20)
int sw_cluster_stats_static(int32_t L, const int32_t* d_labels, sw_cstats* d_out, void* stream);

/* ABLATION BASELINE (S:8f row 4): the same labelling as sw_label, computed the way the PAPER does it -- self-labelling on
 * B x B tiles in shared memory, then tile consolidation by label relaxation (method 0) or by
 * hierarchical sewing (method 1), then a flatten pass -- so that the cost of the paper's design on a B200 can be put
 * next to sw_label's.  Output: canonical labels (minimum site index), bit-identical to sw_label's.  B in {8, 16, 32}, L % B == 0,
 * and L / B a power of two for method 1; square lattice only; else SW_EINVAL.  d_bonds_in / d_labels_out as in sw_label.
 * Uses the cluster-size scratch of the workspace.  The number of active bonds is not counted: a following sw_observables reports
 * n_active_bonds = 0 (n_clusters is filled).  Synchronises `stream` (the relaxation's stopping criterion is read by the
 * host between launches, as in the paper).  h_stats may be NULL.  Not on the sweep path. */
int sw_label_paper(sw_handle* h, int method, int B, const uint8_t* d_bonds_in, int32_t* d_labels_out, sw_paper_stats* h_stats,
                   void* stream);

/* n Wolff single-cluster steps, q = 2 only (SW_EINVAL otherwise; reading 8); t += n.
 * Step at counter t (S:8c.9): seed site i0 = (PHILOX(seed; 0, t, WSEED)[0] * N) >> 32; C = component of i0 in the
 * bond graph of step t on the pre-step spins; s_i -> -s_i for i in C.  Realised as "decompose the whole lattice,
 * flip one cluster" (P:334 option (a)).  h_sizes: NULL, or a HOST array of n int64 that receives |C| of every
 * step -- in that case the call synchronises `stream` before returning. */
int wolff_step(sw_handle* h, int64_t n, int64_t* h_sizes, void* stream);

/* n steps of the FEW-CLUSTER variant (S:8f row 1), q = 2 on the square lattice only (SW_EINVAL otherwise); t += n.
 * The paper grows clusters from many seed sites at once and flips each with "a flipping probability p_flip < 1", and states
 * that this is "logically identical to performing the full SW decomposition and then selecting [...] points on the lattice,
 * followed by flipping all distinct clusters these points belong to"; that is what a step at counter t does (DESIGN.md
 * reading 21 fixes the draws): bonds and canonical labels as in sw_sweep; seed sites i_k = (PHILOX(seed; k, t, WSEED)[0] * N)
 * >> 32, k < n_seeds (k = 0 is wolff_step's seed); every cluster that holds a seed site is selected once; a selected cluster
 * with root r has all its spins negated iff PHILOX(seed; r, t, FLIP)[1] < T_flip, i.e. with probability T_flip / 2^32 < 1.
 * 0 <= n_seeds <= 65536, and the next power of two >= 2 n_seeds must not exceed N (the table of selected roots uses the
 * cluster-size scratch of the workspace).  d_labels holds the canonical labels of the last step's decomposition; the energy
 * series and the cluster part of sw_obs are maintained as by sw_sweep.  h_flipped: NULL, or a HOST array of n int64 that
 * receives the number of flipped sites of every step -- then the call synchronises `stream`. */
int sw_fewcluster_step(sw_handle* h, int64_t n, int32_t n_seeds, uint32_t T_flip, int64_t* h_flipped, void* stream);

/* Frontier growth for wolff_step (P:355 option (b); S:8f.1).  max_levels = 0 (default): every step decomposes the whole
 * lattice and flips one cluster.  max_levels > 0: a step first grows the cluster from the seed site level by level --
 * the bond draws are pure functions of (seed, t, site, direction), so it is the same cluster, and only the bonds that
 * are looked at are drawn; if the frontier is not empty after max_levels levels the spins are restored and the step is
 * done by the labelling path after all.  A level costs about 2 microseconds whatever its width, so this pays for small
 * clusters only (beta < beta_c; at beta_c the median Wolff cluster of a large lattice has ~10^5..10^6 sites).  In this
 * mode wolff_step maintains neither d_labels nor the energy series, and the cluster part of sw_obs is zero. */
int sw_wolff_frontier(sw_handle* h, int max_levels);

/* Energy, magnetisation, state counts of the current spins and cluster statistics of the last labelling, all in
 * int64 (S:8a a6).  Synchronises `stream`.  Equals sw_observables_ex(.., SW_OBS_SPINS | SW_OBS_CLUSTERS, ..). */
int sw_observables(sw_handle* h, sw_obs* h_out, void* stream);

/* The same with a choice of what is computed (fields not asked for are 0):
 *   SW_OBS_SPINS    sat_bonds, energy, magnetisation, state_count: one read of the spins (Eq. 1)
 *   SW_OBS_CLUSTERS max_cluster, sum_sq_cluster: one pass over the labels buffer the last labelling wrote (for a
 *                   sw_label into a caller buffer that buffer must still be alive)
 * n_clusters, n_active_bonds and counter are always reported (the labelling counts them itself).  flags = 0 is
 * valid: it only reads the counters back.  Synchronises `stream`. */
enum { SW_OBS_SPINS = 1, SW_OBS_CLUSTERS = 2 };
int sw_observables_ex(sw_handle* h, sw_obs* h_out, int flags, void* stream);

/* Energy and magnetisation of every configuration a chain passes through, at no extra pass over the spins (S:8a a6;
 * BASELINE.json north_star (5) "a fused energy/magnetisation reduction"): the sweep's scan kernel reads every spin and
 * its two neighbours anyway, so it counts the satisfied bonds and the minus spins of the configuration the sweep (or
 * Wolff step) STARTS from.  The totals of the last 4096 consecutive sweeps / steps are kept on the device, filed under
 * the step counter t the configuration belongs to (t = the number of sweeps / steps performed before it).
 * sw_series_read copies n of them, counters t_first .. t_first + n - 1, to the host: energy as in sw_obs; magnetisation
 * = sum_i s_i for q = 2 (h_magnetisation must be NULL for q > 2: state counts are not recorded on the sweep path).
 * SW_EINVAL if a requested counter is not (or no longer) recorded: only counters of sweeps already performed are --
 * the CURRENT configuration has not been scanned yet (use sw_observables_ex for it).  Synchronises `stream`. */
int sw_series_read(sw_handle* h, uint64_t t_first, int64_t n, int64_t* h_energy, int64_t* h_magnetisation, void* stream);

/* Host-buffer convenience for end-to-end use: copy h_spins_in (N bytes, may be NULL to keep the device state)
 * to the device, run n sweeps, copy spins back to h_spins_out (may be NULL) and labels to h_labels_out (may be
 * NULL), fill h_obs (may be NULL).  Synchronises `stream`. */
int sw_sweep_host(sw_handle* h, const void* h_spins_in, int64_t n, void* h_spins_out, int32_t* h_labels_out,
                  sw_obs* h_obs, void* stream);
/* The same with the parts of h_obs chosen as in sw_observables_ex (SW_OBS_SPINS alone skips the cluster-size pass, 2 ms at
 * L = 16384: energy, magnetisation, state counts, n_clusters and n_active_bonds are still filled). */
int sw_sweep_host_ex(sw_handle* h, const void* h_spins_in, int64_t n, void* h_spins_out, int32_t* h_labels_out,
                     sw_obs* h_obs, int obs_flags, void* stream);

/* MULTI-GPU ROW BANDS (S:8e, S:8f row 3; the paper proposes label relaxation between GPUs over MPI).  G processes, one
 * GPU each, create the SAME lattice (same L, q, beta, seed, full-size buffers) and call sw_set_band(h, rank, G): the handle
 * then works on the strip rows of band `rank` only (L % 32 == 0 and (L / 32) % G == 0; square lattice; SW_EINVAL otherwise;
 * G = 1 restores the whole lattice).  One sweep of a banded handle:
 *   1. the caller copies the spins of row y_halo (sw_band_layout) from the rank that owns it into the same row of d_spins;
 *   2. sw_sweep_band_begin: activation + labelling of the band, seams inside the band, then the strip-local roots on the band's
 *      two outer rows are replaced by the band's roots: L int32 rootN (last row; -1 where the north bond is inactive) at byte
 *      offset work_off_rootN of d_work and L int32 rootS (first row) at work_off_rootS;
 *   3. the caller all-gathers these two rows: the rows of band b of EVERY rank go to sw_band_layout(h, b, ...)'s offsets of
 *      its own d_work (128 KiB per rank and sweep at L = 16384);
 *   4. sw_sweep_band_end: every rank unites the G cross-band seams (redundantly, on its own full-size labels array), then
 *      flattens and flips its band; t += 1.  d_labels / d_spins are valid in the band's rows [y_first, y_first + n_rows).
 * The result is bit-identical to sw_sweep on one GPU (site indices, Philox counters and labels are global).  sw_band_counters
 * returns this band's share of (active bonds, clusters, satisfied bonds and minus spins of the configuration the sweep
 * started from): the caller sums them over the ranks.  sw_sweep, sw_sweep_host, sw_label, sw_activate, wolff_step,
 * sw_observables(_ex) and sw_cluster_stats on the bound labels return SW_ESTATE on a banded handle (it holds its band's rows only).
 * All asynchronous on `stream` except sw_band_counters, which synchronises. */
int sw_set_band(sw_handle* h, int rank, int nranks);
int sw_band_layout(const sw_handle* h, int band, int32_t* y_first, int32_t* n_rows, int32_t* y_halo,
                   size_t* work_off_rootN, size_t* work_off_rootS);
int sw_sweep_band_begin(sw_handle* h, void* stream);
int sw_sweep_band_end(sw_handle* h, void* stream);
int sw_band_counters(sw_handle* h, int64_t h_out[4], void* stream);

/* Per-kernel timing of sw_sweep / sw_label with CUDA events on the launching stream (for roofline reporting; off by
 * default, and the un-instrumented path records no events).  While enabled, each sweep records SW_NPHASE+1
 * events; at most 512 sweeps are kept between reads (further sweeps run untimed).  sw_profile_read synchronises
 * the recorded events, ADDS the elapsed milliseconds of each phase to ms[] and the number of timed sweeps to
 * *n_sweeps, and clears the record.  Phases: 0 = k_scan (activation + strip-local labelling), 1 = k_seam
 * (cross-strip union-find), 2 = k_final (flatten + flip). */
#define SW_NPHASE 3
int sw_profile_enable(sw_handle* h, int on);
int sw_profile_read(sw_handle* h, double ms[SW_NPHASE], uint64_t* n_sweeps);

/* Number of kernels this handle has launched so far (for bench.py's gpu_launches). */
int sw_launch_count(const sw_handle* h, uint64_t* n);

const char* sw_strerror(int code);
/* Text of the last CUDA error seen by this handle ("" if none). */
const char* sw_last_cuda_error(const sw_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* SWB200_H */
