/*
 * include/ic.h -- C ABI of the B200 coupled-pair Metropolis library (libic_b200.so).
 *
 * Hot path of arXiv:2301.11735 (Budrin, Ulitko, Chikov, Panov, Moskvin): the charge-conserving parallel
 * Metropolis sweep with "coupled pairs" (sec. 3.1) on an L x L periodic square lattice of
 * 4-state sites, followed by the per-sweep reductions that feed C(T) and chi(T) (sec. 2.2).
 * All arithmetic of the path runs in hand-written sm_100a CUDA kernels; the host side of the library only
 * validates arguments, builds the acceptance-threshold tables and the O(1) schedule parameters, and launches.
 *
 * Conventions
 *   - plain C, no exceptions; every entry point returns IC_OK (0) or a negative IC_ERR_* code.  Argument errors
 *     (NULL, SIZE, PARAM, WORKSPACE, CHARGE) are detected before anything is touched and leave the context
 *     unchanged.  After IC_ERR_CUDA (a launch or copy failed mid-call) the lattices and the sweep counter are
 *     undefined: the context is only good for ic_destroy.  ic_strerror() gives the text (for IC_ERR_CUDA the
 *     CUDA message).
 *   - pointers named h_* are HOST memory, d_* are DEVICE memory; both stay owned by the caller.  The
 *     library never allocates device memory: everything it keeps on the device lives inside the
 *     caller-provided workspace (a torch tensor in the Python binding).
 *   - site code c (public, in ic_set_state / ic_state):   0 -> sigma=+1 (s=+1/2),  1 -> sigma=-1,
 *     2 -> S=+1,  3 -> S=-1   (S=+-1 charge states, S=0 with s=+-1/2 magnetic states,
 *     sigma = 2(1-S^2)s).  Lattices are row-major, code[y*L + x], periodic in x and y.
 *   - exact integers of a lattice: n2 = sum S_i^2, bV = sum_<ij> S_i S_j, bJ = sum_<ij> sigma_i sigma_j
 *     (each site contributes its +x and +y bond), so that eq. (3) reads
 *     E = Delta*n2 + V*bV + (J/4)*bJ;  M = sum sigma_i, Ms = sum (-1)^(x+y) sigma_i, Q = sum S_i.
 *   - the constraint of eq. (2), sum_i S_i = Q = llround(n*N), holds after every pair update.
 *   - all launches and copies go to the CUDA stream given to ic_create.  ic_sweep is asynchronous;
 *     ic_set_state, ic_init_charges, ic_observables, ic_state, ic_debug_recompute, ic_largest_cluster and
 *     ic_snapshot_ppm synchronise that stream (ic_thresholds and ic_schedule are host-only).  Every call that takes
 *     a context and touches the device makes the device the context was created on current for the calling thread (and
 *     leaves it current); ic_destroy and the host-only getters do not change the current device.
 *   - one context must not be used from two host threads at once.
 */
#ifndef IC_H
#define IC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ic_ctx ic_ctx; /* opaque; owned by the library from ic_create to ic_destroy */

enum {
  IC_OK = 0,
  IC_ERR_NULL = -1,      /* a required pointer is NULL                                                */
  IC_ERR_SIZE = -2,      /* L not a power of two or L < 4 or L > 65536, replicas < 1, bits not 8 or 2,
                            replica index out of range                                                */
  IC_ERR_PARAM = -3,     /* |n| > 1, NaN/inf parameter, T <= 0, nsweeps < 0, sweep counter >= 2^31     */
  IC_ERR_WORKSPACE = -4, /* workspace NULL, smaller than ic_workspace_bytes(), or not 256-B aligned   */
  IC_ERR_CHARGE = -5,    /* ic_set_state: a code outside 0..3 or sum S != Q; ic_init_charges: bad counts */
  IC_ERR_CUDA = -6,      /* a CUDA call failed; ic_strerror(IC_ERR_CUDA) returns its message          */
  IC_ERR_STATIC_MAX = -7 /* ic_largest_cluster_static only: L > IC_STATIC_CLUSTER_MAX_L, the lattice does not
                            fit the scratch array built into the library                              */
};

/* Filled by ic_observables, one per replica (host memory, caller-owned).
 * C and chi follow PAPER.md:51 with k_B = 1:  C = (<E^2> - <E>^2) / (N T^2); the paper names chi(T)
 * (Fig. 6) without a formula, reading G9: chi_u = (<M^2> - <M>^2) / (N T) and
 * chi_s the same with Ms.  Averages are sums / nmeas. */
typedef struct {
  int64_t nmeas;                  /* sweeps accumulated since create / ic_reset_observables          */
  int64_t n2, bV, bJ, M, Ms, Q;   /* exact integers of the current lattice                           */
  double sumE, sumE2, sumM, sumM2, sumAbsM, sumMs, sumMs2, sumAbsMs; /* fp64, added once per sweep   */
  double T, C, chi_u, chi_s;      /* derived with the T given to the last ic_sweep call (0 if none)  */
} ic_obs;

/* Number of acceptance classes per temperature: index = ((dn2/2+1)*33 + (dV+16))*33 + (dJ+16) with
 * dn2 in {-2,0,2}, dV and dJ in [-16,16] (E_Delta, E_V, E_J of eq. 4/5).            */
#define IC_N_CLASSES 3267

/* Bytes of device memory ic_create needs for (L, replicas, bits_per_site); 0 if the arguments are invalid. */
size_t ic_workspace_bytes(int L, int replicas, int bits_per_site);

/* Creates a context for `replicas` independent copies of an L x L lattice (several copies
 * processed in parallel) with parameters Delta, V, J of eq. (1)/(3), charge density n
 * (eq. 2: Q = llround(n*L*L)) and Philox key `seed`.  Every replica r is initialised by stage 1
 * (PAPER.md:59-62): random sigma on all sites, then |Q| distinct random sites set to S = sign(Q), drawn
 * from the counter-based stream (seed, replica r) -- DESIGN.md "U0".  bits_per_site: 8 (one byte per site)
 * or 2 (16 sites per 32-bit word) in device memory.
 * d_workspace: device memory, >= ic_workspace_bytes() bytes, 256-B aligned, owned by the caller and kept
 * alive until ic_destroy.  cuda_stream: a cudaStream_t (NULL = default stream).                      */
int ic_create(ic_ctx** out, int L, double n, double delta, double V, double J, uint64_t seed, int replicas,
              int bits_per_site, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/* Re-runs stage 1 for one replica with nplus sites S=+1 and nminus sites S=-1 (nplus - nminus must equal Q,
 * nplus + nminus <= N); used for neutral lattices with charges of both signs (BASELINE config 3).    */
int ic_init_charges(ic_ctx* ctx, int replica, int64_t nplus, int64_t nminus);

/* Replaces the lattice of one replica by h_codes[L*L] (public codes, row-major, HOST memory) after checking
 * every code and sum S == Q; recomputes the replica's exact integers on the device.                   */
int ic_set_state(ic_ctx* ctx, int replica, const int8_t* h_codes);

/* Runs nsweeps sweeps on all replicas, replica r at temperature h_T[r] (HOST array of `replicas` doubles,
 * read before the call returns).  One sweep = N/2 coupled-pair updates in two conflict-free phases in which
 * every site belongs to exactly one pair (schedule S1 of DESIGN.md; PAPER.md:108-125 requires only that
 * concurrently updated pairs do not interact).  A pair update is PAPER.md:64-98: q = S_a + S_b, new pair
 * configuration drawn from the table of configurations with the same q, dE from eq. (4)/(5), accepted with
 * min(1, exp(-dE/T)) as an integer comparison with a host-built threshold.  After each sweep E, E^2, M, ...
 * are accumulated.  The sweep counter is global: ic_sweep(T,100) == ic_sweep(T,50) twice.
 * Asynchronous on the context's stream.                                                              */
int ic_sweep(ic_ctx* ctx, const double* h_T, int64_t nsweeps);

/* Same, and writes (n2,bV,bJ,M,Ms,Q) after every sweep to d_trace[s][r][6] (DEVICE memory, int64,
 * nsweeps*replicas*6 entries, caller-owned).                                                         */
int ic_sweep_trace(ic_ctx* ctx, const double* h_T, int64_t nsweeps, int64_t* d_trace);

int ic_reset_observables(ic_ctx* ctx);            /* zeroes nmeas and the fp64 sums (not the lattice)  */
int ic_observables(ic_ctx* ctx, ic_obs* h_out);   /* h_out[replicas], HOST; synchronises the stream    */
int ic_state(ic_ctx* ctx, int replica, int8_t* h_codes_out); /* L*L public codes, HOST; synchronises   */

/* The same two calls with the lattice at 2 bits per site on the host side too (a site has four states;
 * BASELINE north_star: "lattice packed at 2 bits or 1 byte per site"): h_words[L*L/16] (HOST), word i holds the sites
 * 16 i .. 16 i + 15 of the row-major lattice, the public code of site k of the word in bits 2k and 2k+1.  A quarter of the
 * bytes cross PCIe; checking (sum S == Q -- every 2-bit pattern is a valid code) and conversion to and from the context's
 * layout run on the device.  Any bits_per_site.  Both synchronise the stream.  A rejected lattice (IC_ERR_CHARGE) leaves
 * the replica untouched.                                                                                                  */
int ic_set_state_packed(ic_ctx* ctx, int replica, const uint32_t* h_words);
int ic_state_packed(ic_ctx* ctx, int replica, uint32_t* h_words_out);

/* Resume.  The lattices, the global sweep counter and the seed determine every later pair update (the random stream is
 * keyed by (seed, replica, sweep, slot)); nmeas and the fp64 sums carry the averages of PAPER.md:49-53 across the break.
 * To save a run: ic_state of every replica, ic_sweep_count, ic_observables.  To continue it: ic_create with the same L, n,
 * Delta, V, J, seed, replicas (bits_per_site and the kernel variant are free), ic_set_state for every replica, then
 * ic_restore(ctx, saved sweep count, saved ic_obs[replicas]): sets the sweep counter and, per replica, nmeas and the eight
 * sums from h_in (HOST); the exact integers in h_in are ignored -- ic_set_state has recomputed them from the lattice.  The
 * continued run is then bit-identical to the uninterrupted one (lattices, integers, sums).  Synchronises the stream.
 * IC_ERR_PARAM: sweep_count outside [0, 2^31), nmeas < 0, a sum that is not finite.                                      */
int ic_restore(ic_ctx* ctx, int64_t sweep_count, const ic_obs* h_in);

/* Full recomputation of (n2,bV,bJ,M,Ms,Q) from the lattice by a device reduction, straight from eq. (3);
 * out6 is HOST memory.  Must equal the incrementally tracked integers at any time.                    */
int ic_debug_recompute(ic_ctx* ctx, int replica, int64_t* out6);

/* The acceptance-threshold table the device uses for temperature T: h_out[IC_N_CLASSES] (HOST).  Entry
 * t29 in [1, 2^29]: a move with 32-bit random word w is accepted iff (w >> 3) < t29, t29 = 2^29 for dE <= 0
 * else clamp(floor(exp(-dE/T) * 2^29), 1, 2^29 - 1), dE = (Delta*dn2 + V*dV) + (J/4)*dJ in IEEE fp64. */
int ic_thresholds(ic_ctx* ctx, double T, uint32_t* h_out);

/* Schedule parameters of sweep `sweep` as the device will use them: out4 = {0, mx, my, 0} for a FAR sweep
 * (partner(x,y) = (x^mx, y^my)), {1, orientation, offset, 0} for a NEAR sweep (dominoes).  HOST.      */
int ic_schedule(ic_ctx* ctx, uint64_t sweep, int32_t* out4);

int64_t ic_sweep_count(const ic_ctx* ctx);        /* global sweep counter; -1 if ctx is NULL           */
int64_t ic_charge(const ic_ctx* ctx);             /* Q = llround(n*N); 0 if ctx is NULL                */

/* ---- maps: the paper's own parallel schedule (sec. 3.2) as an alternative to ic_sweep ----------------
 * A "map" is a randomly generated list of coupled pairs that do not interact: no site of one pair equals or neighbours a
 * site of another (Fig. 1), so all pairs of a map are updated in parallel, one thread each, the
 * same map for every lattice copy.  The paper builds maps of N/10 pairs sequentially on the CPU
 * and ships them over PCIe; here every map is built on the device in one round: K candidate pairs of
 * two distinct uniformly random sites (counter-based stream keyed by the seed and the map index); candidate k is kept iff
 * no candidate of lower index has a site inside its covering (its two sites and their nearest neighbours).
 * ic_sweep_maps runs nmaps maps; after each map ("step" of PAPER.md:167) E, E^2, ... are accumulated as after a sweep and,
 * if d_trace is not NULL, (n2,bV,bJ,M,Ms,Q) are written to d_trace[m][r][6] (DEVICE).  The map index is the context's
 * sweep counter, which advances by one per map.  d_scratch: DEVICE memory of ic_maps_scratch_bytes(L, K) bytes, 256-B
 * aligned, caller-owned, free to reuse after the call's work has finished on the stream.  L <= 32768.
 * Errors: IC_ERR_SIZE (K < 1, L too large), IC_ERR_PARAM (T, nmaps), IC_ERR_WORKSPACE.                                   */
size_t ic_maps_scratch_bytes(int L, int64_t K);
int ic_sweep_maps(ic_ctx* ctx, const double* h_T, int64_t nmaps, int64_t K, void* d_scratch, size_t scratch_bytes,
                  int64_t* d_trace);

/* ---- the "drop" (Fig. 7: with J >> V the whole charge gathers in one place) --------------------------
 * ic_largest_cluster: h_out2 = (size of the largest connected cluster of charged sites, number of clusters) of one
 * replica; 4-neighbour connectivity, periodic; which = 0: sites with S != 0, 1: S = +1, 2: S = -1.  d_scratch: DEVICE
 * memory of ic_cluster_scratch_bytes(L) bytes, 256-B aligned.  Synchronises the stream.  L <= 32768.
 * ic_snapshot_ppm: writes the replica's lattice as a binary PPM image (one pixel per site: S=+1 red, S=-1 blue,
 * sigma=+1 white, sigma=-1 grey) from host memory to `path`; IC_ERR_PARAM if the file cannot be opened.                   */
size_t ic_cluster_scratch_bytes(int L);
int ic_largest_cluster(ic_ctx* ctx, int replica, int which, void* d_scratch, size_t scratch_bytes, int64_t* h_out2);
int ic_snapshot_ppm(ic_ctx* ctx, int replica, const char* path);

/* ---- the same cluster count for callers that have no device memory to give -------------------------------------------
 * ic_largest_cluster needs 8 bytes of device scratch per site (union-find parents and cluster sizes) and every other
 * call of this library needs a workspace, all of it allocated by the caller.  Some callers cannot allocate when they want
 * the size of the drop: an analysis hook that runs inside another program's time step after that
 * program has handed the whole HBM to its own pool; a plug-in whose host forbids cudaMalloc / cudaFree in its steady
 * state because both wait for the whole device and stall every other stream; a monitor that must stay inside a fixed
 * memory budget.  For them this ONE entry point works without a context, a workspace or a scratch argument: its scratch is
 * an array compiled into the library (8 MiB of device memory per GPU, held by every GPU that loads the library from the
 * first CUDA call of the process on that GPU until the process exits, whether or not this call is ever made).
 *
 *   d_codes   DEVICE, L*L public site codes (0..3 as in ic_set_state / ic_state; one byte per site, row-major), read only;
 *             codes are taken modulo 4.  L a power of two, 4 <= L <= IC_STATIC_CLUSTER_MAX_L.
 *   which     0: sites with S != 0, 1: S = +1, 2: S = -1 (as in ic_largest_cluster; 4-neighbour, periodic).
 *   d_out2    DEVICE, two int64 written by the call: (size of the largest cluster, number of clusters).
 *   stream    a cudaStream_t (NULL = default stream) of the calling thread's CURRENT device; d_codes and d_out2 must be
 *             memory of that device.  The call only enqueues four kernels and returns; synchronise the stream (or order
 *             later work on it) before reading d_out2.  Both buffers stay owned by the caller.
 *
 * It calls no cudaMalloc, cudaFree or any library routine that allocates.  The first call on each device (with that
 * device current) looks up the device address of the built-in array with cudaGetSymbolAddress and keeps it; make that
 * first call at start-up, before any stream capture begins in the process.  Later calls only launch.
 * All calls on one GPU share the one array, and it keeps what the previous call left there: every call rewrites the part
 * it uses before reading it (nothing has to be cleared by the caller), but two calls whose kernels can overlap on the
 * GPU -- different streams, different host threads, different contexts of one process -- race on it and give garbage.
 * Put them on one stream or order them with events.
 * Errors (nothing is launched): IC_ERR_NULL (d_codes or d_out2 NULL), IC_ERR_SIZE (L < 4 or not a power of two),
 * IC_ERR_STATIC_MAX (L > IC_STATIC_CLUSTER_MAX_L: the lattice does not fit the built-in array; use ic_largest_cluster
 * with scratch of your own), IC_ERR_PARAM (which outside 0..2), IC_ERR_CUDA.                                              */
#define IC_STATIC_CLUSTER_MAX_L 1024
int ic_largest_cluster_static(const int8_t* d_codes, int L, int which, int64_t* d_out2, void* cuda_stream);

/* Kernel selection: 0 = automatic (default), 1 = reference kernels (one thread per pair, global memory),
 * 2 = tiled kernels (8 bits/site, 64 <= L <= 2048: vectors loaded straight from global memory), 3 = staged kernels
 * (8 or 2 bits/site, L >= 2048: tiles staged in shared memory by TMA bulk copies; the default there).
 * 4 = resident kernel (L <= 64, any bits_per_site: one block per replica keeps its lattice in shared memory and
 * runs all sweeps of an ic_sweep call in one launch, one thread per pair; the default for L < 16).
 * 6 = resident kernel with four-pair items (16 <= L <= 64, any bits_per_site: the same, with the item code of the staged
 * kernels on a byte lattice in shared memory; the default there).
 * 5 = one-launch kernel (8 or 2 bits/site, 128 <= L <= 1024: one cooperative launch runs
 * all sweeps of an ic_sweep call on the whole GPU, the phases separated by a barrier over the replica's blocks; the
 * default there).
 * IC_ERR_PARAM if the variant cannot run this context's (L, bits_per_site).  All variants produce identical
 * lattices and observables.                                                                           */
int ic_set_variant(ic_ctx* ctx, int variant);

/* The kernel family the last ic_sweep / ic_sweep_trace call of this context ran, in the numbering of ic_set_variant (1..6);
 * 0 before the first sweep, -1 if ctx is NULL.  With automatic selection this is how a caller (and the tests) see which
 * kernels did the work, e.g. that a cooperative launch that did not fit the GPU partition fell back to the phase kernels.  */
int ic_kernel_family(const ic_ctx* ctx);

/* Upper bound on the thread blocks per replica of the persistent kernels (variants 2, 3, 5); 0 = automatic (one block per
 * SM divided among the replicas).  Results do not depend on it: the tests run the kernels at several bounds (1, 2, 3, ...)
 * so that every block walks many tasks and ring laps and the task-to-block assignment changes -- the race check this
 * library can offer where no sanitizer is available.  IC_ERR_PARAM if max_blocks < 0.                */
int ic_set_max_blocks(ic_ctx* ctx, int max_blocks);

/* Number of kernels launched by this context since ic_create (for bench.py's gpu_launches).         */
int64_t ic_launch_count(const ic_ctx* ctx);

int ic_destroy(ic_ctx* ctx);
const char* ic_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* IC_H */
