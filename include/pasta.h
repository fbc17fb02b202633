/*
 * pasta.h -- C ABI of the B200 (sm_100a) nuclear-pasta molecular-dynamics hot path.
 *
 * The library computes, entirely in hand-written CUDA kernels on ONE GPU, the per-step two-body
 * force/energy evaluation, the counting-sort cell list that feeds it, the fused velocity-Verlet /
 * isokinetic-rescale / uniform box-scaling update around it, and the friends-of-friends cluster
 * labelling of the final configuration, of the semiclassical model of Caplan, Schneider, Horowitz
 * & Berry, "Pasta Nucleosynthesis", arXiv:1412.8502.  Citations below are "PAPER.md:<line>" (the
 * text of the paper) and "D<n>" (a reading of an ambiguous point, listed in DESIGN.md).
 *
 * Conventions
 *  - Units: lengths fm, times fm/c, energies and temperature MeV, velocities c, forces MeV/fm.
 *  - Every function returns 0 (PASTA_OK) or a negative pasta_status; no exception crosses the ABI;
 *    the text of the last error on the calling thread is pasta_last_error().
 *  - "_dev" pointers are device pointers on the simulation's device, "_host" pointers are host
 *    pointers.  The CALLER owns every buffer it passes; the library keeps no reference to them
 *    after the call returns.  Internal buffers come from pasta_env.alloc (the Python binding hands
 *    out torch CUDA tensors) or, if alloc is NULL, from cudaMalloc.
 *  - All work is enqueued on pasta_env.stream and is stream-ordered.  A call that writes a scalar to
 *    a "_host" pointer synchronises that stream before it returns; all other calls are asynchronous.
 *  - Arrays are row-major: x, v, F are [N][3] doubles; is_proton is [N] bytes (1 = proton).
 *  - There is no CPU fallback: without a usable CUDA device pasta_create fails with PASTA_ECUDA.
 */
#ifndef PASTA_H_
#define PASTA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum pasta_status {
  PASTA_OK = 0,
  PASTA_EINVAL = -1, /* bad argument (see each function) */
  PASTA_ECUDA = -2,  /* CUDA runtime / launch failure; text in pasta_last_error() */
  PASTA_ENOMEM = -3, /* pasta_env.alloc / cudaMalloc returned NULL */
  PASTA_ESTATE = -4  /* call order violated (e.g. pasta_cluster_sizes before pasta_clusters) */
} pasta_status;

/*
 * Model and algorithm parameters (POD, versioned by struct_size = sizeof(pasta_params)).
 * pasta_params_default() fills the paper's values.
 */
typedef struct pasta_params {
  uint32_t struct_size;
  uint32_t reserved0;
  double a, b, c, Lambda;      /* Table I: 110, -26, 24 MeV; 1.25 fm^2 (Eq. 1a-c, :75-82) */
  double alpha_hbarc;          /* alpha*hbar*c = 1.44 MeV fm of the screened Coulomb term (Eq. 1c, :81; D4) */
  double lambda;               /* screening length, fixed to 10 fm (D5) */
  double r_c;                  /* single cut-off for every term of Eq. 1: a pair interacts iff r < r_c (D1, D2) */
  double mass;                 /* nucleon mass M = 939 MeV */
  double scale_per_step;       /* s: each pasta_step multiplies L and x by s in the drift (D9, D10); 1 = fixed box */
  int32_t thermostat_interval; /* rescale |v| so that KE = 3/2 N T after every k-th step (D7, D8); 0 = off */
  int32_t cell_subdiv;         /* k >= 1 of the grid pasta_cells reports: cells per side = max(1, floor(L k / r_c)),
                                  width L/ncell >= r_c/k (D14).  (The force path sizes its own per-species grids with the
                                  same formula: pasta_force_grid / pasta_force_cells.) */
  int32_t energy_every_step;   /* 1 (default): pasta_step evaluates per-particle energies with the forces */
  int32_t skip_exact_zeros;    /* 1 (default): np/nn candidates beyond the distance at which exp2(-r^2 log2e/2 Lambda)
                                  underflows FP32 (14.78 fm for Lambda = 1.25) are not streamed: their terms are exactly
                                  0.0f in the kernel's arithmetic, so F and e are unchanged (D23).  0: stream to r_c */
  int32_t list_reuse;          /* 1 (default): where both species are sparse the sorted order and, for EVERY TARGET, the list
                                  of sorted source slots within reach + halo (skin) are built once and kept across steps
                                  until some particle has moved more than half the halo -- the paper's neighbour list with
                                  its displacement trigger.  F and e do not depend on it (to FP32
                                  summation order).  0: rebuild the cell list every step */
  double list_halo;            /* halo thickness delta_r in fm (PAPER.md:126 uses 4 fm); 0 = library default (6 fm) */
  double r_nuc;                /* > 0: the paper's own range split: the nuclear (Gaussian) terms are zero
                                  and not computed beyond r_nuc (11.5 fm in the paper) while the Coulomb term still reaches
                                  r_c.  0 (default): one cut-off r_c for every term (D1).  Must be <= r_c */
  double xi_dot;               /* > 0: the paper's own expansion (Eq. 3a; D25): after the drift of every step
                                  the box side becomes L0 (1 + xi_dot dt n), n = steps since create / set_state / expand and
                                  L0 the side at that moment; positions and velocities are NOT scaled.  Needs
                                  scale_per_step == 1 and a constant dt.  0 (default): off */
  int32_t coulomb_all_pairs;   /* 1: the Coulomb half of the paper's range split ("we do not use a cutoff radius
                                  for the Coulomb potential ... each proton interacts with the nearest periodic image of
                                  every other proton"): the screened Coulomb term is summed over ALL proton pairs at their
                                  nearest image (a cube of side L, no radial cut-off; N_p^2 pair terms by a kernel of its
                                  own) and the nuclear terms stop at r_nuc, which must be set; r_c then only sizes the
                                  cell list.  0 (default): the Coulomb term lives inside r_c like every other (D1).
                                  Needs a box side L >= PASTA_COULOMB_ALL_PAIRS_MIN_L (120 fm) at all times -- create,
                                  set_state*, expand and a scaling step return PASTA_EINVAL below it.  Why: the image of
                                  a pair is chosen on the FP32 leading parts of the box fractions x/L, so a pair within
                                  6e-8 L of L/2 along an axis can take the other image, which changes its two forces by
                                  2 F_c(L/2): 7e-6 MeV/fm at 120 fm (below the 1e-5 parity gate, and that is the range
                                  the mode is verified in against the oracle), but 1e-3 at 55 fm (reading D26) */
  int32_t reserved1;
} pasta_params;

#define PASTA_COULOMB_ALL_PAIRS_MIN_L 120.0 /* fm; see pasta_params.coulomb_all_pairs */

/* Device environment: where internal memory and the stream come from. */
typedef void* (*pasta_alloc_fn)(size_t bytes, void* user); /* returns a device pointer (256-B aligned) or NULL */
typedef void (*pasta_free_fn)(void* dev_ptr, void* user);
typedef struct pasta_env {
  uint32_t struct_size; /* sizeof(pasta_env) */
  int32_t device;       /* CUDA device ordinal */
  void* stream;         /* cudaStream_t; NULL = the legacy default stream */
  pasta_alloc_fn alloc; /* NULL = cudaMalloc/cudaFree */
  pasta_free_fn free;
  void* user;
} pasta_env;

typedef struct pasta_sim pasta_sim; /* opaque */

/* Fill *p with the paper's constants, r_c = 20 fm, fixed box, thermostat off, library-default cell_subdiv. */
int pasta_params_default(pasta_params* p);

/*
 * Create a simulation of N nucleons, N_p = floor(Y_P N + 1/2) protons at indices [0, N_p) (D12), in a
 * periodic cube of side L = (N/density)^(1/3).  Initial state, generated on the device
 * from `seed` by a counter-based generator: positions uniform in [0,L)^3, velocity components normal
 * with variance T/M (D15).  T is also the thermostat target.  env may be NULL (device 0,
 * default stream, cudaMalloc).
 * EINVAL: out/p NULL, wrong struct_size, N <= 0 or N >= 2^26 (sorted slots are packed in 26 bits), Y_P outside [0,1], density <= 0, T < 0,
 * r_c <= 0, r_c > L/2 (the nearest image would be ambiguous; D3), coulomb_all_pairs with L < 120 fm,
 * Lambda/lambda/mass <= 0,
 * scale_per_step <= 0, thermostat_interval < 0, cell_subdiv < 1.
 */
int pasta_create(pasta_sim** out, int64_t N, double Y_P, double density, double T, const pasta_params* p,
                 uint64_t seed, const pasta_env* env);
int pasta_destroy(pasta_sim* sim); /* frees internal buffers; NULL is a no-op */

/*
 * Force and energy of the current configuration (Eq. 1 + cut-off + nearest image):
 *   F_i = sum_{j != i, r_ij < r_c} -(1/r) dV/dr (x_i - x_j),   PE = sum_{i<j, r_ij < r_c} V(r_ij).
 * Rebuilds the cell list, runs the pair kernel (FP32 pair arithmetic, FP64 accumulation) and leaves
 * the forces cached for the next pasta_step.  F_dev ([N][3], original particle order) and pe_host may
 * each be NULL.  Synchronises the stream iff pe_host != NULL.
 */
int pasta_forces(pasta_sim* sim, double* F_dev, double* pe_host);

/*
 * Advance n velocity-Verlet steps of length dt (D6).  Per step:
 *   v += (dt/2M) F;  x = s (x + dt v), L = s L, wrap into [0,L);  cell list;  F = F(x);
 *   v += (dt/2M) F;  step count += 1;  if interval > 0 and count % interval == 0 and KE > 0:
 *   v *= sqrt(1.5 N T / KE)   (D7, D8).
 * Forces are evaluated first if they are stale (after create / set_state without forces / expand).
 * Asynchronous -- except in the neighbour-list regime (list_reuse), where every step reads one word back from the device
 * (the displacement trigger) while its force kernel runs.  On the chunk path a fixed-box step is replayed
 * as a CUDA graph (pasta_graph_replays).  EINVAL: n < 0, dt <= 0, or the box would shrink below 2 r_c.
 */
int pasta_step(pasta_sim* sim, int64_t n, double dt);

/* One-shot uniform scaling: L *= scale, x *= scale, v unchanged, forces stale (D9).
 * EINVAL: scale <= 0 or scale*L < 2 r_c. */
int pasta_expand(pasta_sim* sim, double scale);

/*
 * Friends-of-friends clusters over ALL nucleons with linking length r_cl (BASELINE variant of the
 * "MST" algorithm of; D13): connected components of {(i,j): r_ij <= r_cl}, nearest
 * image, predicate in FP64 with a pinned operation order.  label_dev[i] (may be NULL) receives the
 * smallest particle index of i's cluster; *n_clusters_host (may be NULL) the number of clusters.
 * EINVAL: r_cl <= 0 or r_cl > L/2.
 */
int pasta_clusters(pasta_sim* sim, double r_cl, int32_t* label_dev, int64_t* n_clusters_host);
/*
 * The paper's own two-radius "MST" cluster algorithm: protons within r_pp
 * (4.5 fm) of each other belong to one cluster, transitively; a neutron within r_np (3 fm) of a proton belongs to
 * that proton's cluster -- to the cluster of its NEAREST proton if several are in range (reading D24); other
 * neutrons are free (clusters of their own).  Nearest images, the pinned FP64 predicate of pasta_clusters.
 * label_dev[i] = smallest proton index of i's cluster (i itself for a free neutron).  pasta_cluster_sizes and
 * pasta_composition apply afterwards.  EINVAL: not 0 < r_np <= r_pp <= L/2.
 */
int pasta_clusters_mst(pasta_sim* sim, double r_pp, double r_np, int32_t* label_dev, int64_t* n_clusters_host);
/* After pasta_clusters / pasta_clusters_mst: A_dev[r], Z_dev[r] = mass and charge number of the cluster labelled r, 0 elsewhere. */
int pasta_cluster_sizes(pasta_sim* sim, int32_t* A_dev, int32_t* Z_dev);
/* After pasta_clusters: out6_host = {free-neutron mass fraction #(A=1,Z=0)/N, number of clusters with
 * A >= a_min, mean A, sigma A, mean Z, sigma Z over those clusters}.  Synchronises. */
int pasta_composition(pasta_sim* sim, int32_t a_min, double* out6_host);

/*
 * Friends-of-friends labels WITHOUT any device allocation -- for callers that cannot get device memory at the moment
 * they need cluster labels.  Two kinds of caller are meant: a process in which another component (a framework's
 * caching allocator, a second library, a job sized to fill the 180 GB) already owns the device's free memory, so that
 * cudaMalloc fails or would have to take memory away from it; and a caller running the analysis beside a simulation
 * that is stepping on other streams, for which the device-wide synchronisation hidden in cudaMalloc / cudaFree would
 * stall those steps.  pasta_clusters reserves up to seven internal arrays through pasta_env.alloc on its first call; this
 * entry point needs no pasta_sim, calls neither cudaMalloc nor cudaFree nor any library routine that allocates, and
 * enqueues only kernels and one 8-byte device-to-device copy on `stream`.  It returns without synchronising.
 *
 * What it computes is pasta_clusters' result (BASELINE variant of PAPER.md:154-158; D13): label_dev[i] = smallest
 * particle index in the connected component of i in the graph {(i, j): r_ij <= r_cl} at the nearest image, the same
 * pinned FP64 predicate, so the labels are identical bit for bit.  (A, Z) histograms and the MST variant are not
 * offered here.
 *   x_dev [N][3]      positions on `device`, as pasta_get_state returns them (input, read only)
 *   label_dev [N]     output, on `device`
 *   n_clusters_dev    output, ONE int64 on `device` (not a host pointer: a host scalar would force a synchronisation);
 *                     may be NULL
 *   device, stream    the CUDA device that holds the buffers -- the call makes it current and leaves it current, as
 *                     every other entry point of this library does -- and a cudaStream_t of it (NULL = default stream)
 *
 * The price is a fixed ceiling.  The union-find forest lives in a static device array inside the library image,
 * PASTA_CLUSTERS_NOALLOC_MAX_N entries (256 KiB), which every GPU that loads the library carries until the process
 * ends.  N above the ceiling is refused with PASTA_EINVAL and a message that names it; nothing is enqueued then.
 * Candidate pairs are enumerated all against all (no cell list, which would need four more scratch arrays): the cost
 * is N^2/2 FP64 predicates, so it is much slower than pasta_clusters, whose cell list makes the work linear in N:
 * measured on a B200 at r_cl = 3 fm, 89 ms at the ceiling (65 536 nucleons at 0.05 fm^-3) and 12 ms for 51 200 dilute
 * ones, where pasta_clusters takes 0.6 and 0.07 ms (profiles/r3_results.md).  It is the fallback, not the fast path.
 *
 * Set-up: the first call on each device looks up the device address of that array (cudaGetSymbolAddress, which also
 * loads the module on that device).  Make that first call outside any stream capture; later calls on the same device
 * do no set-up.
 * Sharing: all calls on one GPU use the SAME array.  Each call re-initialises the part it uses, so stale contents of
 * an earlier call never leak into a result -- but two calls whose kernels may run at the same time on one GPU (two
 * streams, two host threads) race on it and both results are then garbage.  Order them on one stream or with events.
 * EINVAL: N < 0 or N > PASTA_CLUSTERS_NOALLOC_MAX_N; x_dev or label_dev NULL with N > 0; L <= 0; r_cl <= 0 or
 * r_cl > L/2; device outside [0, 64).  N == 0 is allowed (writes 0 to n_clusters_dev).
 */
#define PASTA_CLUSTERS_NOALLOC_MAX_N 65536
int pasta_clusters_noalloc(const double* x_dev, int64_t N, double L, double r_cl, int32_t* label_dev,
                           int64_t* n_clusters_dev, int32_t device, void* stream);

/* State accessors.  Any pointer may be NULL (skipped).  get_* with a host scalar synchronises. */
int pasta_get_state(pasta_sim* sim, double* x_dev, double* v_dev, uint8_t* is_proton_dev, double* L_host,
                    int64_t* step_host);
/* Replace the state.  x is wrapped into [0,L) on the device.  F_dev != NULL supplies the forces F(x)
 * of that configuration (a restart); NULL marks them stale.  EINVAL: L < 2 r_c. */
int pasta_set_state(pasta_sim* sim, const double* x_dev, const double* v_dev, const uint8_t* is_proton_dev,
                    const double* F_dev, double L);
/* The same with HOST buffers (pinned memory recommended): asynchronous copies on the stream, then as
 * above.  get_state_host synchronises before returning.  F_host may be NULL. */
int pasta_get_state_host(pasta_sim* sim, double* x_host, double* v_host, double* F_host, double* L_host,
                         int64_t* step_host);
int pasta_set_state_host(pasta_sim* sim, const double* x_host, const double* v_host, const uint8_t* is_proton_host,
                         const double* F_host, double L);

/*
 * Pipelined host transfers.  The same state exchange as pasta_set_state_host / pasta_get_state_host, but on two side
 * streams with double-buffered device staging, so that while step k is being computed the inputs of step k + 1 are
 * already crossing PCIe in one direction and the result of step k - 1 in the other.  Both calls return at once.
 *   pasta_set_state_host_async: x, v, F (F may be NULL: forces stale) are copied host -> staging on the upload stream;
 *     the simulation's stream then takes them over (device copy, wrap into [0, L)).  The host buffers may be reused
 *     after the NEXT BUT ONE async set has returned, or after pasta_host_sync: from the third call on, a call first
 *     waits ON THE HOST until the copies of the set before last have left their host buffers (normally long done; it
 *     blocks only a host that has run more than two uploads ahead of the device).
 *   pasta_get_state_host_async: the simulation's stream snapshots x, v, F into staging (forces evaluated first if
 *     stale); the download stream copies the snapshot to the host buffers, which are valid after pasta_host_sync (or
 *     after the next but one async get has returned and been synchronised).  L and the step count are returned at once
 *     (the host tracks them).
 *   pasta_host_sync: waits for the simulation's stream and both side streams.
 * Use pinned host memory; pageable memory makes the copies synchronous.
 */
int pasta_set_state_host_async(pasta_sim* sim, const double* x_host, const double* v_host, const double* F_host, double L);
int pasta_get_state_host_async(pasta_sim* sim, double* x_host, double* v_host, double* F_host, double* L_host,
                               int64_t* step_host);
int pasta_host_sync(pasta_sim* sim);

/*
 * Cell assignment of the current positions on the species-independent grid of pasta_params.cell_subdiv
 * (D14) -- NOT the grids the force kernel sorts on, see pasta_force_cells below:
 *   ncell = max(1, floor(L k / r_c)); c = min(ncell-1, floor(x * (ncell/L))) per axis (FP64);
 *   id = (cz ncell + cy) ncell + cx;  cell_start = exclusive prefix sum of the histogram of id.
 * cell_id_dev [N], cell_start_dev [ncell^3 + 1] (size it with pasta_ncell first), either may be NULL.
 */
int pasta_cells(pasta_sim* sim, int32_t* cell_id_dev, int32_t* cell_start_dev, int32_t* ncell_side_host);
int pasta_ncell(pasta_sim* sim, int32_t* ncell_side_host); /* no device work */

/*
 * The cell lists the pair-force kernel really runs on (D14 applied per species).
 * Each species has its own grid: ncell cells per side in y and z, ncx = ncell * (thin cells per cell) along x, both
 * from the O3 formula c = min(n-1, floor(x * (n/L))) in FP64 with n = ncx for x and n = ncell for y, z.
 *   pasta_force_grid:  out4_host = {ncell_p, ncx_p, ncell_n, ncx_n} for the current box (no device work).
 *   pasta_force_cells: rebuilds the list for the CURRENT positions and copies it out:
 *     bin_dev [N]            bin of particle i (original order) = base_s + (cz ncell_s + cy) ncx_s + cx,
 *                            base_p = 0, base_n = ncell_p^2 ncx_p (protons' bins first);
 *     bin_start_dev [B + 1]  exclusive prefix sum of the histogram of bin, B = ncell_p^2 ncx_p + ncell_n^2 ncx_n;
 *     perm_dev [N]           sorted slot -> original index, ascending index inside a bin (a stable counting sort).
 *   Any pointer may be NULL.  Asynchronous.
 */
int pasta_force_grid(pasta_sim* sim, int32_t* out4_host);
int pasta_force_cells(pasta_sim* sim, int32_t* bin_dev, int32_t* bin_start_dev, int32_t* perm_dev);

/* KE = sum 1/2 M v^2 and PE of the current state (forces re-evaluated if stale).  Synchronises. */
int pasta_energy(pasta_sim* sim, double* ke_host, double* pe_host);
/* Per-particle energies e_i = 1/2 sum_j V(r_ij) of the last force evaluation, original order. */
int pasta_particle_energies(pasta_sim* sim, double* e_dev);

/* Number of ordered in-range pairs (i != j, r_ij < r_c) of the current configuration, counted by a
 * kernel in the same FP32 arithmetic the force kernel uses: the work unit of the throughput metric. */
int pasta_pair_count(pasta_sim* sim, int64_t* ordered_pairs_host);
/* The same, and beside it the number of those pairs that carry a term which is not exactly 0.0f in the FP32
 * pair arithmetic: out2_host = {in range, in range and (pp or exp2(-r^2 log2e / 2 Lambda) >= 2^-126)} (D23). */
int pasta_pair_counts(pasta_sim* sim, int64_t* out2_host);

/* Work statistics of one evaluation with the chunk pair kernel: out3_host = {sources streamed from the cell
 * rows (summed over chunks), tiles of <= 32 sources, pair evaluations executed}.  Synchronises.
 * (ordered in-range pairs / pair evaluations = the kernel's useful-work fraction.)  The evaluation covers every
 * target even under pasta_set_shard (no collective is issued; every rank computes the same complete F).  Its forces
 * are kept for the next pasta_step except with coulomb_all_pairs, where the chunk kernel's F lacks the Coulomb term
 * and the next consumer evaluates again. */
int pasta_force_stats(pasta_sim* sim, int64_t* out3_host);
/* Neighbour-list bookkeeping (list_reuse): out2_host = {force evaluations so far, of which rebuilt the list}. */
int pasta_list_stats(pasta_sim* sim, int64_t* out2_host);

/*
 * Instrumentation.  pasta_set_timing(sim, 1) brackets the cell-list, pair-force and integrate kernels
 * of every later step with CUDA events on the stream; pasta_get_timing synchronises and returns the
 * accumulated milliseconds {cell list, pair force, integrate} and the number of force evaluations
 * timed, then resets them.  pasta_launch_count = kernels launched by this simulation so far.
 */
int pasta_set_timing(pasta_sim* sim, int32_t enable);
int pasta_get_timing(pasta_sim* sim, double* ms3_host, int64_t* n_force_evals_host);
int64_t pasta_launch_count(const pasta_sim* sim);
/* A step in a fixed box (scale_per_step == 1, xi_dot == 0) on the chunk path enqueues the same kernels with the same
 * arguments every time; after two such steps pasta_step captures it as a CUDA graph (one for a plain step, one for a
 * step that ends with the velocity rescale) and replays it with a single launch.  Timing brackets, a
 * scaling box, the neighbour-list regime, a new particle set or dt, or PASTA_GRAPHS=0 in the environment take the
 * kernel-by-kernel path; the results are bit-identical either way.  Returns the number of steps replayed so far
 * (pasta_launch_count counts the kernels inside a replayed step as launched). */
int64_t pasta_graph_replays(const pasta_sim* sim);

/*
 * Target-sharded evaluation on several GPUs (the paper's P x Q force
 * decomposition with Q = 1).  Every rank holds the WHOLE state (positions, velocities, species) and keeps it
 * bit-identical; of every force evaluation it computes only the targets of its own stretch of the cell-sorted order
 * (the sorted slots [bounds[rank], bounds[rank+1]) of pasta_shard_bounds: contiguous in space along the sort, balanced
 * by the estimated pair work of the two species), leaves zeros elsewhere, and the ranks' partial F and e -- stored back
 * to back, so ONE call on 4 N doubles, or on the 3 N of F alone when an evaluation computes no energies -- are then
 * summed in place by `allreduce`: the paper's MPI_Allreduce of the forces; every
 * particle's force is complete on exactly one rank, so the sum is exact and the result is bit-identical to the
 * one-GPU evaluation.  Cell list and integration are replicated (they cost a few % of a step).
 *   allreduce(dev_ptr, n, user): sum the n doubles at dev_ptr over all ranks, in place, ordered with the simulation's
 *   stream (the Python binding issues torch.distributed.all_reduce on it); returns 0 on success.
 * world == 1 switches sharding off.  EINVAL: rank outside [0, world), world < 1, allreduce NULL with world > 1.
 */
typedef int (*pasta_allreduce_fn)(void* dev_ptr, int64_t n_doubles, void* user);
int pasta_set_shard(pasta_sim* sim, int32_t rank, int32_t world, pasta_allreduce_fn allreduce, void* user);
/*
 * The partition pasta_set_shard uses (host arithmetic only; no GPU needed): bounds_host[0..world] with bounds[0] = 0,
 * bounds[world] = N, non-decreasing.  Sorted slots [0, Np) are protons, [Np, N) neutrons; a proton target costs
 * cost_p and a neutron target cost_n (any positive units), and every rank gets the same total cost up to one target.
 * EINVAL: N <= 0, Np outside [0, N], world < 1, a cost <= 0, bounds_host NULL.
 */
int pasta_shard_bounds(int64_t N, int64_t Np, double cost_p, double cost_n, int32_t world, int64_t* bounds_host);
/* The costs pasta_set_shard feeds it: streamed candidates times their evaluation cost at uniform density --
 * out2_host = {cost of a proton target, cost of a neutron target} for the simulation's parameters (host only). */
int pasta_shard_costs(const pasta_sim* sim, double* out2_host);

/*
 * Environment variables read once by pasta_create.  None is needed in normal use and none changes a result beyond
 * FP32 summation order; they exist for the tests' cross-checks and for measurements:
 *   PASTA_FORCE_VARIANT=1  the thread-per-target pair kernel on one isotropic grid (k2_force.cu) instead of the chunk
 *                          kernel: the in-library cross-check of the production kernel (no lists, no graphs, no stats)
 *   PASTA_GRAPHS=0         never replay a step as a CUDA graph (see pasta_graph_replays)
 *   PASTA_AUTO_GRID=0      both species' force grids take pasta_params.cell_subdiv instead of a k chosen per species
 *   PASTA_X_SUBDIV=n       n thin cells per cell along x on the force grids instead of the automatic choice
 */
const char* pasta_last_error(void);
const char* pasta_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PASTA_H_ */
