// Internal declarations of the pasta sm_100a library (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "pasta.h"

// targets per chunk of the pair kernel (k1_cells.cu builds the table, k2_chunk.cu consumes it)
#ifndef PASTA_CHUNK_T
#define PASTA_CHUNK_T 8
#endif

namespace pasta {

// ---- error plumbing ------------------------------------------------------------------------------
void set_error(const char* fmt, ...);
#define PASTA_CUDA_OK(expr)                                                                  \
  do {                                                                                       \
    cudaError_t err__ = (expr);                                                              \
    if (err__ != cudaSuccess) {                                                              \
      ::pasta::set_error("%s failed at %s:%d: %s", #expr, __FILE__, __LINE__,                \
                         cudaGetErrorString(err__));                                         \
      return PASTA_ECUDA;                                                                    \
    }                                                                                        \
  } while (0)
#define PASTA_TRY(expr)              \
  do {                               \
    int rc__ = (expr);               \
    if (rc__ != PASTA_OK) return rc__; \
  } while (0)

// ---- device buffer owned through pasta_env ---------------------------------------------------------
struct Sim;
struct Buffer {
  void* ptr = nullptr;
  size_t bytes = 0;
  template <class T>
  T* as() const { return reinterpret_cast<T*>(ptr); }
};
int buffer_reserve(Sim* s, Buffer* b, size_t bytes);  // grow-only; contents are NOT preserved
void buffer_release(Sim* s, Buffer* b);

// ---- grid of the force cell list (host-side description, recomputed whenever L changes) ------------
struct Grid {
  int32_t ncell = 1;   // cells per side in y and z (and in x when xsub == 1)
  int32_t xsub = 1;    // the force grids slice every cell into xsub thin cells along x
  int32_t ncx = 1;     // ncell * xsub
  int64_t nc3 = 1;     // number of cells: ncell^2 * ncx
  double inv_w = 1.0;  // ncell / L  (FP64 division on the host, D14)
  double w = 1.0;      // L / ncell
  double inv_wx = 1.0; // ncx / L
  double wx = 1.0;     // L / ncx
};
Grid make_grid(double L, double r_c, int32_t k, int32_t xsub = 1);
// packed cell coordinates of a sorted slot: cx (12 bits) | cy << 12 (10 bits) | cz << 22 (10 bits)
#define PASTA_CX(c) ((c) & 4095)
#define PASTA_CY(c) (((c) >> 12) & 1023)
#define PASTA_CZ(c) (((c) >> 22) & 1023)

// The two species' grids as the K1 kernels (and the fused kick-drift-count kernel of K3) see them.
struct GridPair {
  int ncell[2], ncx[2];
  int base[2];  // first bin of the species' grid: base[0] = 0, base[1] = number of cells of grid 0
  double inv_w[2], w[2], inv_wx[2], wx[2];
};

#ifdef __CUDACC__
// c = min(ncell-1, floor(x * inv_w)) -- a single correctly rounded FP64 multiply, then floor (D14).
__device__ __forceinline__ int cell_coord(double x, double inv_w, int ncell) {
  int q = (int)floor(__dmul_rn(x, inv_w));
  q = q > ncell - 1 ? ncell - 1 : q;
  return q < 0 ? 0 : q;
}
// (species, cell) bin of a particle on its species' force grid
__device__ __forceinline__ int force_bin(const GridPair& g, int sp, double x, double y, double z) {
  const int nc = g.ncell[sp], ncx = g.ncx[sp];
  const int cx = cell_coord(x, g.inv_wx[sp], ncx), cy = cell_coord(y, g.inv_w[sp], nc), cz = cell_coord(z, g.inv_w[sp], nc);
  return g.base[sp] + (cz * nc + cy) * ncx + cx;
}
#endif

#ifdef __CUDACC__
// List mode (k2_list.cu): what the frozen sorted order needs of a moved particle (k1_refresh_kernel; fused into the
// kick-drift kernel of a step).
struct RefreshArgs {
  const double* xref;     // positions at the list build
  const int32_t* cxyz;    // [slot] frozen packed cell coordinates
  float4* pos4;           // [slot] out
  GridPair g;             // the frozen cell counts with the widths of the current box
  int32_t Np;
  double sigma, L, invL, L0, invL0;
  unsigned* scratch;      // {max displacement^2 (float bits), blocks finished}; zero between launches
  unsigned long long* mbox;
  unsigned seq;
  double delta;           // the lists survive iff 2 * displacement <= delta (halo, less what a shrunken box took of it)
  unsigned* gate;         // device word: 1 = the lists survive this step (read by the force kernel enqueued behind), 0 = not
};
// pos4[slot] = sigma * (x - centre of the slot's frozen cell), nearest image -- bit for bit k1_gather_kernel's value
// while the particle is inside its cell; returns its squared displacement since the build, measured in co-moving
// coordinates u = x / L and expressed at the build's box side (the trigger of the neighbour list).
__device__ __forceinline__ float refresh_slot(const RefreshArgs& R, const int slot, const int64_t i, const double* xi) {
  const int c = R.cxyz[slot], sp = slot < R.Np ? 0 : 1;
  const int cc[3] = {PASTA_CX(c), PASTA_CY(c), PASTA_CZ(c)};
  const double wa[3] = {R.g.wx[sp], R.g.w[sp], R.g.w[sp]};
  float p[3];
  double dd2 = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double d = xi[a] - ((double)cc[a] + 0.5) * wa[a];
    d -= R.L * rint(d * R.invL);
    p[a] = (float)(R.sigma * d);
    double du = xi[a] * R.invL - R.xref[3 * i + a] * R.invL0;
    du -= rint(du);
    du *= R.L0;
    dd2 += du * du;
  }
  R.pos4[slot] = make_float4(p[0], p[1], p[2], __int_as_float(c));
  return __double2float_ru(dd2);
}
// Block maximum of d2, folded into the launch's maximum; the last block to finish posts {seq, maximum} to the host's
// mailbox and re-arms the scratch words.  Every thread of the block must call it.  blockDim.x <= 256.
__device__ __forceinline__ void refresh_post(const RefreshArgs& R, float d2) {
  __shared__ float wmax[8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) d2 = fmaxf(d2, __shfl_xor_sync(0xffffffffu, d2, o));
  if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = d2;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < (int)(blockDim.x >> 5); ++k) d2 = fmaxf(d2, wmax[k]);
    atomicMax(R.scratch, __float_as_uint(d2));  // d2 >= 0: the bit patterns order like the values
    __threadfence();
    if (atomicAdd(R.scratch + 1, 1u) == gridDim.x - 1) {
      const unsigned m = atomicExch(R.scratch, 0u);
      R.scratch[1] = 0u;
      // the trigger, decided here in the host's arithmetic, so that the force kernel already enqueued behind this one
      // runs (or returns at once) without a round trip to the host
      *R.gate = 2.0 * sqrt((double)__uint_as_float(m)) <= R.delta ? 1u : 0u;
      *reinterpret_cast<volatile unsigned long long*>(R.mbox) = ((unsigned long long)R.seq << 32) | m;
      __threadfence_system();
    }
  }
}
#endif

// Constants of the FP32 pair arithmetic, derived on the host in FP64 (k2_force.cu explains them).
struct PairConsts {
  float sigma;       // coordinate pre-scale sqrt(log2(e) / (2 Lambda))
  float inv_sigma;   // 1 / sigma
  float rc2s;        // (sigma r_c)^2
  float rn2s;        // (sigma r_n)^2, r_n = cut-off of the nuclear terms: r_nuc if set, else r_c
  float a;           // a
  float g2a;         // 2 a / (Lambda sigma)          (force constants carry the 1/sigma of d' -> d)
  float B_like, B_unlike;      // b + c, b - c
  float gB_like, gB_unlike;    // B / (Lambda sigma)
  float kappa;       // log2(e) / (sigma lambda):  exp(-r/lambda) = exp2(-kappa r')
  float alpha_s;     // alpha sigma:                E_c = alpha_s exp2(.) / r'
  float alpha_s2;    // alpha sigma^2:              Coulomb part of g'
  float inv_lam_s;   // 1 / (lambda sigma):         (1/r + 1/lambda) = sigma (1/r' + inv_lam_s)
  float v_self;      // a + b + c : V(0) of the like-species self pair, removed analytically
};
PairConsts make_pair_consts(const pasta_params& p);

// Tuning knobs that are not part of the ABI: read once per pasta_create from the environment
// (PASTA_FORCE_VARIANT, PASTA_AUTO_GRID, PASTA_X_SUBDIV); the tests use them to cross-check kernels.
struct Tuning {
  int force_variant = 0;  // 0 = chunk kernel (production); 1 = thread-per-target kernel on one isotropic grid (k2_force.cu)
  int auto_grid = 1;      // 1: each species' force grid picks its own k (about 8 particles per cell); 0: both use cell_subdiv
  int x_subdiv = 0;       // thin cells along x per force-grid cell (0 = automatic: 8, fewer for a sparse species)
  int graphs = 1;         // replay a fixed-box step as a CUDA graph (PASTA_GRAPHS=0: always enqueue kernel by kernel)
};

struct Sim {
  // configuration
  pasta_params prm;
  Tuning tune;
  pasta_env env;
  cudaStream_t stream = nullptr;
  int64_t N = 0;
  int64_t Np = 0;
  double T = 0.0;
  double L = 0.0;
  int64_t step_count = 0;
  double lin_L0 = 0.0;   // linear expansion (xi_dot > 0): side and step count at its start
  int64_t lin_n = 0;
  bool forces_valid = false;
  bool energies_valid = false;
  bool clusters_valid = false;
  bool hist_valid = false;    // bin_count/cell_id hold the histogram of the current x on the current force grids
  bool hist_uniform = false;  // ... built for the uniform (one grid) variant
  int64_t bins_zeroed = 0;    // bin_count[0, bins_zeroed) is known to be all zero (the scatter leaves it so)
  int64_t launches = 0;
  int64_t n_force_evals = 0;  // force evaluations so far, and how many of them (re)built the cell list
  int64_t n_list_builds = 0;

  // state (device)
  Buffer x, v, F, e, is_p;  // double[N][3] x3, double[N], uint8[N]

  // cell list (device)
  Grid grid_sp[2];    // [0] protons' grid, [1] neutrons' grid
  int64_t bin_base[2] = {0, 0};
  Buffer cell_id;     // int32[N]   bin of every particle (force grids) / O3 id (pasta_cells)
  Buffer bin_count;   // int32[2 nc3 + 1] scratch histogram over (species, cell) bins
  Buffer bin_start;   // int32[2 nc3 + 1] exclusive scan; protons' bins first
  Buffer scan_tmp;    // block sums of the scan
  Buffer perm_raw;    // int32[N]   sorted slot -> original index, members of a bin in arrival order
  Buffer perm;        // int32[N]   sorted slot -> original index
  Buffer pos4;        // float4[N]  sorted: sigma * cell-relative position, .w = cell x index
  Buffer cxyz;        // int32[N]   sorted: packed cell coordinates (cx | cy<<10 | cz<<20)
  Buffer cpos;        // float4[2 Np] sorted protons as box fractions x / L, hi and lo parts (k2_coulomb.cu)

  // reductions
  Buffer partials;    // double[>= 4096]
  Buffer scalars;     // double[16] device scalars: [0] KE, [1] PE, [2] rescale factor, [3..] scratch
  Buffer counters;    // unsigned long long[16]

  // clusters
  Buffer cl_parent, cl_A, cl_Z;  // int32[N] each
  Buffer cl_cell_id, cl_count, cl_start, cl_perm;

  // reused neighbour lists (k2_list.cu).  While list.valid the sorted order (perm, cxyz), the cell
  // counts of grid_sp, the chunk table and the lists are FROZEN; pos4 is refreshed from x every step.
  struct ListState {
    bool valid = false;     // the frozen order and the lists describe the current particles (subject to the trigger)
    double L0 = 0.0;        // box side at the build
    double halo = 0.0;      // halo the lists were built with
    unsigned seq = 0;       // sequence number of the displacement readback
    bool pending = false;   // a refresh for the current positions is already enqueued (fused into the kick-drift kernel)
    volatile unsigned long long* mbox_host = nullptr;  // pinned, mapped: {seq << 32 | float bits of max displacement^2}
    unsigned long long* mbox_dev = nullptr;
  } list;
  Buffer xref;        // double[N][3] positions at the build
  Buffer slot_of;     // int32[N] original index -> sorted slot (inverse of perm)
  Buffer list_off, list_pool;  // int4[N] {proton list: first, length; neutron list: first, length}; int32 sorted slots
  int64_t list_entries = 0;
  bool no_lists = false;       // lists are off: for one call (pasta_force_stats needs the chunk kernel's own sort), or since a
                               // list build found the state too dense -- until the next set_state / expand, which retry

  // pair-force chunk table (k1_cells.cu -> k2_chunk.cu): [0, max_chunks) entries first slot | count << 26,
  // [max_chunks, 2 max_chunks) the list of chunks that need several rounds; the counters live in
  // counters[24] (int32 view [48]: number of chunks, [49]: length of that list)
  Buffer chunk_tab;
  Buffer chunk_first;       // int32[N]: first target slot of the chunk a sorted slot belongs to (who owns it under sharding)
  int64_t max_chunks = 0;   // launch bound of the pair kernel: chunk_nprim primary entries + overflow capacity
  int64_t chunk_nprim = 0;
  bool chunks_sparse = false;  // some species' chunks come from the SPARSE (cell block) builder

  // pipelined host transfers (pasta_*_host_async): side streams, double-buffered staging, hand-over events
  struct HostPipe {
    cudaStream_t up = nullptr, down = nullptr;
    Buffer in[2], out[2];                 // 72 N bytes each: x, v, F
    cudaEvent_t in_done[2] = {nullptr, nullptr}, in_taken[2] = {nullptr, nullptr};
    cudaEvent_t out_ready[2] = {nullptr, nullptr}, out_done[2] = {nullptr, nullptr};
    int64_t n_in = 0, n_out = 0;
  } pipe;

  // a fixed-box MD step captured as a CUDA graph (pasta_step): [0] plain step, [1] step that ends with the rescale
  struct StepGraph {
    cudaGraphExec_t exec[2] = {nullptr, nullptr};
    int64_t launches[2] = {0, 0};  // kernels in each
    double L = 0.0, dt = 0.0;      // what the captured kernel arguments were computed for
    int energy = 0;
    int64_t gen = -1;              // value of state_gen at capture
    int64_t replays = 0;           // steps replayed so far
    cudaStream_t cap = nullptr;    // capture happens on a stream of our own (the caller's may be the legacy default stream)
    bool capturing = false;        // s->stream is `cap` right now and must not be synchronised; the caller's stream is `home`
    cudaStream_t home = nullptr;
    int warm = 0;                  // eligible steps enqueued kernel by kernel since the last change (buffers settle)
  } graph;
  // target sharding over several GPUs (pasta_set_shard): this rank evaluates the targets in sorted slots [slot_lo, slot_hi)
  struct Shard {
    int32_t rank = 0, world = 1;
    pasta_allreduce_fn allreduce = nullptr;
    void* user = nullptr;
    int32_t slot_lo = 0, slot_hi = 0x7fffffff;
  } shard;
  int sort_kind = -1;     // what the sorted arrays and grid_sp describe: 0 chunk-path grids, 1 uniform grid, 2 list grid, -1 nothing
  int64_t state_gen = 0;  // bumped whenever a device buffer moves or the particle set changes: captured graphs are stale

  // timing: pairs of events (start, stop) tagged with the kernel group they bracket
  bool timing = false;
  std::vector<cudaEvent_t> evs;
  std::vector<int> ev_kind;
  size_t ev_used = 0;
  double ms_acc[3] = {0, 0, 0};
  int64_t n_timed = 0;
};

// ---- kernel launchers (one translation unit each) ---------------------------------------------------
// K1  k1_cells.cu
bool list_mode_wanted(const Sim* s);                   // would a force evaluation of the current box run on reused lists?
double list_halo(const Sim* s);
void k1_grids(const Sim* s, bool uniform_grid, Grid out[2], GridPair* g);  // the species' grids for the current L (host only)
void k1_frozen_grids(Sim* s, GridPair* g);             // the frozen cell counts at the current L (list mode)
int k1_refresh(Sim* s, double* max_disp_host);         // list mode: pos4 from the moved x; largest displacement since the build
int k1_refresh_wait(Sim* s, double* max_disp_host);    // ... the readback of a refresh already enqueued (fused into K3)
#ifdef __CUDACC__
void k1_refresh_args(Sim* s, RefreshArgs* out);        // (bumps the sequence number)
#endif
int k1_setup(Sim* s, bool uniform_grid, GridPair* g);  // grids for the current L, buffers, a zeroed histogram
int k1_build(Sim* s, bool uniform_grid = false);       // (species,cell) counting sort, pos4/perm, chunk table; uses the
                                                       // histogram of k3_kick_drift_count if s->hist_valid
int k1_export_cells(Sim* s, int32_t* cell_id_dev, int32_t* cell_start_dev);
int scan_exclusive(Sim* s, const int32_t* in, int32_t* out, int64_t n);  // out[0..n] (n+1 entries)
// K2  k2_force.cu
int k2_forces(Sim* s, bool with_energy, double kick = 0.0);  // F, e in original order; kick != 0: v += kick F rides along
int k2_pair_count(Sim* s, int64_t* ordered_pairs_host, int64_t* nonzero_pairs_host);
int k2_reference_forces(Sim* s, bool with_energy);     // variant 1: thread per target (k2_force.cu)
int k2_chunk_forces(Sim* s, bool with_energy, bool stats, double kick = 0.0);  // variant 2: chunk kernel (k2_chunk.cu)
int k2_list_build(Sim* s, double halo);                // neighbour lists of the sorted order k1_build just made (k2_list.cu)
int k2_list_forces(Sim* s, bool with_energy, bool gated = false, double kick = 0.0);  // the pair kernel on those lists; gated:
                                                       // only if the refresh just enqueued lets the lists live; kick: v += kick F
int k2_coulomb_all_pairs(Sim* s, bool with_energy);    // += screened Coulomb of every proton pair, nearest image (k2_coulomb.cu)
// K3  k3_integrate.cu
int k3_init_state(Sim* s, uint64_t seed);
int k3_kick_drift_refresh(Sim* s, double dt, double scale, double L_wrap);  // list mode: kick, drift + the refresh of the frozen order
int k3_kick_drift_count(Sim* s, double dt, double scale, double L_wrap, bool count);  // kick, drift, scale, wrap into
                                                     // [0, L_wrap); count: + cell histogram on the grids of box s->L
int k3_kick_ke(Sim* s, double dt, bool rescale);       // second half kick + KE (+ rescale)
int k3_wrap_scale(Sim* s, double scale, double L_new); // x = wrap(scale x)
int k3_kinetic(Sim* s, double* ke_host);
int k3_sum(Sim* s, const double* in, int64_t n, int slot);  // deterministic sum into scalars[slot]
int k3_count_protons(Sim* s);                          // s->Np from is_p (synchronises)
// K4  k4_clusters.cu
int k4_clusters(Sim* s, double r_cl, double r_np, int32_t* label_dev, int64_t* n_clusters_host);
int k4_composition(Sim* s, int32_t a_min, double* out6_host);

inline int grid_for(int64_t n, int block) { return (int)((n + block - 1) / block); }

}  // namespace pasta
