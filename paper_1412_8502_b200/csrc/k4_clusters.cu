// K4 -- friends-of-friends cluster labelling by lock-free union-find (BASELINE
// variant of the "MST" cluster algorithm; reading D13).
//
// Edges: all pairs with nearest-image r^2 <= r_cl^2, predicate in FP64 with a pinned operation order
// (every operation individually rounded, no FMA contraction), so the edge set -- and with it the
// canonical labels (smallest member index) -- is identical to a brute-force FP64 enumeration.
// Candidates come from a cell grid of width >= r_cl (own + 26 neighbour cells).  Roots are always the
// smaller index (hook larger root under smaller with atomicCAS), so after flattening label = min index.
#include <mutex>

#include "pasta_internal.cuh"

namespace pasta {

__device__ __forceinline__ double pinned_r2(const double* __restrict__ x, int i, int j, double L, double invL) {
  double dx = __dsub_rn(x[3 * i + 0], x[3 * j + 0]);
  double dy = __dsub_rn(x[3 * i + 1], x[3 * j + 1]);
  double dz = __dsub_rn(x[3 * i + 2], x[3 * j + 2]);
  dx = __dsub_rn(dx, __dmul_rn(L, rint(__dmul_rn(dx, invL))));
  dy = __dsub_rn(dy, __dmul_rn(L, rint(__dmul_rn(dy, invL))));
  dz = __dsub_rn(dz, __dmul_rn(L, rint(__dmul_rn(dz, invL))));
  return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

__device__ __forceinline__ bool fof_linked(const double* __restrict__ x, int i, int j, double L, double invL,
                                           double rcl2) {
  double dx = __dsub_rn(x[3 * i + 0], x[3 * j + 0]);
  double dy = __dsub_rn(x[3 * i + 1], x[3 * j + 1]);
  double dz = __dsub_rn(x[3 * i + 2], x[3 * j + 2]);
  dx = __dsub_rn(dx, __dmul_rn(L, rint(__dmul_rn(dx, invL))));
  dy = __dsub_rn(dy, __dmul_rn(L, rint(__dmul_rn(dy, invL))));
  dz = __dsub_rn(dz, __dmul_rn(L, rint(__dmul_rn(dz, invL))));
  const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
  return r2 <= rcl2;
}

__device__ __forceinline__ int uf_find(int* parent, int i) {
  int p = __ldcg(parent + i);
  while (p != i) {
    const int gp = __ldcg(parent + p);
    if (gp != p) parent[i] = gp;  // path halving; racy but monotone (parents only ever decrease)
    i = p;
    p = gp;
  }
  return i;
}

__device__ __forceinline__ void uf_union(int* parent, int a, int b) {
  while (true) {
    a = uf_find(parent, a);
    b = uf_find(parent, b);
    if (a == b) return;
    const int hi = a > b ? a : b, lo = a > b ? b : a;
    const int old = atomicCAS(&parent[hi], hi, lo);
    if (old == hi) return;
    a = old;  // someone else hooked hi first; retry from its new parent
    b = lo;
  }
}

__global__ void k4_init_kernel(int64_t N, int32_t* __restrict__ parent, int32_t* __restrict__ A, int32_t* __restrict__ Z) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  parent[i] = (int32_t)i;
  A[i] = 0;
  Z[i] = 0;
}

__device__ __forceinline__ int cl_cell_coord(double x, double inv_w, int ncell) {
  int q = (int)floor(__dmul_rn(x, inv_w));
  q = q > ncell - 1 ? ncell - 1 : q;
  return q < 0 ? 0 : q;
}

__global__ void k4_count_kernel(int64_t N, const double* __restrict__ x, double inv_w, int ncell,
                                int32_t* __restrict__ cell_id, int32_t* __restrict__ count) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int cx = cl_cell_coord(x[3 * i + 0], inv_w, ncell), cy = cl_cell_coord(x[3 * i + 1], inv_w, ncell),
            cz = cl_cell_coord(x[3 * i + 2], inv_w, ncell);
  const int id = (cz * ncell + cy) * ncell + cx;
  cell_id[i] = id;
  atomicAdd(&count[id], 1);
}

__global__ void k4_scatter_kernel(int64_t N, const int32_t* __restrict__ cell_id, const int32_t* __restrict__ start,
                                  int32_t* __restrict__ count, int32_t* __restrict__ perm) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int id = cell_id[i];
  const int old = atomicSub(&count[id], 1);
  perm[start[id] + old - 1] = (int32_t)i;
}

// One thread per particle i: link with every j < i in the 27 surrounding cells that satisfies the predicate.
__global__ void k4_link_cells_kernel(int64_t N, const double* __restrict__ x, const int32_t* __restrict__ cell_id,
                                     const int32_t* __restrict__ start, const int32_t* __restrict__ perm, int ncell,
                                     double L, double invL, double rcl2, int32_t* __restrict__ parent,
                                     const uint8_t* __restrict__ only) {  // only != NULL: link protons only (MST)
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  if (only && !only[i]) return;
  const int id = cell_id[i];
  const int cx = id % ncell, cy = (id / ncell) % ncell, cz = id / (ncell * ncell);
  for (int dz = -1; dz <= 1; ++dz)
    for (int dy = -1; dy <= 1; ++dy)
      for (int dx = -1; dx <= 1; ++dx) {
        const int jx = (cx + dx + ncell) % ncell, jy = (cy + dy + ncell) % ncell, jz = (cz + dz + ncell) % ncell;
        const int q = (jz * ncell + jy) * ncell + jx;
        for (int s = start[q]; s < start[q + 1]; ++s) {
          const int j = perm[s];
          if (j < i && (!only || only[j]) && fof_linked(x, j, (int)i, L, invL, rcl2)) uf_union(parent, (int)i, j);
        }
      }
}

// MST step 2 (reading D24): a neutron joins the cluster of its nearest proton within r_np (smallest
// pinned r2, then smallest index); it becomes a leaf under that proton -- nothing is ever hooked under a neutron.
// cell_id == NULL: all protons are scanned (small boxes).
__global__ void k4_attach_kernel(int64_t N, const double* __restrict__ x, const uint8_t* __restrict__ is_p,
                                 const int32_t* __restrict__ cell_id, const int32_t* __restrict__ start,
                                 const int32_t* __restrict__ perm, int ncell, double L, double invL, double rnp2,
                                 int32_t* __restrict__ parent) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N || is_p[i]) return;
  int best = -1;
  double best_r2 = 0.0;
  if (cell_id) {
    const int id = cell_id[i];
    const int cx = id % ncell, cy = (id / ncell) % ncell, cz = id / (ncell * ncell);
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          const int jx = (cx + dx + ncell) % ncell, jy = (cy + dy + ncell) % ncell, jz = (cz + dz + ncell) % ncell;
          const int q = (jz * ncell + jy) * ncell + jx;
          for (int s = start[q]; s < start[q + 1]; ++s) {
            const int j = perm[s];
            if (!is_p[j]) continue;
            const double r2 = pinned_r2(x, (int)i, j, L, invL);
            if (r2 <= rnp2 && (best < 0 || r2 < best_r2 || (r2 == best_r2 && j < best))) {
              best = j;
              best_r2 = r2;
            }
          }
        }
  } else {
    for (int j = 0; j < (int)N; ++j) {
      if (!is_p[j]) continue;
      const double r2 = pinned_r2(x, (int)i, j, L, invL);
      if (r2 <= rnp2 && (best < 0 || r2 < best_r2)) {
        best = j;
        best_r2 = r2;
      }
    }
  }
  if (best >= 0) parent[i] = best;
}

// Small boxes (fewer than 3 cells per side): all pairs j < i.
__global__ void k4_link_all_kernel(int64_t N, const double* __restrict__ x, double L, double invL, double rcl2,
                                   int32_t* __restrict__ parent, const uint8_t* __restrict__ only) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  if (only && !only[i]) return;
  for (int j = 0; j < (int)i; ++j)
    if ((!only || only[j]) && fof_linked(x, j, (int)i, L, invL, rcl2)) uf_union(parent, (int)i, j);
}

__global__ void k4_flatten_kernel(int64_t N, int32_t* __restrict__ parent, const uint8_t* __restrict__ is_p,
                                  int32_t* __restrict__ label_out, int32_t* __restrict__ A, int32_t* __restrict__ Z,
                                  unsigned long long* __restrict__ n_clusters) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int r = uf_find(parent, (int)i);
  if (label_out) label_out[i] = r;
  atomicAdd(&A[r], 1);
  if (is_p[i]) atomicAdd(&Z[r], 1);
  if (r == (int)i) atomicAdd(n_clusters, 1ull);
}

// After flatten every parent[i] may still be an intermediate node for readers that raced; a second pass
// makes parent[] itself the label array so that later calls can read it directly.
__global__ void k4_store_labels_kernel(int64_t N, int32_t* __restrict__ parent) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  int r = (int)i;
  for (int p = __ldcg(parent + r); p != r; p = __ldcg(parent + r)) r = p;
  parent[i] = r;  // r is a root: roots are never rewritten, so concurrent readers still terminate at r
}

// r_np > 0: the paper's two-radius MST (protons linked at r_cl = r_pp, neutrons attached at r_np <= r_pp);
// r_np == 0: friends-of-friends over all nucleons at r_cl.
int k4_clusters(Sim* s, double r_cl, double r_np, int32_t* label_dev, int64_t* n_clusters_host) {
  const int64_t N = s->N;
  const bool mst = r_np > 0.0;
  const uint8_t* only = mst ? s->is_p.as<uint8_t>() : nullptr;
  const int B = 256;
  PASTA_TRY(buffer_reserve(s, &s->cl_parent, sizeof(int32_t) * (size_t)N));
  PASTA_TRY(buffer_reserve(s, &s->cl_A, sizeof(int32_t) * (size_t)N));
  PASTA_TRY(buffer_reserve(s, &s->cl_Z, sizeof(int32_t) * (size_t)N));
  int32_t* parent = s->cl_parent.as<int32_t>();
  unsigned long long* counter = s->counters.as<unsigned long long>() + 1;
  PASTA_CUDA_OK(cudaMemsetAsync(counter, 0, sizeof(unsigned long long), s->stream));
  k4_init_kernel<<<grid_for(N, B), B, 0, s->stream>>>(N, parent, s->cl_A.as<int32_t>(), s->cl_Z.as<int32_t>());
  s->launches += 1;

  // grid of width >= r_cl (a hair wider, so that a rounding of x*inv_w can never separate a linked pair
  // by two cells); at most 400 cells per side (256 MB of histogram)
  double q = floor(s->L / (r_cl * (1.0 + 1e-9)));
  if (q > 400.0) q = 400.0;
  const int ncell = (int)q;
  const double L = s->L, invL = 1.0 / s->L, rcl2 = r_cl * r_cl;
  if (ncell >= 3) {
    const int64_t nc3 = (int64_t)ncell * ncell * ncell;
    PASTA_TRY(buffer_reserve(s, &s->cl_cell_id, sizeof(int32_t) * (size_t)N));
    PASTA_TRY(buffer_reserve(s, &s->cl_perm, sizeof(int32_t) * (size_t)N));
    PASTA_TRY(buffer_reserve(s, &s->cl_count, sizeof(int32_t) * (size_t)(nc3 + 1)));
    PASTA_TRY(buffer_reserve(s, &s->cl_start, sizeof(int32_t) * (size_t)(nc3 + 1)));
    int32_t* cnt = s->cl_count.as<int32_t>();
    int32_t* start = s->cl_start.as<int32_t>();
    PASTA_CUDA_OK(cudaMemsetAsync(cnt, 0, sizeof(int32_t) * (size_t)(nc3 + 1), s->stream));
    k4_count_kernel<<<grid_for(N, B), B, 0, s->stream>>>(N, s->x.as<double>(), (double)ncell / L, ncell,
                                                         s->cl_cell_id.as<int32_t>(), cnt);
    s->launches += 1;
    PASTA_TRY(scan_exclusive(s, cnt, start, nc3));
    k4_scatter_kernel<<<grid_for(N, B), B, 0, s->stream>>>(N, s->cl_cell_id.as<int32_t>(), start, cnt,
                                                           s->cl_perm.as<int32_t>());
    k4_link_cells_kernel<<<grid_for(N, 128), 128, 0, s->stream>>>(N, s->x.as<double>(), s->cl_cell_id.as<int32_t>(),
                                                                  start, s->cl_perm.as<int32_t>(), ncell, L, invL, rcl2,
                                                                  parent, only);
    s->launches += 2;
    if (mst) {
      k4_attach_kernel<<<grid_for(N, 128), 128, 0, s->stream>>>(N, s->x.as<double>(), s->is_p.as<uint8_t>(),
                                                                s->cl_cell_id.as<int32_t>(), start,
                                                                s->cl_perm.as<int32_t>(), ncell, L, invL, r_np * r_np,
                                                                parent);
      s->launches += 1;
    }
  } else {
    k4_link_all_kernel<<<grid_for(N, 128), 128, 0, s->stream>>>(N, s->x.as<double>(), L, invL, rcl2, parent, only);
    s->launches += 1;
    if (mst) {
      k4_attach_kernel<<<grid_for(N, 128), 128, 0, s->stream>>>(N, s->x.as<double>(), s->is_p.as<uint8_t>(), nullptr,
                                                                nullptr, nullptr, 0, L, invL, r_np * r_np, parent);
      s->launches += 1;
    }
  }
  k4_flatten_kernel<<<grid_for(N, B), B, 0, s->stream>>>(N, parent, s->is_p.as<uint8_t>(), label_dev,
                                                         s->cl_A.as<int32_t>(), s->cl_Z.as<int32_t>(), counter);
  k4_store_labels_kernel<<<grid_for(N, B), B, 0, s->stream>>>(N, parent);
  s->launches += 2;
  PASTA_CUDA_OK(cudaGetLastError());
  s->clusters_valid = true;
  if (n_clusters_host) {
    unsigned long long h = 0;
    PASTA_CUDA_OK(cudaMemcpyAsync(&h, counter, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
    PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
    *n_clusters_host = (int64_t)h;
  }
  return PASTA_OK;
}

// Composition summary from the per-cluster (A, Z) arrays with exact integer sums:
// counters[2..8) = { #(A=1,Z=0), #heavy, sum A, sum A^2, sum Z, sum Z^2 } over clusters with A >= a_min.
__global__ void k4_composition_kernel(int64_t N, const int32_t* __restrict__ A, const int32_t* __restrict__ Z, int a_min,
                                      unsigned long long* __restrict__ acc) {
  int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= N) return;
  const unsigned long long a = (unsigned long long)A[r], z = (unsigned long long)Z[r];
  if (a == 1 && z == 0) atomicAdd(&acc[0], 1ull);
  if ((int)a >= a_min && a > 0) {
    atomicAdd(&acc[1], 1ull);
    atomicAdd(&acc[2], a);
    atomicAdd(&acc[3], a * a);
    atomicAdd(&acc[4], z);
    atomicAdd(&acc[5], z * z);
  }
}

int k4_composition(Sim* s, int32_t a_min, double* out6_host) {
  unsigned long long* acc = s->counters.as<unsigned long long>() + 2;
  PASTA_CUDA_OK(cudaMemsetAsync(acc, 0, 6 * sizeof(unsigned long long), s->stream));
  k4_composition_kernel<<<grid_for(s->N, 256), 256, 0, s->stream>>>(s->N, s->cl_A.as<int32_t>(), s->cl_Z.as<int32_t>(),
                                                                    a_min, acc);
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  unsigned long long h[6];
  PASTA_CUDA_OK(cudaMemcpyAsync(h, acc, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
  PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  const double nh = (double)h[1];
  out6_host[0] = (double)h[0] / (double)s->N;
  out6_host[1] = nh;
  if (nh > 0) {
    const double mA = (double)h[2] / nh, mZ = (double)h[4] / nh;
    const double vA = (double)h[3] / nh - mA * mA, vZ = (double)h[5] / nh - mZ * mZ;
    out6_host[2] = mA;
    out6_host[3] = sqrt(vA > 0 ? vA : 0);
    out6_host[4] = mZ;
    out6_host[5] = sqrt(vZ > 0 ? vZ : 0);
  } else {
    out6_host[2] = out6_host[3] = out6_host[4] = out6_host[5] = 0.0;
  }
  return PASTA_OK;
}

}  // namespace pasta

// -----------------------------------------------------------------------------------------------------------------
// pasta_clusters_noalloc -- friends-of-friends labels for callers that must not allocate device memory (pasta.h).
//
// Same edges, same predicate, same canonical labels as k4_clusters with r_np == 0; what differs is where the working
// memory lives.  k4_clusters takes its union-find forest (and cell lists) from the simulation's allocator.  Here the
// forest sits in the file-scope array below, which is part of the library image: every GPU on which this module gets
// loaded carries these PASTA_CLUSTERS_NOALLOC_MAX_N * 4 + 256 bytes until the process exits, whether the entry point
// is ever called or not.  That is why the maximum is modest, and why the link step is the all-pairs kernel (it needs
// the forest and nothing else; the cell-list variant would need four more arrays of scratch).
//
//   noalloc_scratch[0 .. MAX_N)   parent[] of the union-find forest
//   noalloc_scratch[MAX_N, +2)    the root counter (one unsigned 64-bit word, 8-byte aligned since MAX_N * 4 % 256 == 0)
//
// The array keeps whatever the previous call left in it, so every call re-initialises the part it uses (parent[i] = i
// for i < N, counter = 0) on the caller's stream before linking.  There is ONE array per GPU: two calls whose kernels
// can overlap on the same GPU (different streams, different host threads) corrupt each other's forest.
// -----------------------------------------------------------------------------------------------------------------
static_assert((PASTA_CLUSTERS_NOALLOC_MAX_N * 4) % 256 == 0, "the root counter must stay 8-byte aligned");
static __device__ __align__(256) int32_t noalloc_scratch[PASTA_CLUSTERS_NOALLOC_MAX_N + 64];

namespace pasta {

__global__ void k4_noalloc_init_kernel(int64_t N, int32_t* __restrict__ parent, unsigned long long* __restrict__ n_roots) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) *n_roots = 0ull;
  if (i < N) parent[i] = (int32_t)i;
}

// The flatten step of k4_flatten_kernel without the (A, Z) histograms, which would be two more scratch arrays.
__global__ void k4_noalloc_labels_kernel(int64_t N, int32_t* __restrict__ parent, int32_t* __restrict__ label_out,
                                         unsigned long long* __restrict__ n_roots) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int r = uf_find(parent, (int)i);
  label_out[i] = r;
  if (r == (int)i) atomicAdd(n_roots, 1ull);
}

// `noalloc_scratch` in HOST code is only a handle for the runtime, not a device address.  The address a kernel can
// use is per device and is asked for once per device, with that device current; it is cached here afterwards.
static const int kNoAllocMaxDevices = 64;
static std::mutex noalloc_mutex;
static int32_t* noalloc_ptr[kNoAllocMaxDevices] = {};

static int noalloc_scratch_on(int device, int32_t** out) {  // `device` is current
  std::lock_guard<std::mutex> lock(noalloc_mutex);
  if (!noalloc_ptr[device]) {
    void* p = nullptr;
    PASTA_CUDA_OK(cudaGetSymbolAddress(&p, noalloc_scratch));
    if (!p) {
      set_error("pasta_clusters_noalloc: cudaGetSymbolAddress returned a null scratch address on device %d", device);
      return PASTA_ECUDA;
    }
    noalloc_ptr[device] = static_cast<int32_t*>(p);
  }
  *out = noalloc_ptr[device];
  return PASTA_OK;
}

}  // namespace pasta

int pasta_clusters_noalloc(const double* x_dev, int64_t N, double L, double r_cl, int32_t* label_dev,
                           int64_t* n_clusters_dev, int32_t device, void* stream) {
  using namespace pasta;
  // every argument is checked before the first CUDA call
  if (N < 0 || N > (int64_t)PASTA_CLUSTERS_NOALLOC_MAX_N) {
    set_error("pasta_clusters_noalloc: N = %lld is outside [0, %d]: the scratch memory of this entry point is a fixed "
              "array of PASTA_CLUSTERS_NOALLOC_MAX_N entries; larger systems need pasta_clusters, which allocates",
              (long long)N, (int)PASTA_CLUSTERS_NOALLOC_MAX_N);
    return PASTA_EINVAL;
  }
  if (N > 0 && (!x_dev || !label_dev)) {
    set_error("pasta_clusters_noalloc: x_dev and label_dev must not be NULL");
    return PASTA_EINVAL;
  }
  if (!(L > 0.0) || !(r_cl > 0.0) || r_cl > 0.5 * L) {
    set_error("pasta_clusters_noalloc: need L > 0 and 0 < r_cl <= L/2");
    return PASTA_EINVAL;
  }
  if (device < 0 || device >= kNoAllocMaxDevices) {
    set_error("pasta_clusters_noalloc: device ordinal %d is outside [0, %d)", (int)device, kNoAllocMaxDevices);
    return PASTA_EINVAL;
  }
  PASTA_CUDA_OK(cudaSetDevice(device));
  int32_t* parent = nullptr;
  PASTA_TRY(noalloc_scratch_on(device, &parent));
  unsigned long long* n_roots = reinterpret_cast<unsigned long long*>(parent + PASTA_CLUSTERS_NOALLOC_MAX_N);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const int B = 256;
  k4_noalloc_init_kernel<<<grid_for(N > 0 ? N : 1, B), B, 0, st>>>(N, parent, n_roots);
  if (N > 0) {
    k4_link_all_kernel<<<grid_for(N, 128), 128, 0, st>>>(N, x_dev, L, 1.0 / L, r_cl * r_cl, parent, nullptr);
    k4_noalloc_labels_kernel<<<grid_for(N, B), B, 0, st>>>(N, parent, label_dev, n_roots);
  }
  PASTA_CUDA_OK(cudaGetLastError());
  if (n_clusters_dev)
    PASTA_CUDA_OK(cudaMemcpyAsync(n_clusters_dev, n_roots, sizeof(int64_t), cudaMemcpyDeviceToDevice, st));
  return PASTA_OK;
}
