// K1 -- counting-sort cell list (cubical cells, here rebuilt
// every step on the GPU instead of a halo'd neighbour list on the CPU).
//
// Each species has its own grid (same O3 formula, its own k): grid[0] for protons, grid[1] for neutrons,
// sized so that a cell holds about one chunk (8 particles) of that species -- chunks of the pair kernel
// are then compact for both species.  Layout produced (all in HBM, L2-resident at these sizes):
//   pbin[N]               bin of every particle, original order: base[species] + (cz*ncell + cy)*ncell + cx
//   bin_start[nbins + 1]  exclusive scan over the bins; protons' bins come first, so sorted slots
//                         [0, Np) are protons and [Np, N) neutrons, each sorted by its own grid's cell id
//   perm[N]               sorted slot -> original index, ascending inside a bin (deterministic order)
//   pos4[N]  (float4)     sigma * (x - cell centre) for x, y, z (|.| <= sigma w / 2)  and .w = (float)cx
//   cxyz[N]               cx | cy << 12 | cz << 22
// pasta_cells() exports the species-independent O3 grid of pasta_params.cell_subdiv with the same
// cell_coord arithmetic.
#include <string.h>

#include <chrono>

#include "pasta_internal.cuh"

namespace pasta {

Grid make_grid(double L, double r_c, int32_t k, int32_t xsub) {
  Grid g;
  double q = floor(L * (double)k / r_c);
  if (q < 1.0) q = 1.0;
  if (q > 1023.0) q = 1023.0;  // cy, cz are packed in 10 bits each, cx in 12
  g.ncell = (int32_t)q;
  g.xsub = xsub < 1 ? 1 : xsub;
  while (g.ncell * g.xsub > 4095) g.xsub -= 1;
  g.ncx = g.ncell * g.xsub;
  g.nc3 = (int64_t)g.ncell * g.ncell * g.ncx;
  g.inv_w = (double)g.ncell / L;
  g.w = L / (double)g.ncell;
  g.inv_wx = (double)g.ncx / L;
  g.wx = L / (double)g.ncx;
  return g;
}

__global__ void k1_count_kernel(int64_t N, const double* __restrict__ x, const uint8_t* __restrict__ is_p,
                                const GridPair g, int32_t* __restrict__ pbin, int32_t* __restrict__ bin_count) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const int bin = force_bin(g, is_p[i] ? 0 : 1, x[3 * i + 0], x[3 * i + 1], x[3 * i + 2]);
  pbin[i] = bin;
  atomicAdd(&bin_count[bin], 1);
}

// O3 ids on the exported grid (species-independent), with the histogram for cell_start.
__global__ void k1_o3_kernel(int64_t N, const double* __restrict__ x, double inv_w, int ncell,
                             int32_t* __restrict__ cell_id, int32_t* __restrict__ count) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  int cx = cell_coord(x[3 * i + 0], inv_w, ncell);
  int cy = cell_coord(x[3 * i + 1], inv_w, ncell);
  int cz = cell_coord(x[3 * i + 2], inv_w, ncell);
  const int id = (cz * ncell + cy) * ncell + cx;
  cell_id[i] = id;
  atomicAdd(&count[id], 1);
}

// ---- exclusive scan: 2048 items per block, three small kernels ----------------------------------------
constexpr int SCAN_T = 512, SCAN_ITEMS = 4, SCAN_TILE = SCAN_T * SCAN_ITEMS;

__device__ __forceinline__ int block_exclusive_scan(int v, int* total) {
  __shared__ int warp_sums[SCAN_T / 32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) warp_sums[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int ws = lane < SCAN_T / 32 ? warp_sums[lane] : 0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, ws, o);
      if (lane >= o) ws += t;
    }
    if (lane < SCAN_T / 32) warp_sums[lane] = ws;
  }
  __syncthreads();
  int base = wid > 0 ? warp_sums[wid - 1] : 0;
  *total = warp_sums[SCAN_T / 32 - 1];
  return base + inc - v;
}

__global__ void __launch_bounds__(SCAN_T) scan_local_kernel(const int32_t* __restrict__ in, int32_t* __restrict__ out,
                                                            int64_t n, int32_t* __restrict__ block_sums) {
  const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
  int v[SCAN_ITEMS], s = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    v[k] = (base + k < n) ? in[base + k] : 0;
    s += v[k];
  }
  int total;
  int ex = block_exclusive_scan(s, &total);
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    if (base + k < n) out[base + k] = ex;
    ex += v[k];
  }
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

// Second (and last) launch of the scan: every block sums the totals of the blocks before it (a few hundred
// numbers), adds that to its tile; the last block also writes the grand total to out[n].
__global__ void __launch_bounds__(SCAN_T) scan_add_kernel(int32_t* __restrict__ out, int64_t n,
                                                          const int32_t* __restrict__ block_sums) {
  __shared__ int ws[SCAN_T / 32];
  __shared__ int add_s;
  int part = 0;
  for (int k = threadIdx.x; k < (int)blockIdx.x; k += SCAN_T) part += block_sums[k];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = part;
  __syncthreads();
  if (threadIdx.x == 0) {
    int a = 0;
    for (int k = 0; k < SCAN_T / 32; ++k) a += ws[k];
    add_s = a;
    if (blockIdx.x == gridDim.x - 1) out[n] = a + block_sums[blockIdx.x];
  }
  __syncthreads();
  const int add = add_s;
  const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k)
    if (base + k < n) out[base + k] += add;
}

int scan_exclusive(Sim* s, const int32_t* in, int32_t* out, int64_t n) {
  const int nb = (int)((n + SCAN_TILE - 1) / SCAN_TILE);
  PASTA_TRY(buffer_reserve(s, &s->scan_tmp, sizeof(int32_t) * (size_t)(nb + 1)));
  int32_t* tmp = s->scan_tmp.as<int32_t>();
  scan_local_kernel<<<nb, SCAN_T, 0, s->stream>>>(in, out, n, tmp);
  scan_add_kernel<<<nb, SCAN_T, 0, s->stream>>>(out, n, tmp);
  s->launches += 2;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

__global__ void k1_scatter_kernel(int64_t N, const int32_t* __restrict__ pbin, const int32_t* __restrict__ bin_start,
                                  int32_t* __restrict__ bin_count, int32_t* __restrict__ perm,
                                  int32_t* __restrict__ zero_me) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0 && zero_me) *zero_me = 0;  // the overflow counter of the chunk table (the kernels behind this one add to it)
  if (i >= N) return;
  const int bin = pbin[i];
  const int old = atomicSub(&bin_count[bin], 1);  // leaves the histogram zeroed for the next build
  perm[bin_start[bin] + old - 1] = (int32_t)i;
}

// One thread per bin: order the bin's members by original index, so the sorted order (and with it the
// summation order of the force kernel) does not depend on the atomics' arrival order.
__global__ void k1_order_kernel(int64_t nbins, const int32_t* __restrict__ bin_start, int32_t* __restrict__ perm) {
  int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= nbins) return;
  const int lo = bin_start[b], hi = bin_start[b + 1];
  for (int p = lo + 1; p < hi; ++p) {
    int key = perm[p], q = p - 1;
    while (q >= lo && perm[q] > key) {
      perm[q + 1] = perm[q];
      --q;
    }
    perm[q + 1] = key;
  }
}

// Sorted slot t -> its particle, positions relative to the cell centre, packed cell coordinates.
// FUSED_ORDER: `perm_in` holds the members of every bin in the arrival order of the scatter's atomics; slot t
// takes the member of its bin with exactly (t - first slot of the bin) smaller indices, so the sorted order
// (and with it the summation order of the force kernel) is ascending in the original index whatever the
// arrival order was, and writes it to `perm_out`.  (Thin-cell bins hold a particle or two; the uniform one-grid
// variant, whose bins hold hundreds, orders them with k1_order_kernel instead.)
// list_format (k2_list.cu): pos4.w carries the bits of the packed cell coordinates instead of the thin-cell index as a float.
struct GatherArgs {
  int64_t N;
  const double* x;
  const int32_t* pbin;
  const int32_t* perm_in;
  int32_t* perm_out;
  const int32_t* bin_start;
  GridPair g;
  double sigma;
  float4* pos4;
  int32_t* cxyz;
  bool list_format;
  int32_t* slot_of;
};
__device__ __forceinline__ int packed_cell_of_bin(const GridPair& g, const int bin) {
  const int sp = bin >= g.base[1] ? 1 : 0;
  const int id = bin - g.base[sp], nc = g.ncell[sp], ncx = g.ncx[sp];
  return (id % ncx) | (((id / ncx) % nc) << 12) | ((id / (ncx * nc)) << 22);
}
// Sorted slot t (t < N); returns its packed cell coordinates.
template <bool FUSED_ORDER>
__device__ __forceinline__ int gather_slot(const GatherArgs& G, const int64_t t) {
  int i = G.perm_in[t];
  const int bin = G.pbin[i];
  if (FUSED_ORDER) {
    const int lo = G.bin_start[bin], hi = G.bin_start[bin + 1];
    if (hi - lo > 1) {
      const int want = (int)t - lo;
      for (int a = lo; a < hi; ++a) {
        const int ia = G.perm_in[a];
        int rank = 0;
        for (int b = lo; b < hi; ++b) rank += G.perm_in[b] < ia ? 1 : 0;
        if (rank == want) i = ia;
      }
    }
    G.perm_out[t] = i;
  }
  if (G.slot_of) G.slot_of[i] = (int32_t)t;
  const GridPair& g = G.g;
  const int sp = bin >= g.base[1] ? 1 : 0;
  const int packed = packed_cell_of_bin(g, bin);
  const int cx = PASTA_CX(packed), cy = PASTA_CY(packed), cz = PASTA_CZ(packed);
  const double w = g.w[sp];
  float4 p;
  p.x = (float)(G.sigma * (G.x[3 * i + 0] - ((double)cx + 0.5) * g.wx[sp]));
  p.y = (float)(G.sigma * (G.x[3 * i + 1] - ((double)cy + 0.5) * w));
  p.z = (float)(G.sigma * (G.x[3 * i + 2] - ((double)cz + 0.5) * w));
  p.w = G.list_format ? __int_as_float(packed) : (float)cx;
  G.pos4[t] = p;
  G.cxyz[t] = packed;
  return packed;
}
template <bool FUSED_ORDER>
__global__ void k1_gather_kernel(const GatherArgs G) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t < G.N) gather_slot<FUSED_ORDER>(G, t);
}

// Chunk table of the pair kernel.  A chunk = the targets of one warp = up to CHUNK_T sorted slots of one species
// that are close together; an entry of the table lists its slots (-1 = none).  Two builders, chosen per species
// by the mean number of particles per cell:
//   DENSE  (row runs): NOMINAL chunks are the stretches [row start + 8 k, row start + 8 k + 8) of every row
//          (a chunk never straddles two rows: the two parts would be a cell width apart in y or z and on
//          opposite faces in x); a nominal chunk is cut further, greedily, wherever its extent reaches xmax thin
//          cells (in a dense system: never).  One thread handles the nominal chunks that START in the slots
//          [8 j, 8 j + 8): it needs the cell coordinates of 16 slots and the first slot of the row of slot 8 j.
//          Entry j of the table is the first chunk it finds (so neighbouring warps of the pair kernel work on
//          neighbouring chunks of a row and share their sources in L1; it may be empty), further ones go to the
//          overflow region.
//   SPARSE (blocks): 8 consecutive particles of a row would be far apart, so the particles of a block of B x B x B
//          cells (B w <= 20 fm) are grouped instead, 8 at a time; one thread per block, entries in the overflow
//          region, reserved once per warp.
constexpr int CHUNK_T = PASTA_CHUNK_T;
struct ChunkGeom {
  int xmax[2];   // DENSE: extent limit of a chunk in thin cells
  int block[2];  // 0 = DENSE, else B of the SPARSE builder
  int nprim;     // primary entries
};

__device__ __forceinline__ void write_entry(int32_t* __restrict__ tab, int64_t e, int first, int n,
                                            int32_t* __restrict__ chunk_first) {
  for (int k = 0; k < n; ++k) chunk_first[first + k] = first;
#pragma unroll
  for (int k = 0; k < CHUNK_T; k += 4) {
    int4 a;
    a.x = n > k ? first + k : -1;
    a.y = n > k + 1 ? first + k + 1 : -1;
    a.z = n > k + 2 ? first + k + 2 : -1;
    a.w = n > k + 3 ? first + k + 3 : -1;
    reinterpret_cast<int4*>(tab + e * CHUNK_T)[k / 4] = a;
  }
}

// Entry j of the DENSE builder; cell_of(p) = packed cell coordinates of sorted slot p (p < N).
template <class CellOf>
__device__ __forceinline__ void chunk_rows_entry(const int j, const int32_t N, const int32_t Np, CellOf cell_of,
                                                 const int32_t* __restrict__ bin_start, const GridPair& g,
                                                 const ChunkGeom& cg, int32_t* __restrict__ chunk_tab,
                                                 int32_t* __restrict__ n_overflow, int32_t* __restrict__ chunk_first) {
  const int lo = j * CHUNK_T;
  if (lo >= N) return;
  // row key of a slot: species and (cy, cz); -1 beyond the end
  int c[2 * CHUNK_T], key[2 * CHUNK_T];
#pragma unroll
  for (int k = 0; k < 2 * CHUNK_T; ++k) {
    const int p = lo + k;
    c[k] = p < N ? cell_of(p) : 0;
    key[k] = p < N ? ((c[k] >> 12) | (p < Np ? 0 : (1 << 24))) : -1;
  }
  // first slot of the row that slot `lo` belongs to
  const int sp0 = lo < Np ? 0 : 1;
  int row_lo = __ldg(bin_start + g.base[sp0] + (PASTA_CZ(c[0]) * g.ncell[sp0] + PASTA_CY(c[0])) * g.ncx[sp0]);
  // up to 2 * CHUNK_T - 1 pieces: a chunk can start at each of the 8 slots (row changes), and the nominal chunk
  // that starts at the last one can be cut at the extent limit into up to 8 more
  int first_slot[2 * CHUNK_T], count[2 * CHUNK_T];
  int m = 0;
#pragma unroll
  for (int k = 0; k < CHUNK_T; ++k) {
    if (key[k] < 0) break;
    if (k > 0 && key[k] != key[k - 1]) row_lo = lo + k;  // sorted: the first slot with a new key starts its row
    if (((lo + k - row_lo) & (CHUNK_T - 1)) != 0) continue;
    const int sp = (key[k] >> 24) & 1;
    if (cg.block[sp] != 0) continue;  // this species is grouped by blocks
    // nominal chunk [lo + k, lo + k + 8) within the row; cut it where the extent limit is reached
    const int xm = cg.xmax[sp];
    int first = k;
#pragma unroll
    for (int q = 1; q <= CHUNK_T; ++q) {
      const bool end = q == CHUNK_T || key[k + q] != key[k];
      if (end || PASTA_CX(c[k + q]) - PASTA_CX(c[first]) >= xm) {
        first_slot[m] = lo + first;
        count[m++] = k + q - first;
        first = k + q;
      }
      if (end) break;
    }
  }
  write_entry(chunk_tab, j, m > 0 ? first_slot[0] : 0, m > 0 ? count[0] : 0, chunk_first);
  if (m > 1) {
    const int at = cg.nprim + atomicAdd(n_overflow, m - 1);
    for (int k = 1; k < m; ++k) write_entry(chunk_tab, at + k - 1, first_slot[k], count[k], chunk_first);
  }
}

// The gather and the DENSE chunk builder in one launch: a block gathers 256 sorted slots, keeps their packed cell
// coordinates in shared memory together with those of the 16 slots behind them (their bins are known from the scatter,
// whatever the order inside a bin will be), and its first 32 threads then write the 32 table entries of these slots.
constexpr int GATHER_T = 256;
__global__ void __launch_bounds__(GATHER_T) k1_gather_chunks_kernel(const GatherArgs G, const int32_t Np, const ChunkGeom cg,
                                                                    int32_t* __restrict__ chunk_tab,
                                                                    int32_t* __restrict__ n_overflow,
                                                                    int32_t* __restrict__ chunk_first) {
  __shared__ int cell[GATHER_T + 2 * CHUNK_T];
  const int64_t base = (int64_t)blockIdx.x * GATHER_T, t = base + threadIdx.x;
  if (t < G.N) cell[threadIdx.x] = gather_slot<true>(G, t);
  if (threadIdx.x < 2 * CHUNK_T) {
    const int64_t u = base + GATHER_T + threadIdx.x;
    if (u < G.N) cell[GATHER_T + threadIdx.x] = packed_cell_of_bin(G.g, G.pbin[G.perm_in[u]]);
  }
  __syncthreads();
  if (threadIdx.x < GATHER_T / CHUNK_T) {
    const int j = blockIdx.x * (GATHER_T / CHUNK_T) + threadIdx.x;
    chunk_rows_entry(j, (int32_t)G.N, Np, [&](int p) { return cell[p - (int)base]; }, G.bin_start, G.g, cg, chunk_tab,
                     n_overflow, chunk_first);
  }
}

__global__ void k1_chunk_blocks_kernel(int sp, const int32_t* __restrict__ bin_start, const GridPair g,
                                       const ChunkGeom cg, int32_t* __restrict__ chunk_tab,
                                       int32_t* __restrict__ n_overflow, int32_t* __restrict__ chunk_first) {
  const int B = cg.block[sp], nc = g.ncell[sp], ncx = g.ncx[sp], xs = ncx / nc;
  const int nb = (nc + B - 1) / B;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = t < nb * nb * nb;
  const int bx = t % nb, by = (t / nb) % nb, bz = t / (nb * nb);
  const int x0 = bx * B * xs, x1 = min(x0 + B * xs, ncx);
  int total = 0;
  if (live)
    for (int cz = bz * B; cz < min(bz * B + B, nc); ++cz)
      for (int cy = by * B; cy < min(by * B + B, nc); ++cy) {
        const int32_t* bs = bin_start + g.base[sp] + (cz * nc + cy) * ncx;
        total += __ldg(bs + x1) - __ldg(bs + x0);
      }
  const int m = (total + CHUNK_T - 1) / CHUNK_T;
  // one reservation per warp
  const int lane = threadIdx.x & 31;
  int incl = m;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  const int wtotal = __shfl_sync(0xffffffffu, incl, 31);
  int at = 0;
  if (lane == 0 && wtotal > 0) at = atomicAdd(n_overflow, wtotal);
  at = cg.nprim + __shfl_sync(0xffffffffu, at, 0) + incl - m;
  if (m == 0) return;
  int32_t* out = chunk_tab + (int64_t)at * CHUNK_T;
  int k = 0;
  for (int cz = bz * B; cz < min(bz * B + B, nc); ++cz)
    for (int cy = by * B; cy < min(by * B + B, nc); ++cy) {
      const int32_t* bs = bin_start + g.base[sp] + (cz * nc + cy) * ncx;
      const int hi = __ldg(bs + x1);
      for (int p = __ldg(bs + x0); p < hi; ++p) out[k++] = p;
    }
  const int n_real = k;
  for (; k < m * CHUNK_T; ++k) out[k] = -1;
  for (k = 0; k < n_real; ++k) chunk_first[out[k]] = out[k - (k % CHUNK_T)];
}

// Cells per side of a species' grid: the O3 formula with the k that puts about CHUNK particles in a cell.
#ifndef PASTA_WMAX
#define PASTA_WMAX 8.0
#endif
static int auto_subdiv(double L, double r_c, int64_t n_species, int k_default) {
  if (n_species <= 0) return k_default;
  const double w_star = L * cbrt((double)PASTA_CHUNK_T / (double)n_species);
  int k = (int)floor(r_c / w_star + 0.5);
  // never wider than 8 fm: sorted coordinates are FP32 offsets from the cell centre, and their quantum
  // (2^-24 of the half width) times the steepest pair-force gradient (~80 MeV/fm^2 inside a cluster) has to
  // stay below the force tolerance
  const int k_min = (int)ceil(r_c / PASTA_WMAX);
  k = k < k_min ? k_min : k;
  return k < 1 ? 1 : (k > 64 ? 64 : k);
}

// Thin cells along x per cell: 8 where the species is dense; fewer where the grid would otherwise have many more
// bins than the species has particles (a sparse species: the bin tables, not the particles, would set the cost).
static int auto_xsub(double L, double r_c, int k, int64_t n_species) {
  const double ncell = floor(L * (double)k / r_c);
  int xsub = 8;
  while (xsub > 1 && ncell * ncell * ncell * xsub > 4.0 * (double)n_species + 65536.0) xsub /= 2;
  return xsub;
}

// ---- list mode (k2_list.cu) -------------------------------------------------------------------------------------------
// One grid for both species, cells as wide as the precision cap allows, no thin cells: rows are only listed when the
// lists are built.
static int list_subdiv(const Sim* s) { return (int)ceil(s->prm.r_c / PASTA_WMAX); }

// The paper's delta_r is 4 fm for a CPU list; here a rebuild costs ten force evaluations and a list entry
// little, and 6 fm measured best at the dilute ends of configs 3 and 5 (profiles/).
double list_halo(const Sim* s) { return s->prm.list_halo > 0.0 ? s->prm.list_halo : 6.0; }

// Lists pay where both species are sparse on that grid (fewer than 3 per cell: the regime of the SPARSE chunk
// builder), i.e. the cold dilute end of a decompression (rebuilt every ~100 steps there); and the box
// must be wide enough for cell offsets to have one nearest image within reach + halo of a chunk.
bool list_mode_wanted(const Sim* s) {
  if (!s->prm.list_reuse || s->tune.force_variant != 0 || s->no_lists) return false;
  if (s->L < 2.0 * (s->prm.r_c + list_halo(s)) + 6.0 * PASTA_WMAX) return false;
  if (s->N > (1 << 20)) return false;  // a list entry packs the sorted slot in 20 bits ...
  const Grid g = make_grid(s->L, s->prm.r_c, list_subdiv(s), 1);
  if (g.ncell < 4) return false;
  if (ceil((s->prm.r_c + list_halo(s)) / g.w + 1e-3) > 7.0) return false;  // ... and a cell offset in 4 signed bits
  const double n_max = (double)(s->Np > s->N - s->Np ? s->Np : s->N - s->Np);
  return n_max / ((double)g.ncell * g.ncell * g.ncell) < 3.0;
}

static void fill_grid_pair(const Grid gr[2], GridPair* gp) {
  GridPair& g = *gp;
  for (int sp = 0; sp < 2; ++sp) {
    g.ncell[sp] = gr[sp].ncell;
    g.ncx[sp] = gr[sp].ncx;
    g.inv_w[sp] = gr[sp].inv_w;
    g.w[sp] = gr[sp].w;
    g.inv_wx[sp] = gr[sp].inv_wx;
    g.wx[sp] = gr[sp].wx;
  }
  g.base[0] = 0;
  g.base[1] = (int)gr[0].nc3;
}

// The frozen cell counts of s->grid_sp with the widths of the current box side (the grid scales with the box).
void k1_frozen_grids(Sim* s, GridPair* gp) {
  for (int sp = 0; sp < 2; ++sp) {
    Grid& g = s->grid_sp[sp];
    g.inv_w = (double)g.ncell / s->L;
    g.w = s->L / (double)g.ncell;
    g.inv_wx = (double)g.ncx / s->L;
    g.wx = s->L / (double)g.ncx;
  }
  fill_grid_pair(s->grid_sp, gp);
}

// Grids of the two species for the current box (host arithmetic only).
void k1_grids(const Sim* s, bool uniform_grid, Grid out[2], GridPair* gp) {
  const int64_t N = s->N;
  // the reference kernel and the pair counter walk ONE isotropic grid; the chunk kernel takes a grid per
  // species, each cell sliced into thin cells along x (rows sorted in x: tight source ranges, compact chunks)
  const bool uniform = uniform_grid || s->tune.force_variant == 1;
  const bool lists = !uniform && list_mode_wanted(s);
  const bool same_k = uniform || s->tune.auto_grid == 0;
  const int k0 = lists ? list_subdiv(s) : same_k ? s->prm.cell_subdiv : auto_subdiv(s->L, s->prm.r_c, s->Np, s->prm.cell_subdiv);
  const int k1 = lists ? list_subdiv(s) : same_k ? s->prm.cell_subdiv : auto_subdiv(s->L, s->prm.r_c, N - s->Np, s->prm.cell_subdiv);
  const int xs0 = uniform || lists ? 1 : (s->tune.x_subdiv > 0 ? s->tune.x_subdiv : auto_xsub(s->L, s->prm.r_c, k0, s->Np));
  const int xs1 = uniform || lists ? 1 : (s->tune.x_subdiv > 0 ? s->tune.x_subdiv : auto_xsub(s->L, s->prm.r_c, k1, N - s->Np));
  out[0] = make_grid(s->L, s->prm.r_c, k0, xs0);
  out[1] = make_grid(s->L, s->prm.r_c, k1, xs1);
  fill_grid_pair(out, gp);
}

// The grids, the buffers, and a zeroed histogram.  (The scatter kernel counts the histogram back down to zero, so the
// memset is needed only when the table grows or somebody else used it.)
int k1_setup(Sim* s, bool uniform_grid, GridPair* gp) {
  const int64_t N = s->N;
  s->list.valid = false;  // whoever sets the grids up again is about to re-sort
  k1_grids(s, uniform_grid, s->grid_sp, gp);
  s->bin_base[0] = 0;
  s->bin_base[1] = s->grid_sp[0].nc3;
  const int64_t nbins = s->grid_sp[0].nc3 + s->grid_sp[1].nc3;
  const void* before = s->bin_count.ptr;
  PASTA_TRY(buffer_reserve(s, &s->bin_count, sizeof(int32_t) * (size_t)(nbins + 1)));
  PASTA_TRY(buffer_reserve(s, &s->bin_start, sizeof(int32_t) * (size_t)(nbins + 1)));
  PASTA_TRY(buffer_reserve(s, &s->perm_raw, sizeof(int32_t) * (size_t)N));
  if (s->bin_count.ptr != before) s->bins_zeroed = 0;
  if (s->bins_zeroed < nbins + 1) {
    PASTA_CUDA_OK(cudaMemsetAsync(s->bin_count.ptr, 0, s->bin_count.bytes, s->stream));
    s->bins_zeroed = (int64_t)(s->bin_count.bytes / sizeof(int32_t));
  }
  return PASTA_OK;
}

int k1_build(Sim* s, bool uniform_grid) {
  const int64_t N = s->N;
  const bool uniform = uniform_grid || s->tune.force_variant == 1;
  const bool lists = !uniform && list_mode_wanted(s);  // per-target neighbour lists follow: no chunk table
  GridPair g;
  const int B = 256;
  if (!(s->hist_valid && s->hist_uniform == uniform)) {
    if (s->hist_valid) s->bins_zeroed = 0;  // a histogram for the other kind of grid is sitting in the table
    PASTA_TRY(k1_setup(s, uniform_grid, &g));
    k1_count_kernel<<<grid_for(N, B), B, 0, s->stream>>>(N, s->x.as<double>(), s->is_p.as<uint8_t>(), g,
                                                         s->cell_id.as<int32_t>(), s->bin_count.as<int32_t>());
    s->launches += 1;
  } else {
    PASTA_TRY(k1_setup(s, uniform_grid, &g));  // same L, same grids: recomputes g, allocates and zeroes nothing
  }
  s->hist_valid = false;
  const int64_t nbins = s->grid_sp[0].nc3 + s->grid_sp[1].nc3;
  int32_t* cnt = s->bin_count.as<int32_t>();
  int32_t* start = s->bin_start.as<int32_t>();
  PASTA_TRY(scan_exclusive(s, cnt, start, nbins));
  const double sigma = sqrt(1.4426950408889634074 / (2.0 * s->prm.Lambda));
  int32_t* n_overflow = s->counters.as<int32_t>() + 2 * 24;
  GatherArgs G;
  G.N = N;
  G.x = s->x.as<double>();
  G.pbin = s->cell_id.as<int32_t>();
  G.bin_start = start;
  G.g = g;
  G.sigma = sigma;
  G.pos4 = s->pos4.as<float4>();
  G.cxyz = s->cxyz.as<int32_t>();
  G.list_format = lists;
  G.slot_of = nullptr;
  if (uniform) {
    G.perm_in = s->perm.as<int32_t>();
    G.perm_out = nullptr;
    k1_scatter_kernel<<<grid_for(N, B), B, 0, s->stream>>>(N, G.pbin, start, cnt, s->perm.as<int32_t>(), nullptr);
    k1_order_kernel<<<grid_for(nbins, B), B, 0, s->stream>>>(nbins, start, s->perm.as<int32_t>());
    k1_gather_kernel<false><<<grid_for(N, B), B, 0, s->stream>>>(G);
    s->launches += 3;
  } else {
    G.perm_in = s->perm_raw.as<int32_t>();
    G.perm_out = s->perm.as<int32_t>();
    // the chunk table of the pair kernel (not in list mode): builder per species (DENSE row runs: at least 3
    // particles per cell on average), the extent limit of a row run (three cell widths, at most 16 fm) and the
    // capacity of the table: a bound on the number of chunks
    //   row runs: primary entries ceil(N / 8); overflow <= one per row (row or species change inside 8 slots)
    //             + ncx / xmax + 1 per row (runs cut at the extent limit cover disjoint stretches >= xmax)
    //   blocks:   n / 8 + one per block
    ChunkGeom cg;
    cg.nprim = 0;
    int64_t overflow = 64;
    bool any_rows = false;
    for (int sp = 0; sp < 2; ++sp) {
      const Grid& gr = s->grid_sp[sp];
      const int64_t n_sp = sp == 0 ? s->Np : N - s->Np;
      const double occ = (double)n_sp / ((double)gr.ncell * gr.ncell * gr.ncell);
      int xm = (int)floor(fmin(3.0 * gr.w, 16.0) / gr.wx);
      cg.xmax[sp] = xm < 1 ? 1 : xm;
      cg.block[sp] = 0;
      if (occ < 3.0 && gr.ncell >= 4) {
        int Bb = (int)ceil(cbrt(8.0 / fmax(occ, 1e-9)));
        const int Bmax = (int)floor(20.0 / gr.w);
        Bb = Bb > 3 ? 3 : Bb;
        Bb = Bb > Bmax ? Bmax : Bb;
        cg.block[sp] = Bb < 1 ? 1 : Bb;
      }
      const int64_t nrow = (int64_t)gr.ncell * gr.ncell;
      if (cg.block[sp] == 0) {
        any_rows = any_rows || n_sp > 0;
        overflow += nrow * (gr.ncx / cg.xmax[sp] + 2);
      } else {
        const int64_t nb = (gr.ncell + cg.block[sp] - 1) / cg.block[sp];
        overflow += n_sp / CHUNK_T + nb * nb * nb;
      }
    }
    if (lists) {
      PASTA_TRY(buffer_reserve(s, &s->slot_of, sizeof(int32_t) * (size_t)N));
      G.slot_of = s->slot_of.as<int32_t>();
    } else {
      cg.nprim = any_rows ? (int)((N + CHUNK_T - 1) / CHUNK_T) : 0;
      s->chunks_sparse = (cg.block[0] != 0 && s->Np > 0) || (cg.block[1] != 0 && N - s->Np > 0);
      s->chunk_nprim = cg.nprim;
      s->max_chunks = cg.nprim + overflow;
      PASTA_TRY(buffer_reserve(s, &s->chunk_tab, sizeof(int32_t) * CHUNK_T * (size_t)(s->max_chunks + 8)));
      PASTA_TRY(buffer_reserve(s, &s->chunk_first, sizeof(int32_t) * (size_t)N));
    }
    k1_scatter_kernel<<<grid_for(N, B), B, 0, s->stream>>>(N, G.pbin, start, cnt, s->perm_raw.as<int32_t>(), n_overflow);
    s->launches += 1;
    if (!lists && any_rows) {
      // gather + the DENSE builder's table entries in one launch
      k1_gather_chunks_kernel<<<grid_for(N, GATHER_T), GATHER_T, 0, s->stream>>>(
          G, (int32_t)s->Np, cg, s->chunk_tab.as<int32_t>(), n_overflow, s->chunk_first.as<int32_t>());
    } else {
      k1_gather_kernel<true><<<grid_for(N, B), B, 0, s->stream>>>(G);
    }
    s->launches += 1;
    if (!lists) {
      for (int sp = 0; sp < 2; ++sp)
        if (cg.block[sp] != 0 && (sp == 0 ? s->Np : N - s->Np) > 0) {
          const int64_t nb = (s->grid_sp[sp].ncell + cg.block[sp] - 1) / cg.block[sp];
          k1_chunk_blocks_kernel<<<grid_for(nb * nb * nb, 128), 128, 0, s->stream>>>(
              sp, start, g, cg, s->chunk_tab.as<int32_t>(), n_overflow, s->chunk_first.as<int32_t>());
          s->launches += 1;
        }
    }
  }
  s->sort_kind = uniform ? 1 : (lists ? 2 : 0);
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

// ---- list mode: the frozen sorted order, refreshed ----------------------------------------------------------------------
// Sorted slot t keeps its particle perm[t] and its cell cxyz[t] from the last build; the particle has moved (and the
// grid has scaled with the box), so pos4[t] = sigma * (x - centre of that cell) in the nearest image -- the arithmetic
// of k1_gather_kernel, which it reproduces bit for bit for a particle that is still inside its cell.  With it, the
// trigger of the paper's neighbour list: the largest displacement since the build, measured in
// co-moving coordinates u = x / L (a uniform scaling of the box moves nothing) and expressed at the build's box side.
// The last block to finish posts {seq, max displacement^2} to the host's mailbox and re-arms the scratch words.
__global__ void __launch_bounds__(256) k1_refresh_kernel(int32_t N, const double* __restrict__ x,
                                                         const int32_t* __restrict__ perm, const RefreshArgs R) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  float d2 = 0.f;
  if (t < N) {
    const int64_t i = perm[t];
    const double xi[3] = {x[3 * i + 0], x[3 * i + 1], x[3 * i + 2]};
    d2 = refresh_slot(R, t, i, xi);
  }
  refresh_post(R, d2);
}

void k1_refresh_args(Sim* s, RefreshArgs* out) {
  RefreshArgs& R = *out;
  k1_frozen_grids(s, &R.g);
  R.xref = s->xref.as<double>();
  R.cxyz = s->cxyz.as<int32_t>();
  R.pos4 = s->pos4.as<float4>();
  R.Np = (int32_t)s->Np;
  R.sigma = sqrt(1.4426950408889634074 / (2.0 * s->prm.Lambda));
  R.L = s->L;
  R.invL = 1.0 / s->L;
  R.L0 = s->list.L0;
  R.invL0 = 1.0 / s->list.L0;
  R.scratch = s->counters.as<unsigned>() + 2 * 28;  // counters[28]: {max bits, ticket}
  R.mbox = s->list.mbox_dev;
  R.seq = ++s->list.seq;
  {
    const double ratio = s->L / s->list.L0;
    R.delta = s->list.halo + (ratio >= 1.0 ? 0.0 : s->prm.r_c * (1.0 - 1.0 / ratio));
  }
  R.gate = s->counters.as<unsigned>() + 2 * 31;  // counters[31]
}

// The host decides whether the lists survive this step: wait for the post of the refresh (a few microseconds after
// the kernel ends).
int k1_refresh_wait(Sim* s, double* max_disp_host) {
  const unsigned seq = s->list.seq;
  s->list.pending = false;
  const auto t0 = std::chrono::steady_clock::now();
  unsigned long long m;
  int spins = 0;
  while ((unsigned)((m = *s->list.mbox_host) >> 32) != seq) {
    if ((++spins & 0xfff) == 0 && std::chrono::steady_clock::now() - t0 > std::chrono::seconds(20)) {
      PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
      if ((unsigned)((m = *s->list.mbox_host) >> 32) != seq) {
        set_error("k1_refresh: the displacement readback never arrived");
        return PASTA_ECUDA;
      }
    }
  }
  float f;
  const unsigned bits = (unsigned)(m & 0xffffffffu);
  memcpy(&f, &bits, sizeof(f));
  *max_disp_host = sqrt((double)f);
  return PASTA_OK;
}

int k1_refresh(Sim* s, double* max_disp_host) {
  RefreshArgs R;
  k1_refresh_args(s, &R);
  k1_refresh_kernel<<<grid_for(s->N, 256), 256, 0, s->stream>>>((int32_t)s->N, s->x.as<double>(), s->perm.as<int32_t>(), R);
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  return k1_refresh_wait(s, max_disp_host);
}

// pasta_cells: the O3 grid of cell_subdiv, species-independent (uses the cell-list scratch buffers; the next
// force evaluation rebuilds them anyway).
int k1_export_cells(Sim* s, int32_t* cell_id_dev, int32_t* cell_start_dev) {
  const Grid g = make_grid(s->L, s->prm.r_c, s->prm.cell_subdiv);
  s->hist_valid = false;  // cell_id and the histogram table are about to hold the exported grid
  s->bins_zeroed = 0;
  s->sort_kind = -1;
  s->list.valid = false;  // reused neighbour lists go with the sort they were built on (their consumers check sort_kind)
  PASTA_TRY(buffer_reserve(s, &s->bin_count, sizeof(int32_t) * (size_t)(g.nc3 + 1)));
  PASTA_TRY(buffer_reserve(s, &s->bin_start, sizeof(int32_t) * (size_t)(g.nc3 + 1)));
  int32_t* cnt = s->bin_count.as<int32_t>();
  PASTA_CUDA_OK(cudaMemsetAsync(cnt, 0, sizeof(int32_t) * (size_t)(g.nc3 + 1), s->stream));
  k1_o3_kernel<<<grid_for(s->N, 256), 256, 0, s->stream>>>(s->N, s->x.as<double>(), g.inv_w, g.ncell,
                                                           s->cell_id.as<int32_t>(), cnt);
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  if (cell_id_dev)
    PASTA_CUDA_OK(cudaMemcpyAsync(cell_id_dev, s->cell_id.ptr, sizeof(int32_t) * (size_t)s->N,
                                  cudaMemcpyDeviceToDevice, s->stream));
  if (cell_start_dev) {
    PASTA_TRY(scan_exclusive(s, cnt, s->bin_start.as<int32_t>(), g.nc3));
    PASTA_CUDA_OK(cudaMemcpyAsync(cell_start_dev, s->bin_start.ptr, sizeof(int32_t) * (size_t)(g.nc3 + 1),
                                  cudaMemcpyDeviceToDevice, s->stream));
  }
  return PASTA_OK;
}

}  // namespace pasta
