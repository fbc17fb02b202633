// K2, production variant -- "chunk" pair-force kernel for sm_100a.
//
// Work decomposition:
//   * a CHUNK is up to T = 8 same-species particles that lie close together, listed in the chunk table that K1
//     builds (k1_cells.cu): in a dense system a short stretch of one row of cells (the force grids are sliced
//     into thin cells along x, so a row -- fixed cy, cz -- is sorted in x), in a sparse one the particles of a
//     small block of cells.  One warp owns one chunk.
//   * SOURCES: for each source species the warp lists the rows of that species' grid that can hold a
//     particle within r_c of the chunk's bounding box, and for every row the tight range of thin cells
//     [lo_x - xr, hi_x + xr]; a range is contiguous in the sorted arrays, i.e. one segment of slots (two
//     where it crosses the periodic boundary: images are enumerated explicitly, there is no per-pair
//     nearest-image arithmetic and small boxes need no special case).  The segments of a pass form one
//     STREAM, consumed 32 positions (a TILE) at a time.
//   * PRODUCER side of a tile: lane l fetches stream position 32 i + l (per-lane cursor into the segment
//     list, plain 16-byte load one tile ahead), shifts it into the chunk's frame and stores it in a
//     double-buffered shared-memory tile.
//   * CONSUMER side: lane = (target pair p, phase h), p = lane / 8, h = lane % 8.  A lane keeps ONE packed
//     pair of targets and their accumulators in registers (96 registers per thread in all, 5 warps per SM
//     sub-partition are resident) and evaluates sources h, h + 8, h + 16, h + 24 of the tile against them
//     with packed FP32 arithmetic (FFMA2/FADD2/FMUL2: two pairs per issued instruction).
//   * There is NO per-candidate test and no divergence: a source that is out of range of a target
//     contributes exactly zero.  The cut-off needs no test for np/nn pairs when sigma^2 r_c^2 > 126:
//     exp2(-r'^2) flushes to exactly zero there (D1: plain truncation; D23).  pp pairs carry the screened
//     Coulomb term and are cut explicitly; small r_c selects the explicitly cut path.
//   * per-lane partial sums are FP32 (a lane sees 1/8 of the chunk's sources); they are combined across
//     the 8 phases and the two passes in FP64 by a transposing butterfly, and written in original order.
#include "k2_chunk.cuh"

namespace pasta {

namespace {

// MINB = resident blocks per SM the registers are budgeted for: K2_MINB (96 registers) where chunks stream hundreds
// of tiles and the arithmetic loop sets the pace; K2_MINB_SPARSE (64 registers, 60 % more warps) where a species is
// sparse, chunks stream a handful of tiles and the latency of the listing does.
template <bool CUT, bool ENERGY, bool STATS, int MINB>
__global__ void __launch_bounds__(WARPS * 32, MINB) k2_chunk_kernel(const ChunkArgs A, const PairConsts c) {
  __shared__ WarpShared shared[WARPS];
  __shared__ __align__(1024) float4 tiles[WARPS][2][32];  // a warp's double buffer: 1024 bytes, 1024-byte aligned
  const int lane = threadIdx.x & 31;
  // the warp index is produced by REDUX so that the compiler can prove it warp-uniform and keep it (and
  // everything derived from it) in uniform registers, off the vector register file
  const int wib = __reduce_or_sync(0xffffffffu, (int)(threadIdx.x >> 5));
  const int pr = lane / NPH;  // this lane's target pair
  // overflow entries first (odd-sized chunks: better at the start of the launch than in its tail), then the
  // primary ones in slot order; the launch covers an upper bound of the number of chunks
  const int widx = blockIdx.x * WARPS + wib, n_over = A.counts[0];
  if (widx >= A.nprim + n_over) return;
  const int chunk = widx < n_over ? A.nprim + widx : widx - n_over;
  WarpShared& sh = shared[wib];

  // ---- targets: lane l < 8 holds the chunk's l-th target (valid ones come first) -----------------------------
  const int slot = lane < T ? __ldg(A.chunk_tab + (int64_t)chunk * T + lane) : -1;
  const unsigned active = __ballot_sync(0xffffffffu, slot >= 0);
  if (active == 0) return;  // empty primary entry
  const int slot0 = __shfl_sync(0xffffffffu, slot, 0);
  if (slot0 < A.slot_lo || slot0 >= A.slot_hi) return;  // another rank's targets (pasta_set_shard)
  const bool chunk_p = slot0 < A.Np;
  const int st_sp = chunk_p ? 0 : 1;
  const SpeciesGrid& gt = A.g[st_sp];
  const int tslot = slot >= 0 ? slot : slot0;
  const float4 tp = __ldg(A.pos4 + tslot);
  const int tc = __ldg(A.cxyz + tslot);

  Accum acc;
  acc.fx = acc.fy = acc.fz = acc.e = make_float2(0.f, 0.f);
  unsigned long long st[3] = {0, 0, 0};

  const unsigned tile_a = (unsigned)__cvta_generic_to_shared(&tiles[wib][0][0]);
  chunk_passes<CUT, ENERGY, STATS, MINB == K2_MINB_SPARSE>(A, c, sh, tile_a, lane, pr, gt, st_sp, chunk_p, tp, tc, active,
                                                           acc, st);

  write_chunk_results<ENERGY>(A, c, acc, lane, slot);
  if (STATS && lane == 0) {
    atomicAdd(A.stats + 0, st[0]);
    atomicAdd(A.stats + 1, st[1]);
    atomicAdd(A.stats + 2, st[2]);
  }
}

}  // namespace

int k2_chunk_forces(Sim* s, bool with_energy, bool stats, double kick) {
  const PairConsts c = make_pair_consts(s->prm);
  const double sigma = sqrt(1.4426950408889634074 / (2.0 * s->prm.Lambda));
  if (s->N >= (1ll << 26)) {
    set_error("the chunk pair kernel packs slot numbers in 26 bits: N must be below 2^26");
    return PASTA_EINVAL;
  }
  ChunkArgs A;
  A.N = (int32_t)s->N;
  A.Np = (int32_t)s->Np;
  A.chunk_tab = s->chunk_tab.as<int32_t>();
  A.counts = s->counters.as<int32_t>() + 2 * 24;
  A.nprim = (int32_t)s->chunk_nprim;
  A.no_coul = s->prm.coulomb_all_pairs ? 1 : 0;
  A.slot_lo = s->shard.slot_lo;
  A.slot_hi = s->shard.slot_hi;
  A.merged = s->grid_sp[0].ncell == s->grid_sp[1].ncell && s->grid_sp[0].ncx == s->grid_sp[1].ncx ? 1 : 0;
  for (int sp = 0; sp < 2; ++sp) {
    const Grid& g = s->grid_sp[sp];
    A.g[sp].ncell = g.ncell;
    A.g[sp].ncx = g.ncx;
    A.g[sp].base = (int32_t)s->bin_base[sp];
    A.g[sp].wS_d = sigma * g.w;
    A.g[sp].wxS_d = sigma * g.wx;
    A.g[sp].wS = (float)A.g[sp].wS_d;
    A.g[sp].inv_wS = (float)(1.0 / A.g[sp].wS_d);
    A.g[sp].wxS = (float)A.g[sp].wxS_d;
    A.g[sp].inv_wxS = (float)(1.0 / A.g[sp].wxS_d);
  }
  A.rcS = (float)(sigma * s->prm.r_c);
  A.rnS = (float)(sigma * (s->prm.r_nuc > 0.0 ? s->prm.r_nuc : s->prm.r_c));
  A.rzeroS = s->prm.skip_exact_zeros ? 11.2472f : 3.0e38f;  // sqrt(126.5): 2^-126.5 is below the FTZ threshold
  A.pos4 = s->pos4.as<float4>();
  A.cxyz = s->cxyz.as<int32_t>();
  A.bin_start = s->bin_start.as<int32_t>();
  A.perm = s->perm.as<int32_t>();
  A.F = s->F.as<double>();
  A.e = s->e.as<double>();
  A.v = s->v.as<double>();
  A.kick = kick;
  A.stats = s->counters.as<unsigned long long>() + 10;
  // exp2(-r'^2) is exactly 0 (FTZ) for r'^2 > 126: then np/nn pairs beyond r_c need no explicit cut
  const bool cut = (double)c.rn2s < 127.0;  // the nuclear cut-off lies inside the FP32 underflow distance
  const int grid = (int)((s->max_chunks + WARPS - 1) / WARPS);
  const dim3 block(WARPS * 32);
  if (stats) PASTA_CUDA_OK(cudaMemsetAsync(A.stats, 0, 3 * sizeof(unsigned long long), s->stream));
#define PASTA_K2_LAUNCH(CUT_, EN_, ST_)                                                                       \
  do {                                                                                                        \
    if (s->chunks_sparse) k2_chunk_kernel<CUT_, EN_, ST_, K2_MINB_SPARSE><<<grid, block, 0, s->stream>>>(A, c); \
    else k2_chunk_kernel<CUT_, EN_, ST_, K2_MINB><<<grid, block, 0, s->stream>>>(A, c);                       \
  } while (0)
  if (stats) {
    if (cut) PASTA_K2_LAUNCH(true, true, true);
    else PASTA_K2_LAUNCH(false, true, true);
  } else if (with_energy) {
    if (cut) PASTA_K2_LAUNCH(true, true, false);
    else PASTA_K2_LAUNCH(false, true, false);
  } else {
    if (cut) PASTA_K2_LAUNCH(true, false, false);
    else PASTA_K2_LAUNCH(false, false, false);
  }
#undef PASTA_K2_LAUNCH
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

}  // namespace pasta
