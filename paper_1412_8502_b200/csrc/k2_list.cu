// K2 with a reused neighbour list -- the paper's own scheme for the nuclear force (a list per target of
// the sources within r + delta_r, "so it does not have to be rebuilt every time step"; rebuilt when the distance a
// target has moved plus the largest distance any source has moved exceeds delta_r; built from a cell
// grid), applied where it pays: the cold, dilute end of the decompression runs, where a target has a few dozen
// sources in range and the chunk kernel of k2_chunk.cu would spend its time listing rows and evaluating empty tiles.
//
//   * A rebuild step sorts the particles (K1, one common grid for both species) and then k2_tlist_build_kernel
//     makes, for every target, two lists of sorted slots: the proton and the neutron sources within reach + halo
//     (reach = r_c for proton-proton pairs -- Coulomb -- and the nuclear reach otherwise).  8 lanes work on a
//     target: they share the rows of cells within range, walk the tight x range of every row, count, reserve a
//     contiguous stretch of the pool with one atomicAdd, and walk again to fill it.
//   * Until the next rebuild the sorted order, the cells the coordinates are relative to and the lists are FROZEN;
//     k1_refresh_kernel (k1_cells.cu) re-expresses the moved positions relative to their frozen cells every step and
//     measures the largest displacement since the rebuild (the trigger).
//   * k2_tlist_kernel evaluates the lists: 8 lanes per target split its sources ("j-split"), FP32 pair arithmetic on
//     per-pair cell-relative displacements, partial sums combined in FP64 by shuffles.  A listed source that is out
//     of range contributes exactly zero (np/nn: exp2 underflow or the explicit nuclear cut; pp: explicit cut at r_c),
//     so F and e are those of the plain evaluation (D1, D23).
#include "pasta_internal.cuh"

namespace pasta {

namespace {

constexpr int GL = 8;  // lanes per target

__device__ __forceinline__ float ex2_ftz(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqrt_ftz(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

struct TListArgs {
  int32_t N, Np;
  const unsigned* gate;     // != NULL: evaluate only if *gate != 0 (the refresh enqueued before this kernel lets the lists live)
  double* v;                // kick != 0: the second half kick v += kick F rides along (O2 step 4)
  double kick;
  int32_t no_coul;          // coulomb_all_pairs: the Coulomb term is summed elsewhere (k2_coulomb.cu)
  int32_t slot_lo, slot_hi; // target sharding: the force kernel evaluates the targets in sorted slots [slot_lo, slot_hi)
  int32_t ncell, ncx;       // ONE grid geometry for both species (list mode)
  int32_t base[2];          // first bin of each species
  float wS, wxS;            // sigma * cell width (y, z) and (x)
  float rcS, nucS, haloS;   // sigma * r_c, sigma * reach of the nuclear terms, sigma * halo
  const float4* pos4;       // sorted; .w = bits of cx | cy << 12 | cz << 22 (list format)
  const int32_t* bin_start;
  const int32_t* perm;
  int4* tl;                 // per target: {first entry of the proton list, its length, first of the neutron list, its length}
  int32_t* pool;            // entries: sorted slots
  int64_t pool_cap;
  unsigned long long* cursor;  // pool entries reserved so far (keeps counting past pool_cap: the size a retry needs)
  double* F;
  double* e;
};

// A list entry: sorted slot of the source (20 bits) and its cell offset from the target's cell in the nearest image,
// 4 signed bits per axis -- frozen with the list, so the force kernel needs no nearest-image arithmetic.
constexpr int SLOT_BITS = 20;
__device__ __forceinline__ int pack_entry(int slot, int mx, int my, int mz) {
  return slot | ((mx & 15) << 20) | ((my & 15) << 24) | ((mz & 15) << 28);
}

// ---- list building -----------------------------------------------------------------------------------------------------
// 8 lanes build the two lists of one target (sorted slot t) in three phases:
//   1. SEGMENTS.  The lanes share the (2 mr + 1)^2 rows of cells around the target's row; in every row the tight
//      range of cells that can hold a source within reach is, per source species, a stretch of sorted slots (two
//      where it crosses the periodic boundary).  The non-empty stretches are appended to the group's segment list in
//      shared memory: their concatenation is the target's CANDIDATE STREAM.
//   2. COUNT + STAGE.  The lanes stride over the stream (a per-lane cursor walks the segment list), test every
//      candidate against the reach, count the proton and neutron sources kept and stage the entries in shared memory
//      (protons from the front, neutrons from the back); lane 0 then reserves a contiguous stretch of the pool for
//      both lists with one atomicAdd and the lanes copy the staged entries out.
//   3. FILL.  Only for a target whose lists do not fit the stage (a target inside a fragment): the same pass again
//      (the candidates are cache-hot), writing the entries straight to the pool in the same stream order.
// A target with more segments than the list holds (never in the dilute regime lists are used in) makes the kernel
// report failure through the cursor's top bit; the host then falls back to rebuilding every step.
constexpr int SEG_CAP = 160;            // segments per target
constexpr int STG = 128;                // staged entries per target
constexpr int BUILD_T = 256;            // threads per block: 32 targets
constexpr unsigned long long LIST_FAIL = 1ull << 62;

struct Seg {
  int start_len;  // first sorted slot (20 bits) | number of slots << 20 (12 bits)
  int where;      // (my + 8) | (mz + 8) << 4 | source species << 8 | periodic part (0: none, 1: from below, 2: from above) << 9
};

__global__ void __launch_bounds__(BUILD_T) k2_tlist_build_kernel(const TListArgs A) {
  extern __shared__ Seg seg_all[];  // [BUILD_T / GL][SEG_CAP], then int32 [BUILD_T / GL][STG]
  const int grp = threadIdx.x / GL, h = threadIdx.x & (GL - 1);
  const int gt = blockIdx.x * (BUILD_T / GL) + grp;  // target = sorted slot
  const bool valid = gt < A.N;
  const int t = valid ? gt : A.N - 1;
  Seg* const seg = seg_all + grp * SEG_CAP;
  int32_t* const stage = reinterpret_cast<int32_t*>(seg_all + (BUILD_T / GL) * SEG_CAP) + grp * STG;
  const unsigned gmask = 0xffu << (threadIdx.x & 24);   // this group's lanes within the warp
  const unsigned lower = gmask & ((1u << (threadIdx.x & 31)) - 1u);
  const float4 tq = __ldg(A.pos4 + t);
  const int tc = __float_as_int(tq.w);
  const int cx = PASTA_CX(tc), cy = PASTA_CY(tc), cz = PASTA_CZ(tc);
  const bool tp = t < A.Np;
  const float R[2] = {(tp ? A.rcS : A.nucS) + A.haloS, A.nucS + A.haloS};   // reach for proton / neutron sources
  const float slack = 1.0e-3f * A.wS;  // ranges of rows and cells: slack against FP32 rounding at cell faces
  const float Rr2[2] = {(R[0] + slack) * (R[0] + slack), (R[1] + slack) * (R[1] + slack)};
  const float R2[2] = {R[0] * R[0] * (1.0f + 2.0e-6f), R[1] * R[1] * (1.0f + 2.0e-6f)};  // a pair exactly at R is kept
  // ---- 1. segments (uniform trip counts for the whole warp: every iteration ends in a group-wide ballot) -------------
  float Rw = fmaxf(R[0], R[1]);  // the largest reach in this warp (its targets are almost always of one species)
#pragma unroll
  for (int o = 8; o < 32; o <<= 1) Rw = fmaxf(Rw, __shfl_xor_sync(0xffffffffu, Rw, o));
  const int mr = (int)ceilf((Rw + slack) / A.wS), side = 2 * mr + 1, rows = side * side;
  const float half = 0.5f * A.wS, inv_wx = 1.0f / A.wxS;
  int nseg = 0, total = 0;
  bool overflow = false;
  for (int r0 = 0; r0 < rows; r0 += GL) {
    const int r = r0 + h;
    const int rq = r / side;
    const int my = r - rq * side - mr, mz = rq - mr;
    const float fy = (float)my * A.wS - tq.y, fz = (float)mz * A.wS - tq.z;
    const float gy = fmaxf(fabsf(fy) - half, 0.f), gz = fmaxf(fabsf(fz) - half, 0.f);
    const float g2 = (r < rows && valid) ? gy * gy + gz * gz : 3.0e38f;
    int ay = cy + my, az = cz + mz;
    ay += ay < 0 ? A.ncell : (ay >= A.ncell ? -A.ncell : 0);
    az += az < 0 ? A.ncell : (az >= A.ncell ? -A.ncell : 0);
    const int row = (az * A.ncell + ay) * A.ncx;
#pragma unroll
    for (int ss = 0; ss < 2; ++ss) {
      const float rem = Rr2[ss] - g2;
      const float xr = sqrtf(fmaxf(rem, 0.f));
      const int lo = cx + (int)floorf((tq.x - xr) * inv_wx + 0.5f), hi = cx + (int)floorf((tq.x + xr) * inv_wx + 0.5f);
      const int32_t* bs = A.bin_start + A.base[ss] + row;
      // [lo, hi] cut at the periodic boundary (the box is wider than 2 R + 3 cells: no source has two images in range)
      const int nparts = __any_sync(0xffffffffu, rem > 0.f && (lo < 0 || hi >= A.ncx)) ? 2 : 1;
      for (int part = 0; part < nparts; ++part) {
        int a_lo = 1, a_hi = 0, code = 0;
        if (rem > 0.f) {
          if (part == 0) {
            a_lo = max(lo, 0);
            a_hi = min(hi, A.ncx - 1);
          } else if (lo < 0) {
            a_lo = lo + A.ncx;
            a_hi = A.ncx - 1;
            code = 1;
          } else if (hi >= A.ncx) {
            a_lo = 0;
            a_hi = hi - A.ncx;
            code = 2;
          }
        }
        int start = 0, len = 0;
        if (a_lo <= a_hi) {
          start = __ldg(bs + a_lo);
          len = __ldg(bs + a_hi + 1) - start;
        }
        const unsigned has = __ballot_sync(0xffffffffu, len > 0) & gmask;
        // (a stretch of 4096 slots or more does not fit a record: not a regime for lists)
        if (len > 0) {
          const int at = nseg + __popc(has & lower);
          if (at < SEG_CAP && len < 4096)
            seg[at] = Seg{start | (len << SLOT_BITS), (my + 8) | ((mz + 8) << 4) | (ss << 8) | (code << 9)};
          else
            overflow = true;
        }
        nseg += __popc(has);
        int incl = len;
#pragma unroll
        for (int o = 1; o < GL; o <<= 1) incl += __shfl_xor_sync(0xffffffffu, incl, o);  // (butterfly: every lane gets the sum)
        total += incl;
      }
    }
  }
  overflow = (__ballot_sync(0xffffffffu, overflow) & gmask) != 0;
  if (overflow && h == 0 && valid) atomicOr(A.cursor, LIST_FAIL);
  if (overflow) total = 0;
  __syncwarp();
  // ---- 2. count, 3. fill: two passes over the candidate stream ----------------------------------------------------------
  int n0 = 0, n1 = 0;             // kept proton / neutron sources (group totals)
  int32_t* out0 = nullptr;
  int32_t* out1 = nullptr;
  const int trips = (total + GL - 1) / GL;
  int trips_max = trips;
#pragma unroll
  for (int o = 8; o < 32; o <<= 1) trips_max = max(trips_max, __shfl_xor_sync(0xffffffffu, trips_max, o));
  for (int pass = 0; pass < 2; ++pass) {
    if (pass == 1 && !__any_sync(0xffffffffu, total > 0)) break;  // every list of this warp was staged
    int cur = 0, begin = 0, end = nseg > 0 ? (seg[0].start_len >> SLOT_BITS) & 4095 : 0;
    Seg sg = seg[0];
    int w0 = 0, w1 = 0;
    for (int i = 0; i < trips_max; ++i) {
      const int k = i * GL + h;
      bool keep = false;
      int ss = 0, e = 0;
      if (k < total) {
        while (k >= end) {
          ++cur;
          sg = seg[cur];
          begin = end;
          end += (sg.start_len >> SLOT_BITS) & 4095;
        }
        const int j = (sg.start_len & ((1 << SLOT_BITS) - 1)) + (k - begin);
        const int my = (sg.where & 15) - 8, mz = ((sg.where >> 4) & 15) - 8, code = sg.where >> 9;
        ss = (sg.where >> 8) & 1;
        const float4 q = __ldg(A.pos4 + j);
        const int mx = (__float_as_int(q.w) & 4095) - cx + (code == 1 ? -A.ncx : (code == 2 ? A.ncx : 0));
        const float dx = fmaf((float)mx, A.wxS, q.x - tq.x), dy = fmaf((float)my, A.wS, q.y - tq.y),
                    dz = fmaf((float)mz, A.wS, q.z - tq.z);
        keep = fmaf(dz, dz, fmaf(dy, dy, dx * dx)) <= R2[ss] && j != t;
        e = pack_entry(j, mx, my, mz);
      }
      const unsigned k0 = __ballot_sync(0xffffffffu, keep && ss == 0) & gmask;
      const unsigned k1 = __ballot_sync(0xffffffffu, keep && ss == 1) & gmask;
      if (keep) {
        const int at = ss == 0 ? w0 + __popc(k0 & lower) : w1 + __popc(k1 & lower);
        if (pass == 1) (ss == 0 ? out0 : out1)[at] = e;
        else if (w0 + __popc(k0) + w1 + __popc(k1) <= STG) stage[ss == 0 ? at : STG - 1 - at] = e;
      }
      w0 += __popc(k0);
      w1 += __popc(k1);
    }
    if (pass == 0) {
      n0 = w0;
      n1 = w1;
      unsigned long long first = 0;
      if (h == 0 && valid) first = atomicAdd(A.cursor, (unsigned long long)(n0 + n1)) & (LIST_FAIL - 1);
      first = __shfl_sync(0xffffffffu, first, 0, GL);
      const bool fits = first + (unsigned long long)(n0 + n1) <= (unsigned long long)A.pool_cap;
      if (h == 0 && valid) A.tl[t] = fits ? make_int4((int)first, n0, (int)first + n0, n1) : make_int4(0, 0, 0, 0);
      out0 = A.pool + first;
      out1 = A.pool + first + n0;
      __syncwarp();  // (outside the branch: every lane of the warp arrives)
      if (fits && n0 + n1 <= STG) {
        for (int k = h; k < n0; k += GL) out0[k] = stage[k];
        for (int k = h; k < n1; k += GL) out1[k] = stage[STG - 1 - k];
      }
      if (!fits || n0 + n1 <= STG) total = 0;  // nothing left to fill (the trip count stays warp-uniform)
    }
  }
}

// ---- force kernel on the lists -----------------------------------------------------------------------------------------
struct Acc4 {
  float fx, fy, fz, e;
};

// displacement source - target in scaled units: cell-relative coordinates + (the entry's frozen cell offset) * cell width
__device__ __forceinline__ void displacement(const TListArgs& A, const float4 tq, const int e, const float4 q, float& dx,
                                             float& dy, float& dz) {
  const int mx = (e << 8) >> 28, my = (e << 4) >> 28, mz = e >> 28;  // sign-extending
  dx = fmaf((float)mx, A.wxS, q.x - tq.x);
  dy = fmaf((float)my, A.wS, q.y - tq.y);
  dz = fmaf((float)mz, A.wS, q.z - tq.z);
}

// Sources [first, first + len) against target tq; lane h takes entries h, h + 8, ..., four at a time so that four
// independent chains (entry -> position -> exp2 -> accumulate) are in flight.
constexpr int UL = 4;
template <bool CUT, bool ENERGY>
__device__ __forceinline__ void run_tlist(const TListArgs& A, const PairConsts& c, const float4 tq, const int first,
                                          const int len, const int h, const bool coul, const float B, const float gB,
                                          Acc4& acc) {
  constexpr int SLOT_MASK = (1 << SLOT_BITS) - 1;
  const int32_t* __restrict__ lst = A.pool + first;
  for (int k0 = h; k0 < len; k0 += GL * UL) {
    int e[UL];
    float4 q[UL];
#pragma unroll
    for (int u = 0; u < UL; ++u) e[u] = k0 + u * GL < len ? __ldg(lst + k0 + u * GL) : 0;
#pragma unroll
    for (int u = 0; u < UL; ++u) {
      q[u] = __ldg(A.pos4 + (e[u] & SLOT_MASK));
      if (k0 + u * GL >= len) q[u].x = 1.0e18f;  // no entry: a source so far away that every term is exactly zero
    }
#pragma unroll
    for (int u = 0; u < UL; ++u) {
      float dx, dy, dz;
      displacement(A, tq, e[u], q[u], dx, dy, dz);
      const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
      float uu = ex2_ftz(-r2);
      if (CUT) uu = r2 < c.rn2s ? uu : 0.f;
      float g = uu * fmaf(c.g2a, uu, gB);
      if (ENERGY) acc.e = fmaf(uu, fmaf(c.a, uu, B), acc.e);
      if (coul) {
        // screened Coulomb, cut at r_c, skipped at r = 0 (coincident protons, D2)
        const float rinv = (r2 < c.rc2s && r2 > 0.f) ? rsqrt_ftz(r2) : 0.f;
        const float r = r2 * rinv;
        const float tq_ = ex2_ftz(-c.kappa * r) * rinv;
        if (ENERGY) acc.e = fmaf(c.alpha_s, tq_, acc.e);
        g = fmaf(c.alpha_s2 * tq_, (rinv + c.inv_lam_s) * rinv, g);
      }
      acc.fx = fmaf(g, dx, acc.fx);
      acc.fy = fmaf(g, dy, acc.fy);
      acc.fz = fmaf(g, dz, acc.fz);
    }
  }
}

template <bool CUT, bool ENERGY>
__global__ void __launch_bounds__(256) k2_tlist_kernel(const TListArgs A, const PairConsts c) {
  if (A.gate && *A.gate == 0u) return;  // a particle has left its halo: the host rebuilds and evaluates again
  const int gt = A.slot_lo + blockIdx.x * (blockDim.x / GL) + (threadIdx.x / GL);
  const int h = threadIdx.x & (GL - 1);
  const bool valid = gt < A.slot_hi;
  const int t = valid ? gt : A.slot_hi - 1;
  const float4 tq = __ldg(A.pos4 + t);
  const bool tp = t < A.Np;
  int4 tl = __ldg(A.tl + t);
  if (!valid) tl.y = tl.w = 0;
  Acc4 acc = {0.f, 0.f, 0.f, 0.f};
  // proton sources: like (+ Coulomb) for a proton target, unlike for a neutron target; then the neutron sources
  run_tlist<CUT, ENERGY>(A, c, tq, tl.x, tl.y, h, tp && A.no_coul == 0, tp ? c.B_like : c.B_unlike, tp ? c.gB_like : c.gB_unlike, acc);
  run_tlist<CUT, ENERGY>(A, c, tq, tl.z, tl.w, h, false, tp ? c.B_unlike : c.B_like, tp ? c.gB_unlike : c.gB_like, acc);
  // the 8 lanes' FP32 partial sums meet in FP64
  double fx = (double)acc.fx, fy = (double)acc.fy, fz = (double)acc.fz, ee = (double)acc.e;
#pragma unroll
  for (int o = GL / 2; o > 0; o >>= 1) {
    fx += __shfl_xor_sync(0xffffffffu, fx, o);
    fy += __shfl_xor_sync(0xffffffffu, fy, o);
    fz += __shfl_xor_sync(0xffffffffu, fz, o);
    if (ENERGY) ee += __shfl_xor_sync(0xffffffffu, ee, o);
  }
  if (h == 0 && valid) {
    const int i = __ldg(A.perm + t);
    A.F[3 * (int64_t)i + 0] = -fx;  // d was x_j - x_i
    A.F[3 * (int64_t)i + 1] = -fy;
    A.F[3 * (int64_t)i + 2] = -fz;
    if (ENERGY) A.e[i] = 0.5 * ee;
    if (A.kick != 0.0) {  // the arithmetic of k3_kick_ke_kernel on the stored force
      const double Fx = -fx, Fy = -fy, Fz = -fz;
      A.v[3 * (int64_t)i + 0] = A.v[3 * (int64_t)i + 0] + A.kick * Fx;
      A.v[3 * (int64_t)i + 1] = A.v[3 * (int64_t)i + 1] + A.kick * Fy;
      A.v[3 * (int64_t)i + 2] = A.v[3 * (int64_t)i + 2] + A.kick * Fz;
    }
  }
}

}  // namespace

static int tlist_args(Sim* s, TListArgs* out, double halo) {
  TListArgs& A = *out;
  const double sigma = sqrt(1.4426950408889634074 / (2.0 * s->prm.Lambda));
  const Grid& g = s->grid_sp[0];
  if (s->grid_sp[1].ncell != g.ncell || s->grid_sp[1].ncx != g.ncx) {
    set_error("neighbour lists need one grid geometry for both species");
    return PASTA_ESTATE;
  }
  A.N = (int32_t)s->N;
  A.Np = (int32_t)s->Np;
  A.gate = nullptr;
  A.v = s->v.as<double>();
  A.kick = 0.0;
  A.no_coul = s->prm.coulomb_all_pairs ? 1 : 0;
  A.slot_lo = s->shard.slot_lo < 0 ? 0 : s->shard.slot_lo;
  A.slot_hi = s->shard.slot_hi > A.N ? A.N : s->shard.slot_hi;
  A.ncell = g.ncell;
  A.ncx = g.ncx;
  A.base[0] = (int32_t)s->bin_base[0];
  A.base[1] = (int32_t)s->bin_base[1];
  A.wS = (float)(sigma * g.w);
  A.wxS = (float)(sigma * g.wx);
  A.rcS = (float)(sigma * s->prm.r_c);
  // reach of the nuclear terms: r_nuc if set, else r_c -- but never beyond the distance at which exp2(-r'^2) is exactly
  // 0 in the kernel's arithmetic (sqrt(126.5) in scaled units, D23) when skip_exact_zeros allows
  const double rn = sigma * (s->prm.r_nuc > 0.0 ? s->prm.r_nuc : s->prm.r_c);
  A.nucS = (float)(s->prm.skip_exact_zeros && rn > 11.2472 ? 11.2472 : rn);
  A.haloS = (float)(sigma * halo);
  A.pos4 = s->pos4.as<float4>();
  A.bin_start = s->bin_start.as<int32_t>();
  A.perm = s->perm.as<int32_t>();
  A.tl = s->list_off.as<int4>();
  A.pool = s->list_pool.as<int32_t>();
  A.pool_cap = (int64_t)(s->list_pool.bytes / sizeof(int32_t));
  A.cursor = s->counters.as<unsigned long long>() + 29;
  A.F = s->F.as<double>();
  A.e = s->e.as<double>();
  return PASTA_OK;
}

// Build the per-target lists of the sorted order k1_build has just made.  One launch; the stream is synchronised once to
// learn the pool size (a second launch follows only if the pool was too small).  Returns 1 (not an error) if the
// configuration is too dense for the lists' segment table: the caller then evaluates without lists.
int k2_list_build(Sim* s, double halo) {
  const int64_t N = s->N;
  PASTA_TRY(buffer_reserve(s, &s->list_off, sizeof(int4) * (size_t)N));
  if (!s->list_pool.ptr) {
    // first guess: uniform gas at the current density within (nuclear reach + halo), twice over, plus 32 per target
    const double R = (s->prm.skip_exact_zeros ? fmin(s->prm.r_c, 14.78) : s->prm.r_c) + halo;
    const double per = 2.0 * ((double)N / (s->L * s->L * s->L)) * 4.18879 * R * R * R + 32.0;
    PASTA_TRY(buffer_reserve(s, &s->list_pool, sizeof(int32_t) * (size_t)(per * (double)N)));
  }
  for (int attempt = 0; attempt < 2; ++attempt) {
    TListArgs A;
    PASTA_TRY(tlist_args(s, &A, halo));
    PASTA_CUDA_OK(cudaMemsetAsync(A.cursor, 0, sizeof(unsigned long long), s->stream));
    const size_t smem = (sizeof(Seg) * SEG_CAP + sizeof(int32_t) * STG) * (BUILD_T / GL);
    PASTA_CUDA_OK(cudaFuncSetAttribute(k2_tlist_build_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k2_tlist_build_kernel<<<grid_for(N * GL, BUILD_T), BUILD_T, smem, s->stream>>>(A);
    s->launches += 1;
    PASTA_CUDA_OK(cudaGetLastError());
    unsigned long long total = 0;
    PASTA_CUDA_OK(cudaMemcpyAsync(&total, A.cursor, sizeof(total), cudaMemcpyDeviceToHost, s->stream));
    PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
    if (total & LIST_FAIL) return 1;  // a target with more row segments than a list holds: not a regime for lists
    s->list_entries = (int64_t)total;
    if ((int64_t)total <= A.pool_cap) return PASTA_OK;
    if (total >= (1ull << 31)) {
      set_error("neighbour lists need %llu entries (limit 2^31)", total);
      return PASTA_ENOMEM;
    }
    PASTA_TRY(buffer_reserve(s, &s->list_pool, sizeof(int32_t) * (size_t)(total + total / 4)));
  }
  set_error("neighbour-list pool still too small after a resize");
  return PASTA_ESTATE;
}

int k2_list_forces(Sim* s, bool with_energy, bool gated, double kick) {
  const PairConsts c = make_pair_consts(s->prm);
  const bool cut = (double)c.rn2s < 127.0;  // the nuclear cut-off lies inside the FP32 underflow distance
  TListArgs A;
  PASTA_TRY(tlist_args(s, &A, 0.0));
  if (gated) A.gate = s->counters.as<unsigned>() + 2 * 31;
  A.kick = kick;
  if (A.slot_hi <= A.slot_lo) return PASTA_OK;  // this rank owns no target (pasta_set_shard)
  const int grid = grid_for((int64_t)(A.slot_hi - A.slot_lo) * GL, 256);
  if (with_energy) {
    if (cut) k2_tlist_kernel<true, true><<<grid, 256, 0, s->stream>>>(A, c);
    else k2_tlist_kernel<false, true><<<grid, 256, 0, s->stream>>>(A, c);
  } else {
    if (cut) k2_tlist_kernel<true, false><<<grid, 256, 0, s->stream>>>(A, c);
    else k2_tlist_kernel<false, false><<<grid, 256, 0, s->stream>>>(A, c);
  }
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

}  // namespace pasta
