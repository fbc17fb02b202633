// K2, production variant -- "chunk" pair-force kernel for sm_100a.
//
// Work decomposition:
//   * a CHUNK is T = 8 consecutive same-species particles of the cell-sorted order.  The force grids are
//     sliced into thin cells along x, so a row of cells (fixed cy, cz) is sorted in x and a chunk is a
//     short stretch of one row: spatially compact.  One warp owns one chunk.  The 8 targets live in
//     registers, replicated in every lane and packed two by two, so that the pair arithmetic runs as
//     packed FP32 (FFMA2/FADD2/FMUL2: two pairs per issued instruction).
//   * LANES run over SOURCES.  For each source species the warp lists the rows of that species' grid
//     that can hold a particle within r_c of the chunk's bounding box, and for every row the tight range
//     of thin cells [lo_x - xr, hi_x + xr]; a range is contiguous in the sorted arrays, i.e. one segment
//     of slots (two where it crosses the periodic boundary: images are enumerated explicitly, there is
//     no per-pair nearest-image arithmetic and small boxes need no special case).  Segments are cut into
//     TILES of <= 32 slots described by 16 bytes in shared memory.
//   * tiles are streamed through a 4-deep cp.async ring (global -> shared, no registers), so the L2
//     latency of the position loads is off the critical path; every lane takes one source of the tile
//     and evaluates it against all 8 targets.  There is NO per-candidate test and no divergence: a
//     source that is out of range of a target contributes exactly zero (next point).
//   * the cut-off needs no test for np/nn pairs when sigma^2 r_c^2 > 126: exp2(-r'^2) flushes to exactly
//     zero there, so out-of-range pairs contribute exactly 0 (D1: plain truncation).  pp pairs carry the
//     screened Coulomb term and are cut explicitly; small r_c selects the explicitly cut path.
//   * per-lane partial sums are FP32 (about 70 terms per target and pass); they are combined across
//     lanes and passes in FP64 by a transposing butterfly, and written in original particle order.
#include "pasta_internal.cuh"

namespace pasta {

namespace {

constexpr int T = 8;            // targets per chunk
constexpr int NP = T / 2;       // packed target pairs
#ifndef K2_MINB
#define K2_MINB 4
#endif
#ifndef K2_UNIFORM
#define K2_UNIFORM 1
#endif
#ifndef K2_WARPS
#define K2_WARPS 4
#endif
constexpr int WARPS = K2_WARPS;  // warps (= chunks) per block
constexpr int DEPTH = 4;        // cp.async stages per warp
constexpr int SEG_CAP = 224;    // segment records per warp (7 rounds of 32 rows)
constexpr float XOFF_IDLE = 1.0e12f;  // cell offset given to idle lanes: puts their source ~1e11 away
constexpr float FAR = 1.0e10f;  // coordinate of padding sources/targets: exp2(-FAR^2) == 0, 0 * FAR == 0

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// Broadcast of lane `src`'s value through REDUX.OR: the result is provably warp-uniform (a uniform register).
__device__ __forceinline__ float bcast_uniform(float v, int lane, int src) {
  return __int_as_float(__reduce_or_sync(0xffffffffu, lane == src ? __float_as_int(v) : 0));
}
__device__ __forceinline__ float2 dup(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src, int src_bytes) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

struct SpeciesGrid {
  int32_t ncell, ncx, base;  // cells per side in y/z, thin cells per side in x, first bin
  float wS, inv_wS;          // sigma * cell width (y, z) and its inverse
  float wxS, inv_wxS;        // sigma * thin-cell width (x) and its inverse
  double wS_d, wxS_d;        // the widths in FP64 (frame shifts between the two grids)
};

struct ChunkArgs {
  int32_t N, Np;
  int32_t n_chunks_p, n_chunks;
  SpeciesGrid g[2];
  float rcS;  // sigma * r_c
  const float4* pos4;
  const int32_t* cxyz;
  const int32_t* bin_start;
  const int32_t* perm;
  double* F;
  double* e;
  unsigned long long* stats;  // [0] sources streamed, [1] tiles, [2] pair evaluations (STATS only)
};

// Shared memory of one warp.  The sources of a pass form one STREAM: the concatenation of its segments
// (runs of consecutive sorted slots, one periodic image of part of a row of cells each).  Tile j of the
// stream is positions [32 j, 32 j + 32): always full except the last one, whatever the segment lengths.
//   seg[k]  = { int bits: first slot - stream position of the segment's start, xoff, yoff, zoff }
//             xoff: add to pos4.w (thin-cell index) to get the cell offset from the frame's reference
//             cell; yoff, zoff: the row's offsets from the reference cell centre, times the cell width
//   cum[k]  = stream position at which segment k starts (cum[nseg] = stream length, then +infinity)
//   stage   = raw pos4 of the tile's sources (cp.async), meta = the lane's {xoff, yoff, zoff} for it
struct WarpShared {
  float4 seg[SEG_CAP + 1];
  int cum[SEG_CAP + 1 + 32];
};

// Targets and accumulators of one warp.  Targets are replicated in all lanes; accumulators hold this
// lane's partial sums.  Convention: d = x_j - x_i (so the accumulated forces are -F_i).
struct Targets {
  float2 ntx[NP], nty[NP], ntz[NP];  // minus the target coordinates, two targets per register pair
};
struct Accum {
  float2 fx[NP], fy[NP], fz[NP], e[NP];
};
struct PassConsts {
  float2 g2a, gB, a2, B2;
};

template <bool COUL, bool CUT, bool ENERGY>
__device__ __forceinline__ void evaluate(const float4 s, const Targets& t, Accum& acc, const PassConsts& k,
                                         const PairConsts& c) {
  // phase 1: displacements and -r'^2 of all 8 pairs; phase 2: the 8 exponentials back to back on the MUFU;
  // phase 3: polynomials and accumulation.  (Written in phases so that the MUFU latency of one pair is
  // covered by the arithmetic of the others.)
  float2 dx[NP], dy[NP], dz[NP], nr2[NP], u[NP];
#pragma unroll
  for (int p = 0; p < NP; ++p) {
    dx[p] = __fadd2_rn(dup(s.x), t.ntx[p]);
    dy[p] = __fadd2_rn(dup(s.y), t.nty[p]);
    dz[p] = __fadd2_rn(dup(s.z), t.ntz[p]);
    // minus r'^2, accumulated with negated operands (free on FFMA2) because MUFU.EX2 takes no negation
    nr2[p] = __fmul2_rn(neg2(dx[p]), dx[p]);
    nr2[p] = __ffma2_rn(neg2(dy[p]), dy[p], nr2[p]);
    nr2[p] = __ffma2_rn(neg2(dz[p]), dz[p], nr2[p]);
  }
#pragma unroll
  for (int p = 0; p < NP; ++p) {
    u[p] = make_float2(ex2_approx(nr2[p].x), ex2_approx(nr2[p].y));
    if (CUT) {
      u[p].x = nr2[p].x > -c.rc2s ? u[p].x : 0.f;
      u[p].y = nr2[p].y > -c.rc2s ? u[p].y : 0.f;
    }
  }
#pragma unroll
  for (int p = 0; p < NP; ++p) {
    float2 g = __fmul2_rn(u[p], __ffma2_rn(k.g2a, u[p], k.gB));
    float2 V;
    if (ENERGY) V = __fmul2_rn(u[p], __ffma2_rn(k.a2, u[p], k.B2));
    if (COUL) {
      // screened Coulomb, cut at r_c, skipped at r = 0 (the self pair and coincident protons, D2):
      // 1/r' := 0 for excluded pairs, which zeroes every Coulomb factor without creating inf * 0
      const bool in0 = nr2[p].x > -c.rc2s && nr2[p].x < 0.f, in1 = nr2[p].y > -c.rc2s && nr2[p].y < 0.f;
      const float2 rinv = make_float2(in0 ? rsqrt_approx(-nr2[p].x) : 0.f, in1 ? rsqrt_approx(-nr2[p].y) : 0.f);
      const float2 nr = __fmul2_rn(nr2[p], rinv);  // -r'
      const float2 ex = make_float2(ex2_approx(c.kappa * nr.x), ex2_approx(c.kappa * nr.y));
      const float2 tq = __fmul2_rn(ex, rinv);
      if (ENERGY) V = __ffma2_rn(dup(c.alpha_s), tq, V);
      const float2 q = __fmul2_rn(__fadd2_rn(rinv, dup(c.inv_lam_s)), rinv);
      g = __ffma2_rn(__fmul2_rn(dup(c.alpha_s2), tq), q, g);
    }
    acc.fx[p] = __ffma2_rn(g, dx[p], acc.fx[p]);
    acc.fy[p] = __ffma2_rn(g, dy[p], acc.fy[p]);
    acc.fz[p] = __ffma2_rn(g, dz[p], acc.fz[p]);
    if (ENERGY) acc.e[p] = __fadd2_rn(acc.e[p], V);
  }
}


__device__ __forceinline__ int floor_div(int a, int b) {  // b > 0
  const int q = a / b;
  return (a % b < 0) ? q - 1 : q;
}

// Per-lane cursor into the segment list of a pass: the segment holding the lane's current stream position.
struct Cursor {
  int cur;     // segment index
  int end;     // stream position at which segment `cur` ends
  float4 rec;  // its record
};

// Raw source of stream position `pos` for this lane (zeros past the end of the stream) and the record of the
// segment it belongs to.  A lane's positions grow by 32 per tile, so the cursor only ever moves forward.
__device__ __forceinline__ void fetch(const ChunkArgs& A, const WarpShared& sh, Cursor& cu, const int pos,
                                      const int total, float4& q, float4& m) {
  if (pos >= cu.end) {
    do {
      ++cu.cur;
      cu.end = sh.cum[cu.cur + 1];
    } while (pos >= cu.end);
    cu.rec = sh.seg[cu.cur];
  }
  m = cu.rec;
  q = make_float4(0.f, 0.f, 0.f, 0.f);
  if (pos < total) q = __ldg(A.pos4 + (__float_as_int(cu.rec.x) + pos));
}

// source position in the frame: cell-relative coordinate + integer cell offset * cell width
__device__ __forceinline__ float4 to_frame(const float4 q, const float4 m, const float wxS) {
  float4 s;
  s.x = fmaf(q.w + m.y, wxS, q.x);
  s.y = __fadd_rn(q.y, m.z);
  s.z = __fadd_rn(q.z, m.w);
  s.w = 0.f;
  return s;
}

// Stream the listed segments, 32 stream positions at a time, and evaluate every source against the 8
// targets.  Sources are fetched straight into registers two tiles ahead (the positions are L2-resident);
// the loop handles two tiles per trip so that the double buffer needs no register moves.  An odd tail is
// padded with one tile of idle lanes, which contribute exact zeros.
template <bool COUL, bool CUT, bool ENERGY, bool STATS>
__device__ __forceinline__ void run_stream(const ChunkArgs& A, const PairConsts& c, WarpShared& sh, const int lane,
                                           const int nseg, const int total, const float wxS, const Targets& t,
                                           Accum& acc, const PassConsts& k, unsigned long long* st) {
  if (total == 0) return;
  const int ntile = (total + 31) >> 5;
  Cursor cu;
  cu.cur = 0;
  cu.end = sh.cum[1];
  cu.rec = sh.seg[0];
  float4 qa, ma, qb, mb;
  fetch(A, sh, cu, lane, total, qa, ma);
  fetch(A, sh, cu, 32 + lane, total, qb, mb);
#pragma unroll 1
  for (int i = 0; i < ntile; i += 2) {
    const float4 sa = to_frame(qa, ma, wxS);
    fetch(A, sh, cu, ((i + 2) << 5) + lane, total, qa, ma);
    evaluate<COUL, CUT, ENERGY>(sa, t, acc, k, c);
    const float4 sb = to_frame(qb, mb, wxS);
    fetch(A, sh, cu, ((i + 3) << 5) + lane, total, qb, mb);
    evaluate<COUL, CUT, ENERGY>(sb, t, acc, k, c);
  }
  if (STATS && lane == 0) {
    st[0] += (unsigned long long)total;
    st[1] += (unsigned long long)((ntile + 1) & ~1);
    st[2] += 32ull * T * (unsigned long long)((ntile + 1) & ~1);
  }
}

// Bounding box of the chunk in the frame of a pass.
struct Box {
  float lo_x, hi_x, lo_y, hi_y, lo_z, hi_z;
};

// One pass of a chunk over one source species: list the segments, stream them.
template <bool COUL, bool CUT, bool ENERGY, bool STATS>
__device__ __forceinline__ void source_pass(const ChunkArgs& A, const PairConsts& c, WarpShared& sh, const int lane,
                                            const SpeciesGrid& gs, const int rx, const int ry, const int rz,
                                            const Box& b, const Targets& t, Accum& acc, const PassConsts& k,
                                            unsigned long long* st) {
  const float half = 0.5f * gs.wS;
  // a hair of slack covers FP32 rounding of cell-relative coordinates against the cell boundaries
  const float slack = 1.0e-3f * gs.wS;
  const float rc = A.rcS + slack, rc2 = rc * rc;
  const int my_lo = (int)floorf((b.lo_y - rc) * gs.inv_wS + 0.5f), my_hi = (int)floorf((b.hi_y + rc) * gs.inv_wS + 0.5f);
  const int mz_lo = (int)floorf((b.lo_z - rc) * gs.inv_wS + 0.5f), mz_hi = (int)floorf((b.hi_z + rc) * gs.inv_wS + 0.5f);
  const int ny = my_hi - my_lo + 1, nrows = ny * (mz_hi - mz_lo + 1);
  const int nc = gs.ncell, ncx = gs.ncx;
  const unsigned lt_mask = (1u << lane) - 1u;
  int nseg_list = 0, total = 0;

  // close the list (dummy record for idle lanes, +infinity boundaries) and stream it
  auto flush = [&]() {
    if (lane == 0) sh.seg[nseg_list] = make_float4(0.f, XOFF_IDLE, 0.f, 0.f);
    sh.cum[nseg_list + lane] = lane == 0 ? total : 0x3fffffff;
    if (lane == 0) sh.cum[nseg_list + 32] = 0x3fffffff;
    __syncwarp();
    run_stream<COUL, CUT, ENERGY, STATS>(A, c, sh, lane, nseg_list, total, gs.wxS, t, acc, k, st);
    nseg_list = 0;
    total = 0;
    __syncwarp();
  };

  for (int rbase = 0; rbase < nrows; rbase += 32) {
    const int r = rbase + lane;
    int nseg = 0, ax_lo = 0, ax_hi = 0, q_lo = 0, rowbase = 0;
    float yoff = 0.f, zoff = 0.f;
    if (r < nrows) {
      const int my = my_lo + r % ny, mz = mz_lo + r / ny;
      yoff = __fmul_rn((float)my, gs.wS);
      zoff = __fmul_rn((float)mz, gs.wS);
      // gap between the row's slab [off - w/2, off + w/2] and the box interval, per axis
      const float gy = fmaxf(fmaxf(b.lo_y - (yoff + half), (yoff - half) - b.hi_y), 0.f);
      const float gz = fmaxf(fmaxf(b.lo_z - (zoff + half), (zoff - half) - b.hi_z), 0.f);
      const float rem = rc2 - gy * gy - gz * gz;
      if (rem > 0.f) {
        const float xr = sqrtf(rem);
        ax_lo = rx + (int)floorf((b.lo_x - xr) * gs.inv_wxS + 0.5f);
        ax_hi = rx + (int)floorf((b.hi_x + xr) * gs.inv_wxS + 0.5f);
        q_lo = floor_div(ax_lo, ncx);
        nseg = floor_div(ax_hi, ncx) - q_lo + 1;
        int ay = (ry + my) % nc, az = (rz + mz) % nc;
        ay += ay < 0 ? nc : 0;
        az += az < 0 ? nc : 0;
        rowbase = gs.base + (az * nc + ay) * ncx;
      }
    }
    for (int round = 0; __any_sync(0xffffffffu, round < nseg); ++round) {
      if (nseg_list + 32 > SEG_CAP) flush();  // (warp-uniform) list full: stream what is there
      int start = 0, len = 0;
      float xoff = 0.f;
      if (round < nseg) {
        const int q = q_lo + round, qb = q * ncx;
        const int a_lo = max(ax_lo, qb) - qb, a_hi = min(ax_hi, qb + ncx - 1) - qb;
        start = __ldg(A.bin_start + rowbase + a_lo);
        len = __ldg(A.bin_start + rowbase + a_hi + 1) - start;
        xoff = (float)(qb - rx);
      }
      // append the non-empty segments in lane order; stream positions by an inclusive scan of the lengths
      int incl = len;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
      }
      const unsigned has = __ballot_sync(0xffffffffu, len > 0);
      if (len > 0) {
        const int at = nseg_list + __popc(has & lt_mask), begin = total + incl - len;
        sh.seg[at] = make_float4(__int_as_float(start - begin), xoff, yoff, zoff);
        sh.cum[at] = begin;
      }
      nseg_list += __popc(has);
      total += __shfl_sync(0xffffffffu, incl, 31);
    }
  }
  flush();
}

// Sum v over the warp for 32 different quantities at once: on entry lane l holds its partial of quantity
// q in v[q]; on exit lane l holds the full sum of quantity l.  31 shuffles instead of 160.
__device__ __forceinline__ double transpose_reduce(double (&v)[32], const int lane) {
#pragma unroll
  for (int w = 16; w >= 1; w >>= 1) {
    const bool upper = (lane & w) != 0;
#pragma unroll
    for (int q = 0; q < w; ++q) {
      const double keep = upper ? v[q + w] : v[q];
      const double give = upper ? v[q] : v[q + w];
      v[q] = keep + __shfl_xor_sync(0xffffffffu, give, w);
    }
  }
  return v[0];
}

__device__ __forceinline__ int min_image_cells(int m, int nc) {
  const int hc = nc / 2;
  return m + (m > hc ? -nc : (m < -hc ? nc : 0));
}

template <bool CUT, bool ENERGY, bool STATS>
__global__ void __launch_bounds__(WARPS * 32, K2_MINB) k2_chunk_kernel(const ChunkArgs A, const PairConsts c) {
  __shared__ WarpShared shared[WARPS];
  const int lane = threadIdx.x & 31;
#if K2_UNIFORM
  // warp-uniform values are produced by REDUX so that the compiler can prove them uniform and keep them
  // (and everything derived from them) in uniform registers, off the vector register file
  const int wib = __reduce_or_sync(0xffffffffu, (int)(threadIdx.x >> 5));
#else
  const int wib = threadIdx.x >> 5;
#endif
  const int chunk = blockIdx.x * WARPS + wib;
  if (chunk >= A.n_chunks) return;
  WarpShared& sh = shared[wib];

  const bool chunk_p = chunk < A.n_chunks_p;
  const int st_sp = chunk_p ? 0 : 1;
  const SpeciesGrid gt = A.g[st_sp];
  const int base = chunk_p ? chunk * T : A.Np + (chunk - A.n_chunks_p) * T;
  const int nvalid = min(T, (chunk_p ? A.Np : A.N) - base);

  // ---- targets: lane l < nvalid holds target l; all other lanes mirror target 0 ------------------------
  const int tl = lane < nvalid ? lane : 0;
  const float4 tp = __ldg(A.pos4 + base + tl);
  const int tc = __ldg(A.cxyz + base + tl);
  const int oc = __shfl_sync(0xffffffffu, tc, 0);
  const int ox = PASTA_CX(oc), oy = PASTA_CY(oc), oz = PASTA_CZ(oc);
  // cell offset from the origin cell, taken in the nearest periodic image (chunks may wrap a row end)
  const int mx = min_image_cells(PASTA_CX(tc) - ox, gt.ncx);
  const int my = min_image_cells(PASTA_CY(tc) - oy, gt.ncell);
  const int mz = min_image_cells(PASTA_CZ(tc) - oz, gt.ncell);

  Accum acc;
#pragma unroll
  for (int p = 0; p < NP; ++p) acc.fx[p] = acc.fy[p] = acc.fz[p] = acc.e[p] = make_float2(0.f, 0.f);
  unsigned long long st[3] = {0, 0, 0};

  // ---- pass 0: proton sources, pass 1: neutron sources -------------------------------------------------
#pragma unroll 1
  for (int sp = 0; sp < 2; ++sp) {
    const SpeciesGrid gs = A.g[sp];
    // Frame of the pass: origin = centre of the source-grid cell (rx, ry, rz) that contains the centre of
    // the chunk's origin cell.  Same grid: identical arithmetic for targets and sources (a target meets
    // itself at d == 0 exactly).  Other grid: the shift between the two cell centres is taken in FP64.
    int rx = ox, ry = oy, rz = oz;
    float X, Y, Z;
    if (gs.ncell == gt.ncell && gs.ncx == gt.ncx) {  // same grid geometry (always true for the chunk's own species)
      X = fmaf((float)mx, gs.wxS, tp.x);
      Y = __fadd_rn(tp.y, __fmul_rn((float)my, gs.wS));
      Z = __fadd_rn(tp.z, __fmul_rn((float)mz, gs.wS));
    } else {
      const double cx0 = ((double)ox + 0.5) * gt.wxS_d, cy0 = ((double)oy + 0.5) * gt.wS_d, cz0 = ((double)oz + 0.5) * gt.wS_d;
      rx = min(gs.ncx - 1, (int)(cx0 / gs.wxS_d));
      ry = min(gs.ncell - 1, (int)(cy0 / gs.wS_d));
      rz = min(gs.ncell - 1, (int)(cz0 / gs.wS_d));
      X = (float)((double)tp.x + (double)mx * gt.wxS_d + (cx0 - ((double)rx + 0.5) * gs.wxS_d));
      Y = (float)((double)tp.y + (double)my * gt.wS_d + (cy0 - ((double)ry + 0.5) * gs.wS_d));
      Z = (float)((double)tp.z + (double)mz * gt.wS_d + (cz0 - ((double)rz + 0.5) * gs.wS_d));
    }
    // bounding box of the chunk (lanes >= nvalid mirror target 0)
    Box b = {X, X, Y, Y, Z, Z};
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      b.lo_x = fminf(b.lo_x, __shfl_xor_sync(0xffffffffu, b.lo_x, o));
      b.hi_x = fmaxf(b.hi_x, __shfl_xor_sync(0xffffffffu, b.hi_x, o));
      b.lo_y = fminf(b.lo_y, __shfl_xor_sync(0xffffffffu, b.lo_y, o));
      b.hi_y = fmaxf(b.hi_y, __shfl_xor_sync(0xffffffffu, b.hi_y, o));
      b.lo_z = fminf(b.lo_z, __shfl_xor_sync(0xffffffffu, b.lo_z, o));
      b.hi_z = fmaxf(b.hi_z, __shfl_xor_sync(0xffffffffu, b.hi_z, o));
    }
    Targets t;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
#if K2_UNIFORM
      // lane j < 8 contributes minus its coordinate (FAR if it holds no valid target), every other lane 0
      const float nX = lane < nvalid ? -X : FAR, nY = lane < nvalid ? -Y : FAR, nZ = lane < nvalid ? -Z : FAR;
      t.ntx[p] = make_float2(bcast_uniform(nX, lane, 2 * p), bcast_uniform(nX, lane, 2 * p + 1));
      t.nty[p] = make_float2(bcast_uniform(nY, lane, 2 * p), bcast_uniform(nY, lane, 2 * p + 1));
      t.ntz[p] = make_float2(bcast_uniform(nZ, lane, 2 * p), bcast_uniform(nZ, lane, 2 * p + 1));
#else
      const float x0 = __shfl_sync(0xffffffffu, X, 2 * p), x1 = __shfl_sync(0xffffffffu, X, 2 * p + 1);
      const float y0 = __shfl_sync(0xffffffffu, Y, 2 * p), y1 = __shfl_sync(0xffffffffu, Y, 2 * p + 1);
      const float z0 = __shfl_sync(0xffffffffu, Z, 2 * p), z1 = __shfl_sync(0xffffffffu, Z, 2 * p + 1);
      const bool v0 = 2 * p < nvalid, v1 = 2 * p + 1 < nvalid;
      t.ntx[p] = make_float2(v0 ? -x0 : FAR, v1 ? -x1 : FAR);
      t.nty[p] = make_float2(v0 ? -y0 : FAR, v1 ? -y1 : FAR);
      t.ntz[p] = make_float2(v0 ? -z0 : FAR, v1 ? -z1 : FAR);
#endif
    }
    const bool like = sp == st_sp;
    PassConsts k;
    k.g2a = dup(c.g2a);
    k.gB = dup(like ? c.gB_like : c.gB_unlike);
    k.a2 = dup(c.a);
    k.B2 = dup(like ? c.B_like : c.B_unlike);
    if (chunk_p && sp == 0)
      source_pass<true, CUT, ENERGY, STATS>(A, c, sh, lane, gs, rx, ry, rz, b, t, acc, k, st);
    else
      source_pass<false, CUT, ENERGY, STATS>(A, c, sh, lane, gs, rx, ry, rz, b, t, acc, k, st);
  }

  // ---- combine the lanes' FP32 partials in FP64: quantity index = 4 * target + {fx, fy, fz, e} ------------
  double v[32];
#pragma unroll
  for (int p = 0; p < NP; ++p) {
    v[8 * p + 0] = (double)acc.fx[p].x; v[8 * p + 1] = (double)acc.fy[p].x;
    v[8 * p + 2] = (double)acc.fz[p].x; v[8 * p + 3] = (double)acc.e[p].x;
    v[8 * p + 4] = (double)acc.fx[p].y; v[8 * p + 5] = (double)acc.fy[p].y;
    v[8 * p + 6] = (double)acc.fz[p].y; v[8 * p + 7] = (double)acc.e[p].y;
  }
  const double sum = transpose_reduce(v, lane);
  const int tgt = lane >> 2, comp = lane & 3;
  if (tgt < nvalid) {
    const int i = __ldg(A.perm + base + tgt);
    if (comp < 3) {
      A.F[3 * (int64_t)i + comp] = -sum;  // d was x_j - x_i
    } else if (ENERGY) {
      // every target met itself once in its own species' pass at r = 0: remove V(0) = a + b + c
      A.e[i] = 0.5 * (sum - (double)c.v_self);
    }
  }
  if (STATS && lane == 0) {
    atomicAdd(A.stats + 0, st[0]);
    atomicAdd(A.stats + 1, st[1]);
    atomicAdd(A.stats + 2, st[2]);
  }
}

}  // namespace

int k2_chunk_forces(Sim* s, bool with_energy, bool stats) {
  const PairConsts c = make_pair_consts(s->prm);
  const double sigma = sqrt(1.4426950408889634074 / (2.0 * s->prm.Lambda));
  if (s->N >= (1ll << 26)) {
    set_error("the chunk pair kernel packs slot numbers in 26 bits: N must be below 2^26");
    return PASTA_EINVAL;
  }
  ChunkArgs A;
  A.N = (int32_t)s->N;
  A.Np = (int32_t)s->Np;
  A.n_chunks_p = (int32_t)((s->Np + T - 1) / T);
  A.n_chunks = A.n_chunks_p + (int32_t)((s->N - s->Np + T - 1) / T);
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
  A.pos4 = s->pos4.as<float4>();
  A.cxyz = s->cxyz.as<int32_t>();
  A.bin_start = s->bin_start.as<int32_t>();
  A.perm = s->perm.as<int32_t>();
  A.F = s->F.as<double>();
  A.e = s->e.as<double>();
  A.stats = s->counters.as<unsigned long long>() + 10;
  // exp2(-r'^2) is exactly 0 (FTZ) for r'^2 > 126: then np/nn pairs beyond r_c need no explicit cut
  const bool cut = (double)c.rc2s < 127.0;
  const int grid = (A.n_chunks + WARPS - 1) / WARPS;
  const dim3 block(WARPS * 32);
  if (stats) {
    PASTA_CUDA_OK(cudaMemsetAsync(A.stats, 0, 3 * sizeof(unsigned long long), s->stream));
    if (cut) k2_chunk_kernel<true, true, true><<<grid, block, 0, s->stream>>>(A, c);
    else k2_chunk_kernel<false, true, true><<<grid, block, 0, s->stream>>>(A, c);
  } else if (with_energy) {
    if (cut) k2_chunk_kernel<true, true, false><<<grid, block, 0, s->stream>>>(A, c);
    else k2_chunk_kernel<false, true, false><<<grid, block, 0, s->stream>>>(A, c);
  } else {
    if (cut) k2_chunk_kernel<true, false, false><<<grid, block, 0, s->stream>>>(A, c);
    else k2_chunk_kernel<false, false, false><<<grid, block, 0, s->stream>>>(A, c);
  }
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

}  // namespace pasta
