// Device-side machinery of the chunk pair kernel (k2_chunk.cu): the pair evaluation, the segment listing of a chunk's
// sources, the tile streamer, the chunk frame and the FP64 epilogue.  Everything lives in an anonymous namespace.
#pragma once
#include "pasta_internal.cuh"

namespace pasta {
namespace {


// Launch shape, settled by the sweeps of rounds 1 and 2 (profiles/r2_k2_experiments.md): 4 warps per
// block; 5 resident blocks per SM (96 registers) where chunks stream hundreds of tiles, 8 (64 registers) where a species
// is sparse and the latency of the listing sets the pace.
constexpr int K2_MINB = 5, K2_MINB_SPARSE = 8, K2_WARPS = 4;
constexpr int T = PASTA_CHUNK_T;   // targets per chunk
constexpr int NPAIR = T / 2;       // packed target pairs per chunk
constexpr int NPH = 32 / NPAIR;    // phases: lanes that share a target pair and split the sources of a tile
constexpr int STEPS = 32 / NPH;    // sources a lane takes from each tile
constexpr int WARPS = K2_WARPS;    // warps (= chunks) per block
constexpr int SEG_CAP = 160;       // segment records per warp (5 rounds of 32 rows)
constexpr float XOFF_IDLE = 1.0e12f;  // cell offset given to idle lanes: puts their source ~1e11 away
constexpr float FAR = 1.0e10f;  // coordinate of padding targets: exp2(-FAR^2) == 0, 0 * FAR == 0

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
__device__ __forceinline__ float2 dup(float a) { return make_float2(a, a); }
template <int OFF>
__device__ __forceinline__ float4 lds128(const unsigned a) {  // 16 bytes from shared-window address a + OFF
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a), "n"(OFF) : "memory");
  return v;
}
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }

struct SpeciesGrid {
  int32_t ncell, ncx, base;  // cells per side in y/z, thin cells per side in x, first bin
  float wS, inv_wS;          // sigma * cell width (y, z) and its inverse
  float wxS, inv_wxS;        // sigma * thin-cell width (x) and its inverse
  double wS_d, wxS_d;        // the widths in FP64 (frame shifts between the two grids)
};

struct ChunkArgs {
  int32_t N, Np;
  const int32_t* chunk_tab;  // [chunk][8] sorted slots of the chunk's targets, -1 = none (k1_cells.cu)
  const int32_t* counts;     // [0] number of chunks in the overflow region
  int32_t nprim;             // primary entries (some of them empty)
  int32_t slot_lo, slot_hi;  // target sharding: only chunks whose first target's slot lies in [slot_lo, slot_hi) are evaluated
  int32_t no_coul;           // coulomb_all_pairs: the Coulomb term is summed elsewhere (k2_coulomb.cu); nuclear terms only
  int32_t merged;            // the two species' grids are identical: neutron chunks take both in one pass
  SpeciesGrid g[2];
  float rcS;     // sigma * r_c
  float rnS;     // sigma * r_n (cut-off of the nuclear terms)
  float rzeroS;  // scaled distance beyond which exp2(-r'^2) is exactly 0 in FP32 with FTZ (sqrt(126.5))
  const float4* pos4;
  const int32_t* cxyz;
  const int32_t* bin_start;
  const int32_t* perm;
  double* F;
  double* e;
  double* v;       // kick != 0: the second half kick v += kick F rides along with the force write (O2 step 4)
  double kick;
  unsigned long long* stats;  // [0] sources streamed, [1] tiles, [2] pair evaluations (STATS only)
};

// Shared memory of one warp.  The sources of a pass form one STREAM: the concatenation of its segments
// (runs of consecutive sorted slots, one periodic image of part of a row of cells each).  Tile j of the
// stream is positions [32 j, 32 j + 32): always full except the last one, whatever the segment lengths.
//   seg[k]  = { int bits: first slot - stream position of the segment's start, xoff, yoff, zoff }
//             xoff: add to pos4.w (thin-cell index) to get the cell offset from the frame's reference
//             cell; yoff, zoff: the row's offsets from the reference cell centre, times the cell width
//   cum[k]  = stream position at which segment k starts (cum[nseg] = stream length, then +infinity)
// The tiles themselves -- the sources of two consecutive tiles in the chunk's frame, a double buffer of 2 x 512 bytes per
// warp -- live in an array of their own (k2_chunk_kernel), 1024-byte aligned, so that the two buffers of a warp differ
// in exactly one address bit and the toggle is a single XOR.
struct WarpShared {
  float4 seg[SEG_CAP + 1];
  int cum[SEG_CAP + 1 + 32];
  float flag[SEG_CAP + 1];  // BOTH-species streams: 0 = the segment holds protons, 1 = neutrons
};

// A lane's packed pair of targets (minus their coordinates) and its partial sums.
// Convention: d = x_j - x_i (so the accumulated forces are -F_i).
struct Targets {
  float2 ntx, nty, ntz;
};
struct Accum {
  float2 fx, fy, fz, e;
};
struct PassConsts {
  float g2a, gB, a, B;
  float gB_n, B_n;  // BOTH-species streams: gB, B apply to proton sources, gB_n, B_n to neutron sources
};

// One source against the lane's two targets.
template <bool COUL, bool CUT, bool ENERGY, bool BOTH>
__device__ __forceinline__ void evaluate(const float4 s, const Targets& t, Accum& acc, const PassConsts& k,
                                         const PairConsts& c) {
  // BOTH: the stream mixes the two source species; s.w tells which, and with it the isospin constants
  const float gB = BOTH ? (s.w != 0.f ? k.gB_n : k.gB) : k.gB, B = BOTH ? (s.w != 0.f ? k.B_n : k.B) : k.B;
  const float2 dx = __fadd2_rn(dup(s.x), t.ntx);
  const float2 dy = __fadd2_rn(dup(s.y), t.nty);
  const float2 dz = __fadd2_rn(dup(s.z), t.ntz);
  // minus r'^2, accumulated with negated operands (free on FFMA2) because MUFU.EX2 takes no negation
  float2 nr2 = __fmul2_rn(neg2(dx), dx);
  nr2 = __ffma2_rn(neg2(dy), dy, nr2);
  nr2 = __ffma2_rn(neg2(dz), dz, nr2);
  float2 u = make_float2(ex2_approx(nr2.x), ex2_approx(nr2.y));
  if (CUT) {
    u.x = nr2.x > -c.rn2s ? u.x : 0.f;
    u.y = nr2.y > -c.rn2s ? u.y : 0.f;
  }
  float2 g = __fmul2_rn(u, __ffma2_rn(dup(k.g2a), u, dup(gB)));
  if (ENERGY) acc.e = __ffma2_rn(u, __ffma2_rn(dup(k.a), u, dup(B)), acc.e);
  if (COUL) {
    // screened Coulomb, cut at r_c, skipped at r = 0 (the self pair and coincident protons, D2):
    // 1/r' := 0 for excluded pairs, which zeroes every Coulomb factor without creating inf * 0
    const bool in0 = nr2.x > -c.rc2s && nr2.x < 0.f, in1 = nr2.y > -c.rc2s && nr2.y < 0.f;
    const float2 rinv = make_float2(in0 ? rsqrt_approx(-nr2.x) : 0.f, in1 ? rsqrt_approx(-nr2.y) : 0.f);
    const float2 nr = __fmul2_rn(nr2, rinv);  // -r'
    const float2 ex = make_float2(ex2_approx(c.kappa * nr.x), ex2_approx(c.kappa * nr.y));
    const float2 tq = __fmul2_rn(ex, rinv);
    if (ENERGY) acc.e = __ffma2_rn(dup(c.alpha_s), tq, acc.e);
    const float2 q = __fmul2_rn(__fadd2_rn(rinv, dup(c.inv_lam_s)), rinv);
    g = __ffma2_rn(__fmul2_rn(dup(c.alpha_s2), tq), q, g);
  }
  acc.fx = __ffma2_rn(g, dx, acc.fx);
  acc.fy = __ffma2_rn(g, dy, acc.fy);
  acc.fz = __ffma2_rn(g, dz, acc.fz);
}

// floor(a / b), b > 0.  The listing only ever asks with -b <= a < 2 b (reach + box < L), where it is a
// comparison; the generic integer division (dozens of instructions) is the fallback.
__device__ __forceinline__ int floor_div(int a, int b) {
  if (a >= -b && a < 2 * b) return (a < 0 ? -1 : 0) + (a >= b ? 1 : 0);
  const int q = a / b;
  return (a % b < 0) ? q - 1 : q;
}
// a mod n in [0, n) for -n <= a < 2 n, generic otherwise
__device__ __forceinline__ int wrap_cell(int a, int n) {
  if (a >= -n && a < 2 * n) return a + (a < 0 ? n : 0) - (a >= n ? n : 0);
  a %= n;
  return a + (a < 0 ? n : 0);
}

// Per-lane cursor into the segment list of a pass: the segment holding the lane's current stream position.
struct Cursor {
  int cur;     // segment index
  int end;     // stream position at which segment `cur` ends
  float4 rec;  // its record
  float flag;  // BOTH-species streams: its species flag
};

// Raw source of stream position `pos` for this lane (zeros past the end of the stream) and the record of the
// segment it belongs to.  A lane's positions grow by 32 per tile, so the cursor only ever moves forward.
template <bool BOTH>
__device__ __forceinline__ void fetch(const ChunkArgs& A, const WarpShared& sh, Cursor& cu, const int pos,
                                      const int total, float4& q, float4& m) {
  if (pos >= cu.end) {
    do {
      ++cu.cur;
      cu.end = sh.cum[cu.cur + 1];
    } while (pos >= cu.end);
    cu.rec = sh.seg[cu.cur];
    if (BOTH) cu.flag = sh.flag[cu.cur];
  }
  m = cu.rec;
  // positions past the end of the stream sit on the closing dummy record, whose cell offset throws whatever is loaded
  // 1e11 away: any valid address will do
  (void)total;
  q = __ldg(A.pos4 + min(__float_as_int(cu.rec.x) + pos, A.N - 1));

  if (BOTH) m.x = cu.flag;  // the slot offset has served; its place carries the species flag to to_frame
}

// source position in the frame: cell-relative coordinate + integer cell offset * cell width
template <bool BOTH>
__device__ __forceinline__ float4 to_frame(const float4 q, const float4 m, const float wxS) {
  float4 s;
  s.x = fmaf(q.w + m.y, wxS, q.x);
  s.y = __fadd_rn(q.y, m.z);
  s.z = __fadd_rn(q.z, m.w);
  s.w = BOTH ? m.x : q.w;  // (only BOTH streams read it)
  return s;
}

// Stream the listed segments, 32 stream positions at a time.  Producer: every lane fetches one source of the
// next tile (straight into registers, one tile ahead; the positions are L2-resident), moves the current
// one into the chunk's frame and stores it in the shared double buffer.  Consumer: every lane evaluates
// STEPS sources of the tile against its pair of targets.  Positions past the end of the stream become idle
// sources ~1e11 away, which contribute exact zeros.
template <bool COUL, bool CUT, bool ENERGY, bool STATS, bool BOTH>
__device__ __forceinline__ void run_stream(const ChunkArgs& A, const PairConsts& c, WarpShared& sh, const unsigned tile_a,
                                           const int lane, const int total, const float wxS, const Targets& t, Accum& acc,
                                           const PassConsts& k, unsigned long long* st) {
  if (total == 0) return;
  const int ntile = (total + 31) >> 5;
  const int ph = lane % NPH;
  Cursor cu;
  cu.cur = 0;
  cu.end = sh.cum[1];
  cu.rec = sh.seg[0];
  cu.flag = BOTH ? sh.flag[0] : 0.f;
  float4 q, m;
  fetch<BOTH>(A, sh, cu, lane, total, q, m);
  // shared-window addresses of this lane's store slot and first load slot in buffer 0 (tile_a is 1024-byte aligned, the
  // second buffer sits 512 bytes above the first: the toggle flips address bit 9)
  unsigned wr_a = tile_a + 16u * (unsigned)lane;
  unsigned rd_a = tile_a + 16u * (unsigned)ph;
#pragma unroll 1
  for (int i = 0; i < ntile; ++i) {
    const float4 s = to_frame<BOTH>(q, m, wxS);
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(wr_a), "f"(s.x), "f"(s.y), "f"(s.z), "f"(s.w) : "memory");
    fetch<BOTH>(A, sh, cu, ((i + 1) << 5) + lane, total, q, m);

    __syncwarp();
    static_assert(STEPS == 4, "written out for 4 steps per tile");
    evaluate<COUL, CUT, ENERGY, BOTH>(lds128<0>(rd_a), t, acc, k, c);
    evaluate<COUL, CUT, ENERGY, BOTH>(lds128<NPH * 16>(rd_a), t, acc, k, c);
    evaluate<COUL, CUT, ENERGY, BOTH>(lds128<NPH * 32>(rd_a), t, acc, k, c);
    evaluate<COUL, CUT, ENERGY, BOTH>(lds128<NPH * 48>(rd_a), t, acc, k, c);
    wr_a ^= 512u;
    rd_a ^= 512u;
  }
  __syncwarp();
  if (STATS && lane == 0) {
    st[0] += (unsigned long long)total;
    st[1] += (unsigned long long)ntile;
    st[2] += 32ull * T * (unsigned long long)ntile;
  }
}

// Bounding box of the chunk in the frame of a pass.
struct Box {
  float lo_x, hi_x, lo_y, hi_y, lo_z, hi_z;
};

// One pass of a chunk over one source species: list the segments (lanes run over the rows of the source
// grid), stream them whenever the list is full and at the end.
// BOTH: the two species share one grid geometry (gs = either) and the pass lists the segments of both, every row
// once: a "round" is then a (periodic image, species) pair.
template <bool COUL, bool CUT, bool ENERGY, bool STATS, bool BOTH>
__device__ __forceinline__ void source_pass(const ChunkArgs& A, const PairConsts& c, WarpShared& sh, const unsigned tile_a,
                                            const int lane, const SpeciesGrid& gs, const int rx, const int ry, const int rz,
                                            const Box& b, const Targets& t, Accum& acc, const PassConsts& k,
                                            unsigned long long* st) {
  const float half = 0.5f * gs.wS;
  // a hair of slack covers FP32 rounding of cell-relative coordinates against the cell boundaries
  const float slack = 1.0e-3f * gs.wS;
  // np/nn passes without an explicit cut: beyond r'^2 = 126 the pair term is exactly 0 in this arithmetic
  // (ex2.approx.ftz flushes), so sources farther than that from every target need not be streamed at all --
  // the sums are the same to the last bit of every addend (D23).  pp pairs reach out to r_c (Coulomb).
  const float reach = COUL ? A.rcS : (CUT ? A.rnS : fminf(A.rcS, A.rzeroS));
  const float rc = reach + slack, rc2 = rc * rc;
  const int my_lo = (int)floorf((b.lo_y - rc) * gs.inv_wS + 0.5f), my_hi = (int)floorf((b.hi_y + rc) * gs.inv_wS + 0.5f);
  const int mz_lo = (int)floorf((b.lo_z - rc) * gs.inv_wS + 0.5f), mz_hi = (int)floorf((b.hi_z + rc) * gs.inv_wS + 0.5f);
  const int ny = my_hi - my_lo + 1, nrows = ny * (mz_hi - mz_lo + 1);
  const float inv_ny = 1.0f / (float)ny;
  const int nc = gs.ncell, ncx = gs.ncx;
  const unsigned lt_mask = (1u << lane) - 1u;

  // state of the row batch being listed: 32 rows starting at rbase, `round` = periodic image along x
  int rbase = 0, round = 0;
  int nseg = 0, ax_lo = 0, ax_hi = 0, q_lo = 0, rowbase = 0;
  float yoff = 0.f, zoff = 0.f;
  do {
    int nseg_list = 0, total = 0;
    while (rbase < nrows && nseg_list + 32 <= SEG_CAP) {
      if (round == 0) {  // geometry of this lane's row
        const int r = rbase + lane;
        nseg = 0;
        if (r < nrows) {
          const int rq = (int)(((float)r + 0.5f) * inv_ny);  // r / ny (ny, r < 2^20: exact)
          const int my = my_lo + (r - rq * ny), mz = mz_lo + rq;
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
            nseg = (floor_div(ax_hi, ncx) - q_lo + 1) * (BOTH ? 2 : 1);
            const int ay = wrap_cell(ry + my, nc), az = wrap_cell(rz + mz, nc);
            rowbase = gs.base + (az * nc + ay) * ncx;
          }
        }
      }
      int start = 0, len = 0;
      float xoff = 0.f;
      const int spi = BOTH ? (round & 1) : 0;  // BOTH: species of this round's segments
      if (round < nseg) {
        const int q = q_lo + (BOTH ? round >> 1 : round), qb = q * ncx;
        const int a_lo = max(ax_lo, qb) - qb, a_hi = min(ax_hi, qb + ncx - 1) - qb;
        const int rb = rowbase + (BOTH ? A.g[spi].base - gs.base : 0);
        start = __ldg(A.bin_start + rb + a_lo);
        len = __ldg(A.bin_start + rb + a_hi + 1) - start;
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
        if (BOTH) sh.flag[at] = (float)spi;
      }
      nseg_list += __popc(has);
      total += __shfl_sync(0xffffffffu, incl, 31);
      ++round;
      if (!__any_sync(0xffffffffu, round < nseg)) {
        rbase += 32;
        round = 0;
      }
    }
    // close the list (dummy record for idle lanes, +infinity boundaries) and stream it
    if (lane == 0) {
      sh.seg[nseg_list] = make_float4(0.f, XOFF_IDLE, 0.f, 0.f);
      if (BOTH) sh.flag[nseg_list] = 0.f;
    }
    sh.cum[nseg_list + lane] = lane == 0 ? total : 0x3fffffff;
    if (lane == 0) sh.cum[nseg_list + 32] = 0x3fffffff;
    __syncwarp();
    run_stream<COUL, CUT, ENERGY, STATS, BOTH>(A, c, sh, tile_a, lane, total, gs.wxS, t, acc, k, st);
  } while (rbase < nrows);
}

__device__ __forceinline__ int min_image_cells(int m, int nc) {
  const int hc = nc / 2;
  return m + (m > hc ? -nc : (m < -hc ? nc : 0));
}

// Both passes of one chunk.  The chunk table (k1_cells.cu) makes every chunk COMPACT: up to 8 same-species targets
// from a few neighbouring cells, at most ~16-20 fm apart.  In a dense system that is 8 consecutive particles of a
// row (they span about one cell width); where a species is sparse or clustered the table groups the particles of
// a small block of cells instead.  Compact chunks keep the bounding box tight (few wasted candidates) and the
// frame coordinates small (FP32 ulp of a displacement <= 1e-6 fm).  The frame's origin cell is the middle of the
// targets' cell range.
// MERGE: on identical grids a neutron chunk takes both source species in ONE pass (one listing instead of two: it
// is the listing, not the arithmetic, that a sparse system pays for).
template <bool CUT, bool ENERGY, bool STATS, bool MERGE>
__device__ __forceinline__ void chunk_passes(const ChunkArgs& A, const PairConsts& c, WarpShared& sh, const unsigned tile_a,
                                             const int lane, const int pr, const SpeciesGrid& gt, const int st_sp, const bool chunk_p,
                                             const float4 tp, const int tc, const unsigned active, Accum& acc,
                                             unsigned long long* st) {
  const bool mine = ((active >> lane) & 1u) != 0;
  const int j0 = 0;
  // cell offsets from target 0's cell in the nearest periodic image, then the middle of their range as origin
  const int c0 = __shfl_sync(0xffffffffu, tc, 0);
  int mx = min_image_cells(PASTA_CX(tc) - PASTA_CX(c0), gt.ncx);
  int my = min_image_cells(PASTA_CY(tc) - PASTA_CY(c0), gt.ncell);
  int mz = min_image_cells(PASTA_CZ(tc) - PASTA_CZ(c0), gt.ncell);
  int lo_x = mine ? mx : 0, hi_x = lo_x, lo_y = mine ? my : 0, hi_y = lo_y, lo_z = mine ? mz : 0, hi_z = lo_z;
#pragma unroll
  for (int o = 1; o < T; o <<= 1) {  // targets sit in lanes [0, T)
    lo_x = min(lo_x, __shfl_xor_sync(0xffffffffu, lo_x, o)); hi_x = max(hi_x, __shfl_xor_sync(0xffffffffu, hi_x, o));
    lo_y = min(lo_y, __shfl_xor_sync(0xffffffffu, lo_y, o)); hi_y = max(hi_y, __shfl_xor_sync(0xffffffffu, hi_y, o));
    lo_z = min(lo_z, __shfl_xor_sync(0xffffffffu, lo_z, o)); hi_z = max(hi_z, __shfl_xor_sync(0xffffffffu, hi_z, o));
  }
  const int sx = __shfl_sync(0xffffffffu, (lo_x + hi_x) >> 1, 0), sy = __shfl_sync(0xffffffffu, (lo_y + hi_y) >> 1, 0),
            sz = __shfl_sync(0xffffffffu, (lo_z + hi_z) >> 1, 0);
  mx -= sx; my -= sy; mz -= sz;
  int ox = (PASTA_CX(c0) + sx) % gt.ncx, oy = (PASTA_CY(c0) + sy) % gt.ncell, oz = (PASTA_CZ(c0) + sz) % gt.ncell;
  ox += ox < 0 ? gt.ncx : 0;
  oy += oy < 0 ? gt.ncell : 0;
  oz += oz < 0 ? gt.ncell : 0;
  // ---- pass 0: proton sources, pass 1: neutron sources -------------------------------------------------
  const bool both = MERGE && A.merged != 0 && !chunk_p;
#pragma unroll
  for (int sp = 0; sp < 2; ++sp) {
    if (MERGE && both && sp == 0) continue;  // the neutron pass below lists the protons too
    const SpeciesGrid& gs = A.g[sp];
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
    // bounding box of the round's targets (every other lane mirrors the first one)
    {
      const float Xo = __shfl_sync(0xffffffffu, X, j0), Yo = __shfl_sync(0xffffffffu, Y, j0),
                  Zo = __shfl_sync(0xffffffffu, Z, j0);
      X = mine ? X : Xo;
      Y = mine ? Y : Yo;
      Z = mine ? Z : Zo;
    }
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
    // this lane's pair of targets: 2 pr and 2 pr + 1 (FAR where the chunk has no such target)
    Targets t;
    {
      const float x0 = __shfl_sync(0xffffffffu, X, 2 * pr), x1 = __shfl_sync(0xffffffffu, X, 2 * pr + 1);
      const float y0 = __shfl_sync(0xffffffffu, Y, 2 * pr), y1 = __shfl_sync(0xffffffffu, Y, 2 * pr + 1);
      const float z0 = __shfl_sync(0xffffffffu, Z, 2 * pr), z1 = __shfl_sync(0xffffffffu, Z, 2 * pr + 1);
      const bool v0 = ((active >> (2 * pr)) & 1u) != 0, v1 = ((active >> (2 * pr + 1)) & 1u) != 0;
      t.ntx = make_float2(v0 ? -x0 : FAR, v1 ? -x1 : FAR);
      t.nty = make_float2(v0 ? -y0 : FAR, v1 ? -y1 : FAR);
      t.ntz = make_float2(v0 ? -z0 : FAR, v1 ? -z1 : FAR);
    }
    const bool like = sp == st_sp;
    PassConsts k;
    k.g2a = c.g2a;
    k.gB = like ? c.gB_like : c.gB_unlike;
    k.a = c.a;
    k.B = like ? c.B_like : c.B_unlike;
    k.gB_n = c.gB_like;  // (BOTH: neutron targets; proton sources are unlike, neutron sources like)
    k.B_n = c.B_like;
    // the selected isospin constants stay in registers: without this the tile loop of the unlike-species pass re-derives
    // them from the constant bank every iteration (a compare, two loads, two predicated loads: 5 of its 108 instructions)
    asm volatile("" : "+f"(k.gB), "+f"(k.B));
    if (MERGE && both) {
      k.gB = c.gB_unlike;
      k.B = c.B_unlike;
      source_pass<false, CUT, ENERGY, STATS, true>(A, c, sh, tile_a, lane, gs, rx, ry, rz, b, t, acc, k, st);
    } else if (sp == 0 && chunk_p && A.no_coul == 0) {
      source_pass<true, CUT, ENERGY, STATS, false>(A, c, sh, tile_a, lane, gs, rx, ry, rz, b, t, acc, k, st);
    } else {
      source_pass<false, CUT, ENERGY, STATS, false>(A, c, sh, tile_a, lane, gs, rx, ry, rz, b, t, acc, k, st);
    }
  }
}

// Combine the phases' FP32 partial sums of a chunk in FP64 and write F and e of its targets in original order.
// quantity index q = 4 * (target within the pair) + {fx, fy, fz, e}; a transposing butterfly over the phase bits of
// the lane index leaves every lane with the full sums of nq quantities starting at qbase.
template <bool ENERGY>
__device__ __forceinline__ void write_chunk_results(const ChunkArgs& A, const PairConsts& c, const Accum& acc, const int lane,
                                                    const int slot) {
  const int pr = lane / NPH, ph = lane % NPH;
  double v[8] = {(double)acc.fx.x, (double)acc.fy.x, (double)acc.fz.x, (double)acc.e.x,
                 (double)acc.fx.y, (double)acc.fy.y, (double)acc.fz.y, (double)acc.e.y};
#pragma unroll
  for (int w = NPH / 2; w >= 8; w >>= 1) {  // more than 8 phases: fold the upper ones first
#pragma unroll
    for (int q = 0; q < 8; ++q) v[q] += __shfl_xor_sync(0xffffffffu, v[q], w);
  }
  constexpr int L8 = NPH < 8 ? NPH : 8;
  int qbase = 0;
  int nq = 8;
#pragma unroll
  for (int w = L8 / 2; w >= 1; w >>= 1) {
    const bool upper = (ph & w) != 0;
    const int half = nq / 2;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      if (q < half) {
        const double keep = upper ? v[q + half] : v[q];
        const double give = upper ? v[q] : v[q + half];
        v[q] = keep + __shfl_xor_sync(0xffffffffu, give, w);
      }
    }
    qbase += upper ? half : 0;
    nq = half;
  }
#pragma unroll
  for (int j = 0; j < 8 / L8; ++j) {
    const int q = qbase + j, tgt = 2 * pr + (q >> 2), comp = q & 3;
    const int tgt_slot = __shfl_sync(0xffffffffu, slot, tgt);
    if (ph < L8 && tgt_slot >= 0) {
      const int i = __ldg(A.perm + tgt_slot);
      if (comp < 3) {
        const double Fc = -v[j];  // d was x_j - x_i
        A.F[3 * (int64_t)i + comp] = Fc;
        if (A.kick != 0.0) A.v[3 * (int64_t)i + comp] = A.v[3 * (int64_t)i + comp] + A.kick * Fc;  // as k3_kick_ke_kernel
      } else if (ENERGY) {
        // every target met itself once in its own species' pass at r = 0: remove V(0) = a + b + c
        A.e[i] = 0.5 * (v[j] - (double)c.v_self);
      }
    }
  }
}

}  // namespace
}  // namespace pasta
