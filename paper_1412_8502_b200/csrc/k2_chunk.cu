// K2, production variant -- "chunk" pair-force kernel for sm_100a.
//
// Work decomposition:
//   * a CHUNK is T = 8 consecutive same-species particles of the cell-sorted order (about one cell of that
//     species' grid, so it is spatially compact); one warp owns one chunk.  The 8 targets live in
//     registers, replicated in every lane and packed two by two, so that the pair arithmetic runs as
//     packed FP32 (FFMA2/FADD2/FMUL2: two pairs per issued instruction -- the FMA pipe, not the issue
//     port, is then the binding unit).
//   * LANES run over SOURCES.  For each source species the warp lists the rows of cells (fixed cy, cz)
//     of that species' grid that intersect the chunk's bounding sphere inflated by r_c; a row's cells
//     are contiguous in the sorted arrays, so a row is one segment of slots (two where it crosses the
//     periodic boundary: images are enumerated explicitly, there is no per-pair nearest-image
//     arithmetic and small boxes need no special case).
//   * the segments are streamed 32 slots at a time through a 4-deep cp.async ring (global -> shared,
//     no registers), so the L2 latency of the position loads is off the critical path.
//   * every lane tests its source against the inflated sphere and the survivors are compacted through
//     a 64-entry shared-memory ring (ballot + popc); whenever 32 survivors are queued, each lane takes
//     one and evaluates it against all 8 targets.  The expensive part therefore runs on dense warps
//     although only ~45 % of the raw candidates of a cell stencil lie inside the sphere.
//   * the cut-off needs no test for np/nn pairs when sigma^2 r_c^2 > 126: exp2(-r'^2) flushes to exactly
//     zero there, so out-of-range pairs contribute exactly 0 (D1: plain truncation).  pp pairs carry the
//     screened Coulomb term and are cut explicitly; small r_c selects the explicitly cut path.
//   * per-lane partial sums are FP32 (about 130 terms per target and pass); they are combined across
//     lanes and passes in FP64 by a transposing butterfly, and written in original particle order.
#include "pasta_internal.cuh"

namespace pasta {

namespace {

constexpr int T = 8;            // targets per chunk
constexpr int NP = T / 2;       // packed target pairs
constexpr int WARPS = 4;        // warps (= chunks) per block
constexpr int DEPTH = 4;        // cp.async stages per warp
constexpr int SEG_CAP = 160;    // segment descriptors per warp
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
  int32_t ncell, base;  // cells per side, first bin
  float wS, inv_wS;     // sigma * cell width and its inverse
  double wS_d;          // the same in FP64 (frame shifts between the two grids)
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
  unsigned long long* stats;  // [0] raw candidates, [1] queued candidates, [2] pair evaluations (STATS only)
};

struct __align__(16) Segment {  // slots [start, start + len): one periodic image of part of a row of cells
  int start, len;
  float xoff;  // add to pos4.w (cell x index) to get the cell offset from the frame's reference cell
  float my, mz;  // cell offsets of the row from the reference cell
  int pad[3];
};

struct WarpShared {
  float4 ring[64];
  float4 stage[DEPTH][32];
  Segment seg[SEG_CAP];
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
#pragma unroll
  for (int p = 0; p < NP; ++p) {
    const float2 dx = __fadd2_rn(dup(s.x), t.ntx[p]);
    const float2 dy = __fadd2_rn(dup(s.y), t.nty[p]);
    const float2 dz = __fadd2_rn(dup(s.z), t.ntz[p]);
    // minus r'^2, accumulated with negated operands (free on FFMA2) because MUFU.EX2 takes no negation
    float2 nr2 = __fmul2_rn(neg2(dx), dx);
    nr2 = __ffma2_rn(neg2(dy), dy, nr2);
    nr2 = __ffma2_rn(neg2(dz), dz, nr2);
    float2 u = make_float2(ex2_approx(nr2.x), ex2_approx(nr2.y));
    if (CUT) {
      u.x = nr2.x > -c.rc2s ? u.x : 0.f;
      u.y = nr2.y > -c.rc2s ? u.y : 0.f;
    }
    float2 g = __fmul2_rn(u, __ffma2_rn(k.g2a, u, k.gB));
    float2 V;
    if (ENERGY) V = __fmul2_rn(u, __ffma2_rn(k.a2, u, k.B2));
    if (COUL) {
      // screened Coulomb, cut at r_c, skipped at r = 0 (the self pair and coincident protons, D2):
      // 1/r' := 0 for excluded pairs, which zeroes every Coulomb factor without creating inf * 0
      const bool in0 = nr2.x > -c.rc2s && nr2.x < 0.f, in1 = nr2.y > -c.rc2s && nr2.y < 0.f;
      const float2 rinv = make_float2(in0 ? rsqrt_approx(-nr2.x) : 0.f, in1 ? rsqrt_approx(-nr2.y) : 0.f);
      const float2 nr = __fmul2_rn(nr2, rinv);  // -r'
      const float2 ex = make_float2(ex2_approx(c.kappa * nr.x), ex2_approx(c.kappa * nr.y));
      const float2 tq = __fmul2_rn(ex, rinv);
      if (ENERGY) V = __ffma2_rn(dup(c.alpha_s), tq, V);
      const float2 q = __fmul2_rn(__fadd2_rn(rinv, dup(c.inv_lam_s)), rinv);
      g = __ffma2_rn(__fmul2_rn(dup(c.alpha_s2), tq), q, g);
    }
    acc.fx[p] = __ffma2_rn(g, dx, acc.fx[p]);
    acc.fy[p] = __ffma2_rn(g, dy, acc.fy[p]);
    acc.fz[p] = __ffma2_rn(g, dz, acc.fz[p]);
    if (ENERGY) acc.e[p] = __fadd2_rn(acc.e[p], V);
  }
}

__device__ __forceinline__ int floor_div(int a, int b) {  // b > 0
  const int q = a / b;
  return (a % b < 0) ? q - 1 : q;
}

// State of the compaction ring and of the frame of one pass.
struct Frame {
  float cX, cY, cZ, R2;  // bounding sphere (centre, inflated radius squared) of the chunk in this frame
  float wS;              // sigma * cell width of the source grid
};

// Stream the listed segments: stage 32 slots at a time through the cp.async ring, test, compact into the
// survivor ring, evaluate 32 survivors whenever they are available.
template <bool COUL, bool CUT, bool ENERGY, bool STATS>
__device__ __forceinline__ void run_segments(const ChunkArgs& A, const PairConsts& c, WarpShared& sh, const int lane,
                                             const int nseg, const int ntiles, const Frame& f, const Targets& t,
                                             Accum& acc, const PassConsts& k, int& head, int& tail,
                                             unsigned long long* st) {
  if (nseg == 0) return;
  const unsigned lt_mask = (1u << lane) - 1u;
  // prefetch cursor
  int ps = 0, po = 0;
  int p_start = sh.seg[0].start, p_len = sh.seg[0].len;
  auto issue = [&](int slot) {
    const bool live = ps < nseg;
    const bool in = live && (po + lane < p_len);
    cp_async16(&sh.stage[slot][lane], A.pos4 + (in ? p_start + po + lane : 0), in ? 16 : 0);
    cp_async_commit();
    if (live) {
      po += 32;
      if (po >= p_len) {
        ++ps;
        po = 0;
        if (ps < nseg) {
          p_start = sh.seg[ps].start;
          p_len = sh.seg[ps].len;
        }
      }
    }
  };
#pragma unroll
  for (int d = 0; d < DEPTH; ++d) issue(d);

  int cs = 0, co = 0;
  Segment g = sh.seg[0];
  for (int i = 0; i < ntiles; ++i) {
    cp_async_wait<DEPTH - 1>();
    const int slot = i & (DEPTH - 1);
    const float4 q = sh.stage[slot][lane];
    const bool valid = co + lane < g.len;
    // source position in the frame: cell-relative coordinate + integer cell offset * w'
    const float X = fmaf(q.w + g.xoff, f.wS, q.x), Y = fmaf(g.my, f.wS, q.y), Z = fmaf(g.mz, f.wS, q.z);
    const float dx = X - f.cX, dy = Y - f.cY, dz = Z - f.cZ;
    const bool pass = valid && fmaf(dz, dz, fmaf(dy, dy, dx * dx)) < f.R2;
    issue(slot);  // refill the stage just read (q has been consumed above)
    const unsigned pm = __ballot_sync(0xffffffffu, pass);
    if (pass) sh.ring[(tail + __popc(pm & lt_mask)) & 63] = make_float4(X, Y, Z, 0.f);
    tail += __popc(pm);
    if (STATS && lane == 0) {
      st[0] += (unsigned long long)min(32, g.len - co);
      st[1] += (unsigned long long)__popc(pm);
    }
    co += 32;
    if (co >= g.len) {
      ++cs;
      co = 0;
      if (cs < nseg) g = sh.seg[cs];
    }
    __syncwarp();
    if (tail - head >= 32) {
      const float4 cnd = sh.ring[(head + lane) & 63];
      head += 32;
      evaluate<COUL, CUT, ENERGY>(cnd, t, acc, k, c);
      if (STATS && lane == 0) st[2] += 32ull * T;
      __syncwarp();
    }
  }
  cp_async_wait<0>();
}

// One pass of a chunk over one source species.
template <bool COUL, bool CUT, bool ENERGY, bool STATS>
__device__ __forceinline__ void source_pass(const ChunkArgs& A, const PairConsts& c, WarpShared& sh, const int lane,
                                            const SpeciesGrid& gs, const int rx, const int ry, const int rz,
                                            const Frame& f, const float R, const Targets& t, Accum& acc,
                                            const PassConsts& k, unsigned long long* st) {
  const float half = 0.5f * gs.wS;
  // rows of cells (my, mz) whose slab can intersect the sphere; a hair of slack covers FP32 rounding of the
  // cell-relative coordinates (every candidate is tested individually, so slack costs nothing but time)
  const float slack = 1.0e-3f * gs.wS;
  const int my_lo = (int)floorf((f.cY - R - slack) * gs.inv_wS + 0.5f), my_hi = (int)floorf((f.cY + R + slack) * gs.inv_wS + 0.5f);
  const int mz_lo = (int)floorf((f.cZ - R - slack) * gs.inv_wS + 0.5f), mz_hi = (int)floorf((f.cZ + R + slack) * gs.inv_wS + 0.5f);
  const int ny = my_hi - my_lo + 1, nrows = ny * (mz_hi - mz_lo + 1);
  const unsigned lt_mask = (1u << lane) - 1u;
  const int nc = gs.ncell;
  int head = 0, tail = 0;
  int nseg_list = 0, ntiles = 0;

  for (int rbase = 0; rbase < nrows; rbase += 32) {
    const int r = rbase + lane;
    int nseg = 0, ax_lo = 0, ax_hi = 0, q_lo = 0, rowbase = 0;
    float myf = 0.f, mzf = 0.f;
    if (r < nrows) {
      const int my = my_lo + r % ny, mz = mz_lo + r / ny;
      myf = (float)my;
      mzf = (float)mz;
      const float gy = fmaxf(fabsf(f.cY - myf * gs.wS) - half - slack, 0.f);
      const float gz = fmaxf(fabsf(f.cZ - mzf * gs.wS) - half - slack, 0.f);
      const float rem = f.R2 - gy * gy - gz * gz;
      if (rem > 0.f) {
        const float xr = sqrtf(rem) + slack;
        ax_lo = rx + (int)floorf((f.cX - xr) * gs.inv_wS + 0.5f);
        ax_hi = rx + (int)floorf((f.cX + xr) * gs.inv_wS + 0.5f);
        q_lo = floor_div(ax_lo, nc);
        nseg = floor_div(ax_hi, nc) - q_lo + 1;
        int ay = (ry + my) % nc, az = (rz + mz) % nc;
        ay += ay < 0 ? nc : 0;
        az += az < 0 ? nc : 0;
        rowbase = gs.base + (az * nc + ay) * nc;
      }
    }
    for (int round = 0; __any_sync(0xffffffffu, round < nseg); ++round) {
      if (nseg_list + 32 > SEG_CAP) {  // (warp-uniform) list full: stream what is there
        __syncwarp();
        run_segments<COUL, CUT, ENERGY, STATS>(A, c, sh, lane, nseg_list, ntiles, f, t, acc, k, head, tail, st);
        nseg_list = 0;
        ntiles = 0;
        __syncwarp();
      }
      bool has = round < nseg;
      Segment sg;
      sg.start = 0;
      sg.len = 0;
      if (has) {
        const int q = q_lo + round, qb = q * nc;
        const int a_lo = max(ax_lo, qb) - qb, a_hi = min(ax_hi, qb + nc - 1) - qb;
        sg.start = __ldg(A.bin_start + rowbase + a_lo);
        sg.len = __ldg(A.bin_start + rowbase + a_hi + 1) - sg.start;
        sg.xoff = (float)(qb - rx);
        sg.my = myf;
        sg.mz = mzf;
        has = sg.len > 0;
      }
      const unsigned m = __ballot_sync(0xffffffffu, has);
      if (has) sh.seg[nseg_list + __popc(m & lt_mask)] = sg;
      nseg_list += __popc(m);
      ntiles += __reduce_add_sync(0xffffffffu, has ? (sg.len + 31) >> 5 : 0);
    }
  }
  __syncwarp();
  run_segments<COUL, CUT, ENERGY, STATS>(A, c, sh, lane, nseg_list, ntiles, f, t, acc, k, head, tail, st);
  if (tail > head) {  // drain the ring; idle lanes take a far-away source that contributes exactly zero
    float4 cnd = sh.ring[(head + lane) & 63];
    if (head + lane >= tail) cnd = make_float4(FAR, FAR, FAR, 0.f);
    evaluate<COUL, CUT, ENERGY>(cnd, t, acc, k, c);
    if (STATS && lane == 0) st[2] += 32ull * T;
  }
  __syncwarp();
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
__global__ void __launch_bounds__(WARPS * 32, 3) k2_chunk_kernel(const ChunkArgs A, const PairConsts c) {
  __shared__ WarpShared shared[WARPS];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
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
  const int ox = oc & 1023, oy = (oc >> 10) & 1023, oz = (oc >> 20) & 1023;
  // cell offset from the origin cell, taken in the nearest periodic image (chunks may wrap a row end)
  const int mx = min_image_cells((tc & 1023) - ox, gt.ncell);
  const int my = min_image_cells(((tc >> 10) & 1023) - oy, gt.ncell);
  const int mz = min_image_cells(((tc >> 20) & 1023) - oz, gt.ncell);

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
    if (gs.ncell == gt.ncell) {  // same grid geometry (always true for the chunk's own species)
      X = fmaf((float)mx, gs.wS, tp.x);
      Y = fmaf((float)my, gs.wS, tp.y);
      Z = fmaf((float)mz, gs.wS, tp.z);
    } else {
      const double cx0 = ((double)ox + 0.5) * gt.wS_d, cy0 = ((double)oy + 0.5) * gt.wS_d, cz0 = ((double)oz + 0.5) * gt.wS_d;
      rx = min(gs.ncell - 1, (int)(cx0 / gs.wS_d));
      ry = min(gs.ncell - 1, (int)(cy0 / gs.wS_d));
      rz = min(gs.ncell - 1, (int)(cz0 / gs.wS_d));
      X = (float)((double)tp.x + (double)mx * gt.wS_d + (cx0 - ((double)rx + 0.5) * gs.wS_d));
      Y = (float)((double)tp.y + (double)my * gt.wS_d + (cy0 - ((double)ry + 0.5) * gs.wS_d));
      Z = (float)((double)tp.z + (double)mz * gt.wS_d + (cz0 - ((double)rz + 0.5) * gs.wS_d));
    }
    // bounding sphere of the chunk
    float lo_x = X, hi_x = X, lo_y = Y, hi_y = Y, lo_z = Z, hi_z = Z;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo_x = fminf(lo_x, __shfl_xor_sync(0xffffffffu, lo_x, o));
      hi_x = fmaxf(hi_x, __shfl_xor_sync(0xffffffffu, hi_x, o));
      lo_y = fminf(lo_y, __shfl_xor_sync(0xffffffffu, lo_y, o));
      hi_y = fmaxf(hi_y, __shfl_xor_sync(0xffffffffu, hi_y, o));
      lo_z = fminf(lo_z, __shfl_xor_sync(0xffffffffu, lo_z, o));
      hi_z = fmaxf(hi_z, __shfl_xor_sync(0xffffffffu, hi_z, o));
    }
    Frame f;
    f.cX = 0.5f * (lo_x + hi_x);
    f.cY = 0.5f * (lo_y + hi_y);
    f.cZ = 0.5f * (lo_z + hi_z);
    f.wS = gs.wS;
    float rho2 = (X - f.cX) * (X - f.cX) + (Y - f.cY) * (Y - f.cY) + (Z - f.cZ) * (Z - f.cZ);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) rho2 = fmaxf(rho2, __shfl_xor_sync(0xffffffffu, rho2, o));
    const float R = A.rcS + sqrtf(rho2) * 1.0001f + 1.0e-4f;
    f.R2 = R * R;

    Targets t;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
      const float x0 = __shfl_sync(0xffffffffu, X, 2 * p), x1 = __shfl_sync(0xffffffffu, X, 2 * p + 1);
      const float y0 = __shfl_sync(0xffffffffu, Y, 2 * p), y1 = __shfl_sync(0xffffffffu, Y, 2 * p + 1);
      const float z0 = __shfl_sync(0xffffffffu, Z, 2 * p), z1 = __shfl_sync(0xffffffffu, Z, 2 * p + 1);
      const bool v0 = 2 * p < nvalid, v1 = 2 * p + 1 < nvalid;
      t.ntx[p] = make_float2(v0 ? -x0 : FAR, v1 ? -x1 : FAR);
      t.nty[p] = make_float2(v0 ? -y0 : FAR, v1 ? -y1 : FAR);
      t.ntz[p] = make_float2(v0 ? -z0 : FAR, v1 ? -z1 : FAR);
    }
    const bool like = sp == st_sp;
    PassConsts k;
    k.g2a = dup(c.g2a);
    k.gB = dup(like ? c.gB_like : c.gB_unlike);
    k.a2 = dup(c.a);
    k.B2 = dup(like ? c.B_like : c.B_unlike);
    if (chunk_p && sp == 0)
      source_pass<true, CUT, ENERGY, STATS>(A, c, sh, lane, gs, rx, ry, rz, f, R, t, acc, k, st);
    else
      source_pass<false, CUT, ENERGY, STATS>(A, c, sh, lane, gs, rx, ry, rz, f, R, t, acc, k, st);
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
  ChunkArgs A;
  A.N = (int32_t)s->N;
  A.Np = (int32_t)s->Np;
  A.n_chunks_p = (int32_t)((s->Np + T - 1) / T);
  A.n_chunks = A.n_chunks_p + (int32_t)((s->N - s->Np + T - 1) / T);
  for (int sp = 0; sp < 2; ++sp) {
    A.g[sp].ncell = s->grid_sp[sp].ncell;
    A.g[sp].base = (int32_t)s->bin_base[sp];
    A.g[sp].wS_d = sigma * s->grid_sp[sp].w;
    A.g[sp].wS = (float)A.g[sp].wS_d;
    A.g[sp].inv_wS = (float)(1.0 / A.g[sp].wS_d);
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
