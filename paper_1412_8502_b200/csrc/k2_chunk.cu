// K2, production variant -- "chunk" pair-force kernel for sm_100a.
//
// Work decomposition:
//   * a CHUNK is T = 8 consecutive same-species particles of the cell-sorted order (spatially compact);
//     one warp owns one chunk.  The 8 targets live in registers, replicated in every lane, packed two
//     by two so that the pair arithmetic runs on the packed FP32 pipe (FFMA2/FADD2/FMUL2: two pairs per
//     issued instruction -- the FMA pipe, not the issue port, is then the binding unit).
//   * LANES run over SOURCES.  For each source species the warp walks the rows of cells (fixed cy, cz)
//     that intersect the chunk's bounding sphere inflated by r_c; a row's cells are contiguous in the
//     sorted arrays, so sources arrive as coalesced float4 loads.  Periodic images are enumerated
//     explicitly (each row is split at the box boundary), so there is no per-pair nearest-image
//     arithmetic and small boxes need no special case.
//   * every lane tests its source against the inflated sphere and the survivors are compacted through
//     a 64-entry shared-memory ring (ballot + popc); whenever 32 survivors are queued, each lane takes
//     one and evaluates it against all 8 targets.  The expensive part therefore runs on dense warps
//     even though only ~45 % of the raw candidates of a cell stencil lie inside the sphere.
//   * the cut-off needs no test for np/nn pairs when sigma^2 r_c^2 > 126: exp2(-r'^2) flushes to exactly
//     zero there, so out-of-range pairs contribute exactly 0 (D1: plain truncation).  pp pairs carry the
//     screened Coulomb term and are cut explicitly; small r_c selects the explicitly cut path.
//   * per-lane partial sums are FP32 (about 130 terms per target and pass); they are combined across
//     lanes and passes in FP64 by a transposing butterfly, and written in original particle order.
#include "pasta_internal.cuh"

namespace pasta {

namespace {

constexpr int T = 8;           // targets per chunk
constexpr int NP = T / 2;      // packed target pairs
constexpr int WARPS = 4;       // warps (= chunks) per block
constexpr float FAR = 1.0e10f; // coordinate of padding sources/targets: exp2(-FAR^2) == 0, 0 * FAR == 0

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

struct ChunkArgs {
  int32_t N, Np;
  int32_t n_chunks_p, n_chunks;
  int32_t ncell, nc3;
  float wS;      // sigma * cell width
  float inv_wS;  // 1 / (sigma * cell width)
  float rcS;     // sigma * r_c
  const float4* pos4;
  const int32_t* cxyz;
  const int32_t* bin_start;
  const int32_t* perm;
  double* F;
  double* e;
  unsigned long long* stats;  // [0] raw candidates, [1] queued candidates, [2] pair evaluations (STATS only)
};

struct Segment {  // a run of sorted slots [start, end) that is one periodic image of part of a cell row
  int start, end;
  float xoff;  // add to pos4.w (cell x index) to get the cell offset from the chunk's origin cell
  float my, mz;  // cell offsets of the row from the origin cell
};

struct WarpShared {
  float4 ring[64];
  Segment seg[32];
};

// Accumulators and targets of one warp: everything is replicated in all lanes except the accumulators,
// which hold this lane's partial sums.  Convention: d = x_j - x_i (so accumulated forces are -F_i).
struct Targets {
  float2 ntx[NP], nty[NP], ntz[NP];  // minus the target coordinates, packed two targets per register pair
};
struct Accum {
  float2 fx[NP], fy[NP], fz[NP], e[NP];
};

template <bool COUL, bool CUT, bool ENERGY>
__device__ __forceinline__ void evaluate(const float4 s, const Targets& t, Accum& acc, const float2 g2a,
                                         const float2 gB, const float2 a2, const float2 B2, const PairConsts& c) {
  const float2 sx = dup(s.x), sy = dup(s.y), sz = dup(s.z);
#pragma unroll
  for (int k = 0; k < NP; ++k) {
    const float2 dx = __fadd2_rn(sx, t.ntx[k]);
    const float2 dy = __fadd2_rn(sy, t.nty[k]);
    const float2 dz = __fadd2_rn(sz, t.ntz[k]);
    float2 r2 = __fmul2_rn(dx, dx);
    r2 = __ffma2_rn(dy, dy, r2);
    r2 = __ffma2_rn(dz, dz, r2);
    float2 u = make_float2(ex2_approx(-r2.x), ex2_approx(-r2.y));
    if (CUT && !COUL) {
      u.x = r2.x < c.rc2s ? u.x : 0.f;
      u.y = r2.y < c.rc2s ? u.y : 0.f;
    }
    float2 g = __fmul2_rn(u, __ffma2_rn(g2a, u, gB));
    float2 V;
    if (ENERGY) V = __fmul2_rn(u, __ffma2_rn(a2, u, B2));
    if (COUL) {
      // screened Coulomb, cut at r_c, skipped at r = 0 (the self pair and coincident protons, D2)
      const bool in0 = r2.x < c.rc2s && r2.x > 0.f, in1 = r2.y < c.rc2s && r2.y > 0.f;
      // 1/r' := 0 for excluded pairs, which zeroes every Coulomb factor below without creating inf * 0
      const float2 rinv = make_float2(in0 ? rsqrt_approx(r2.x) : 0.f, in1 ? rsqrt_approx(r2.y) : 0.f);
      const float2 r = __fmul2_rn(r2, rinv);
      const float2 ex = make_float2(ex2_approx(-c.kappa * r.x), ex2_approx(-c.kappa * r.y));
      const float2 tq = __fmul2_rn(ex, rinv);
      if (CUT) {  // the nuclear terms are not yet negligible at r_c: cut them too
        u.x = r2.x < c.rc2s ? u.x : 0.f;
        u.y = r2.y < c.rc2s ? u.y : 0.f;
        g = __fmul2_rn(u, __ffma2_rn(g2a, u, gB));
        if (ENERGY) V = __fmul2_rn(u, __ffma2_rn(a2, u, B2));
      }
      if (ENERGY) V = __ffma2_rn(dup(c.alpha_s), tq, V);
      const float2 q = __fmul2_rn(__fadd2_rn(rinv, dup(c.inv_lam_s)), rinv);
      g = __ffma2_rn(__fmul2_rn(dup(c.alpha_s2), tq), q, g);
    }
    acc.fx[k] = __ffma2_rn(g, dx, acc.fx[k]);
    acc.fy[k] = __ffma2_rn(g, dy, acc.fy[k]);
    acc.fz[k] = __ffma2_rn(g, dz, acc.fz[k]);
    if (ENERGY) acc.e[k] = __fadd2_rn(acc.e[k], V);
  }
}

__device__ __forceinline__ int floor_div(int a, int b) {  // b > 0
  int q = a / b;
  return (a % b < 0) ? q - 1 : q;
}

// One pass of a chunk over one source species.
template <bool COUL, bool CUT, bool ENERGY, bool STATS>
__device__ __forceinline__ void source_pass(const ChunkArgs& A, const PairConsts& c, WarpShared& sh, const int lane,
                                            const int sp, const int ox, const int oy, const int oz, const float cX,
                                            const float cY, const float cZ, const float R, const Targets& t,
                                            Accum& acc, const float B, const float gB, unsigned long long* st) {
  const float2 g2a = dup(c.g2a), gB2 = dup(gB), a2 = dup(c.a), B2 = dup(B);
  const float R2 = R * R;
  const float half = 0.5f * A.wS;
  // rows of cells (my, mz) whose slab can intersect the sphere; a hair of slack covers FP32 rounding of the
  // cell-relative coordinates (every candidate is tested individually, so slack costs nothing but time)
  const float slack = 1.0e-3f * A.wS;
  const int my_lo = (int)floorf((cY - R - slack) * A.inv_wS + 0.5f), my_hi = (int)floorf((cY + R + slack) * A.inv_wS + 0.5f);
  const int mz_lo = (int)floorf((cZ - R - slack) * A.inv_wS + 0.5f), mz_hi = (int)floorf((cZ + R + slack) * A.inv_wS + 0.5f);
  const int ny = my_hi - my_lo + 1, nrows = ny * (mz_hi - mz_lo + 1);
  const unsigned lt_mask = (1u << lane) - 1u;
  int head = 0, tail = 0;

  for (int rbase = 0; rbase < nrows; rbase += 32) {
    const int r = rbase + lane;
    int nseg = 0, ax_lo = 0, ax_hi = 0, q_lo = 0, rowbase = 0;
    float myf = 0.f, mzf = 0.f;
    if (r < nrows) {
      const int my = my_lo + r % ny, mz = mz_lo + r / ny;
      myf = (float)my;
      mzf = (float)mz;
      const float gy = fmaxf(fabsf(cY - myf * A.wS) - half - slack, 0.f);
      const float gz = fmaxf(fabsf(cZ - mzf * A.wS) - half - slack, 0.f);
      const float rem = R2 - gy * gy - gz * gz;
      if (rem > 0.f) {
        const float xr = sqrtf(rem) + slack;
        ax_lo = ox + (int)floorf((cX - xr) * A.inv_wS + 0.5f);
        ax_hi = ox + (int)floorf((cX + xr) * A.inv_wS + 0.5f);
        q_lo = floor_div(ax_lo, A.ncell);
        nseg = floor_div(ax_hi, A.ncell) - q_lo + 1;
        int ay = (oy + my) % A.ncell, az = (oz + mz) % A.ncell;
        ay += ay < 0 ? A.ncell : 0;
        az += az < 0 ? A.ncell : 0;
        rowbase = sp * A.nc3 + (az * A.ncell + ay) * A.ncell;
      }
    }
    for (int round = 0; __any_sync(0xffffffffu, round < nseg); ++round) {
      bool has = round < nseg;
      Segment sg;
      sg.start = sg.end = 0;
      if (has) {
        const int q = q_lo + round, qb = q * A.ncell;
        const int a_lo = max(ax_lo, qb) - qb, a_hi = min(ax_hi, qb + A.ncell - 1) - qb;
        sg.start = __ldg(A.bin_start + rowbase + a_lo);
        sg.end = __ldg(A.bin_start + rowbase + a_hi + 1);
        sg.xoff = (float)(qb - ox);
        sg.my = myf;
        sg.mz = mzf;
        has = sg.end > sg.start;
      }
      const unsigned m = __ballot_sync(0xffffffffu, has);
      if (has) sh.seg[__popc(m & lt_mask)] = sg;
      const int nlist = __popc(m);
      __syncwarp();
      for (int s = 0; s < nlist; ++s) {
        const Segment g = sh.seg[s];
        for (int p0 = g.start; p0 < g.end; p0 += 32) {
          const int p = p0 + lane;
          const bool valid = p < g.end;
          float4 q = make_float4(FAR, FAR, FAR, 0.f);
          if (valid) q = __ldg(A.pos4 + p);
          // source position in the chunk's frame: cell-relative coordinate + integer cell offset * w'
          const float X = fmaf(q.w + g.xoff, A.wS, q.x), Y = fmaf(g.my, A.wS, q.y), Z = fmaf(g.mz, A.wS, q.z);
          const float dx = X - cX, dy = Y - cY, dz = Z - cZ;
          const bool pass = valid && fmaf(dz, dz, fmaf(dy, dy, dx * dx)) < R2;
          const unsigned pm = __ballot_sync(0xffffffffu, pass);
          if (pass) sh.ring[(tail + __popc(pm & lt_mask)) & 63] = make_float4(X, Y, Z, 0.f);
          tail += __popc(pm);
          if (STATS && lane == 0) {
            st[0] += (unsigned long long)min(32, g.end - p0);
            st[1] += (unsigned long long)__popc(pm);
          }
          __syncwarp();
          if (tail - head >= 32) {
            const float4 cnd = sh.ring[(head + lane) & 63];
            head += 32;
            evaluate<COUL, CUT, ENERGY>(cnd, t, acc, g2a, gB2, a2, B2, c);
            if (STATS && lane == 0) st[2] += 32ull * T;
            __syncwarp();
          }
        }
      }
      __syncwarp();
    }
  }
  if (tail > head) {  // drain the ring; idle lanes take a far-away source that contributes exactly zero
    float4 cnd = sh.ring[(head + lane) & 63];
    if (head + lane >= tail) cnd = make_float4(FAR, FAR, FAR, 0.f);
    evaluate<COUL, CUT, ENERGY>(cnd, t, acc, g2a, gB2, a2, B2, c);
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
      // keep quantities [q] if lower half-lane, [q + w] if upper; send the other one to the partner
      const double keep = upper ? v[q + w] : v[q];
      const double give = upper ? v[q] : v[q + w];
      v[q] = keep + __shfl_xor_sync(0xffffffffu, give, w);
    }
  }
  return v[0];
}

template <bool CUT, bool ENERGY, bool STATS>
__global__ void __launch_bounds__(WARPS * 32, 3) k2_chunk_kernel(const ChunkArgs A, const PairConsts c) {
  __shared__ WarpShared shared[WARPS];
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int chunk = blockIdx.x * WARPS + wib;
  if (chunk >= A.n_chunks) return;
  WarpShared& sh = shared[wib];

  const bool chunk_p = chunk < A.n_chunks_p;
  const int base = chunk_p ? chunk * T : A.Np + (chunk - A.n_chunks_p) * T;
  const int nvalid = min(T, (chunk_p ? A.Np : A.N) - base);

  // ---- targets: lane l < nvalid holds target l; all other lanes mirror target 0 ------------------------
  const int tl = lane < nvalid ? lane : 0;
  const float4 tp = __ldg(A.pos4 + base + tl);
  const int tc = __ldg(A.cxyz + base + tl);
  const int oc = __shfl_sync(0xffffffffu, tc, 0);
  const int ox = oc & 1023, oy = (oc >> 10) & 1023, oz = (oc >> 20) & 1023;
  // cell offset from the origin cell, taken in the nearest periodic image (chunks may wrap a row end)
  int mx = (tc & 1023) - ox, my = ((tc >> 10) & 1023) - oy, mz = ((tc >> 20) & 1023) - oz;
  const int hc = A.ncell / 2;
  mx += mx > hc ? -A.ncell : (mx < -hc ? A.ncell : 0);
  my += my > hc ? -A.ncell : (my < -hc ? A.ncell : 0);
  mz += mz > hc ? -A.ncell : (mz < -hc ? A.ncell : 0);
  const float X = fmaf((float)mx, A.wS, tp.x), Y = fmaf((float)my, A.wS, tp.y), Z = fmaf((float)mz, A.wS, tp.z);

  // ---- bounding sphere of the chunk ------------------------------------------------------------------
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
  const float cX = 0.5f * (lo_x + hi_x), cY = 0.5f * (lo_y + hi_y), cZ = 0.5f * (lo_z + hi_z);
  float rho2 = (X - cX) * (X - cX) + (Y - cY) * (Y - cY) + (Z - cZ) * (Z - cZ);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) rho2 = fmaxf(rho2, __shfl_xor_sync(0xffffffffu, rho2, o));
  const float R = A.rcS + sqrtf(rho2) * 1.0001f + 1.0e-4f;

  Targets t;
#pragma unroll
  for (int k = 0; k < NP; ++k) {
    const float x0 = __shfl_sync(0xffffffffu, X, 2 * k), x1 = __shfl_sync(0xffffffffu, X, 2 * k + 1);
    const float y0 = __shfl_sync(0xffffffffu, Y, 2 * k), y1 = __shfl_sync(0xffffffffu, Y, 2 * k + 1);
    const float z0 = __shfl_sync(0xffffffffu, Z, 2 * k), z1 = __shfl_sync(0xffffffffu, Z, 2 * k + 1);
    const bool v0 = 2 * k < nvalid, v1 = 2 * k + 1 < nvalid;
    t.ntx[k] = make_float2(v0 ? -x0 : FAR, v1 ? -x1 : FAR);
    t.nty[k] = make_float2(v0 ? -y0 : FAR, v1 ? -y1 : FAR);
    t.ntz[k] = make_float2(v0 ? -z0 : FAR, v1 ? -z1 : FAR);
  }
  Accum acc;
#pragma unroll
  for (int k = 0; k < NP; ++k) acc.fx[k] = acc.fy[k] = acc.fz[k] = acc.e[k] = make_float2(0.f, 0.f);

  unsigned long long st[3] = {0, 0, 0};
  // ---- pass 0: proton sources, pass 1: neutron sources -------------------------------------------------
#pragma unroll 1
  for (int sp = 0; sp < 2; ++sp) {
    const bool like = chunk_p == (sp == 0);
    const float B = like ? c.B_like : c.B_unlike, gB = like ? c.gB_like : c.gB_unlike;
    if (chunk_p && sp == 0)
      source_pass<true, CUT, ENERGY, STATS>(A, c, sh, lane, sp, ox, oy, oz, cX, cY, cZ, R, t, acc, B, gB, st);
    else
      source_pass<false, CUT, ENERGY, STATS>(A, c, sh, lane, sp, ox, oy, oz, cX, cY, cZ, R, t, acc, B, gB, st);
  }

  // ---- combine the lanes' FP32 partials in FP64: quantity index = 4 * target + {fx, fy, fz, e} ------------
  double v[32];
#pragma unroll
  for (int k = 0; k < NP; ++k) {
    v[8 * k + 0] = (double)acc.fx[k].x; v[8 * k + 1] = (double)acc.fy[k].x;
    v[8 * k + 2] = (double)acc.fz[k].x; v[8 * k + 3] = (double)acc.e[k].x;
    v[8 * k + 4] = (double)acc.fx[k].y; v[8 * k + 5] = (double)acc.fy[k].y;
    v[8 * k + 6] = (double)acc.fz[k].y; v[8 * k + 7] = (double)acc.e[k].y;
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
  A.ncell = s->grid.ncell;
  A.nc3 = (int32_t)s->grid.nc3;
  A.wS = (float)(sigma * s->grid.w);
  A.inv_wS = (float)(1.0 / (sigma * s->grid.w));
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
