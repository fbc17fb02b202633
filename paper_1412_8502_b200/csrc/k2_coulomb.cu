// K2, the Coulomb half of the paper's own range split ("we do not use a cutoff radius
// for the Coulomb potential ... each proton interacts with the nearest periodic image of every other proton";
// in IUMD this sum ran on the K20s).  With pasta_params.coulomb_all_pairs the chunk / list kernels
// evaluate the nuclear terms only (cut at r_nuc) and this kernel adds, for every proton, the screened Coulomb term of
// ALL other protons at their nearest image -- a cube of side L around the target, no radial cut-off, N_p^2 pairs.
//
// Layout: the protons are the sorted slots [0, Np).  A first kernel writes their positions as box fractions
// u = x / L, as a PAIR of FP32 numbers (hi = the nearest float, lo = the rest): one float alone has an ulp of 6e-8,
// i.e. 1e-5 .. 4e-5 fm in boxes of 170 .. 690 fm, and the Coulomb force of a proton pair 1 fm apart (1.4 MeV/fm) would
// then be off by 2e-5 of itself -- over the force gate in a dilute system.  The difference of two hi parts is exact to
// its own last bit, the lo parts add the representation error back: du is good to 1e-7 of itself.  The pair kernel is
// the chunk kernel's evaluation loop without any listing: one warp owns 8 consecutive
// proton slots, lane = (target pair, phase), the whole proton array streams through a shared double buffer 32 at a
// time, and the nearest image is per pair: du -= rint(du), rint by the 1.5 * 2^23 trick (two packed adds, no
// conversion instruction).  In box fractions, with r = L |du|:
//   V = (alpha / L) t,  t = exp2(-kL |du|) / |du|,  kL = log2(e) L / lambda
//   F_i = -(alpha / L) sum_j t (1/|du| / L + 1/lambda) / |du| * du
// FP32 partial sums per lane (1/8 of the protons), combined over the phases in FP64, ADDED to F and e.
#include "pasta_internal.cuh"

namespace pasta {

namespace {

constexpr int CW = 4;  // warps (groups of 8 targets) per block

struct CoulArgs {
  int32_t Np;
  int32_t t_lo, t_hi;  // proton slots the launch covers
  int32_t w_lo, w_hi;  // target sharding: a target is evaluated iff its OWNER slot lies in [w_lo, w_hi)
  const int32_t* owner;  // chunk path: first slot of the target's chunk (the rank that owns the chunk owns the target, so
                         // that a particle is complete on one rank); NULL (list path): the target's own slot
  const float4* cpos;  // [2 Np] box fractions: [2 t] = hi parts (.w = 1), [2 t + 1] = lo parts
  const int32_t* perm;
  double* F;
  double* e;
  float kL, invL, invlam;
  double aL;  // alpha / L
};

__global__ void k2c_fractions_kernel(int32_t Np, const double* __restrict__ x, const int32_t* __restrict__ perm, double invL,
                                     float4* __restrict__ cpos) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= Np) return;
  const int64_t i = perm[t];
  float hi[3], lo[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const double u = x[3 * i + a] * invL;
    hi[a] = (float)u;
    lo[a] = (float)(u - (double)hi[a]);
  }
  cpos[2 * t] = make_float4(hi[0], hi[1], hi[2], 1.f);
  cpos[2 * t + 1] = make_float4(lo[0], lo[1], lo[2], 0.f);
}

__device__ __forceinline__ float ex2f(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqf(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float2 dup2(float a) { return make_float2(a, a); }

struct CAcc {
  float2 fx, fy, fz, e;
};

// nearest image of a difference of box fractions: d = (s_hi - t_hi) - rint(s_hi - t_hi) + (s_lo - t_lo); every step but
// the last addition is exact
__device__ __forceinline__ float2 image_difference(const float s_hi, const float2 nt_hi, const float s_lo, const float2 nt_lo) {
  const float2 a = __fadd2_rn(dup2(s_hi), nt_hi);
  const float2 magic = dup2(12582912.f);  // 1.5 * 2^23: adding it rounds to the nearest integer
  const float2 r = __fadd2_rn(__fadd2_rn(a, magic), make_float2(-12582912.f, -12582912.f));
  return __fadd2_rn(__fadd2_rn(a, make_float2(-r.x, -r.y)), __fadd2_rn(dup2(s_lo), nt_lo));
}
struct CTargets {
  float2 hx, hy, hz, lx, ly, lz;  // minus the two targets' hi and lo parts
};

template <bool ENERGY>
__device__ __forceinline__ void coulomb_step(const float4 s, const float4 sl, const CTargets& tg, CAcc& acc,
                                             const CoulArgs& A) {
  const float2 dx = image_difference(s.x, tg.hx, sl.x, tg.lx);
  const float2 dy = image_difference(s.y, tg.hy, sl.y, tg.ly);
  const float2 dz = image_difference(s.z, tg.hz, sl.z, tg.lz);
  float2 r2 = __fmul2_rn(dx, dx);
  r2 = __ffma2_rn(dy, dy, r2);
  r2 = __ffma2_rn(dz, dz, r2);
  // the self pair, coincident protons (D2) and padding sources (.w == 0) get 1/|du| := 0, which zeroes every factor
  const bool live = s.w != 0.f;
  const float2 rinv = make_float2(live && r2.x > 0.f ? rsqf(r2.x) : 0.f, live && r2.y > 0.f ? rsqf(r2.y) : 0.f);
  const float2 nr = __fmul2_rn(__fmul2_rn(r2, rinv), dup2(-A.kL));  // -kL |du|
  const float2 t = __fmul2_rn(make_float2(ex2f(nr.x), ex2f(nr.y)), rinv);
  const float2 q = __fmul2_rn(__ffma2_rn(rinv, dup2(A.invL), dup2(A.invlam)), rinv);
  const float2 g = __fmul2_rn(t, q);
  if (ENERGY) acc.e = __fadd2_rn(acc.e, t);
  acc.fx = __ffma2_rn(g, dx, acc.fx);
  acc.fy = __ffma2_rn(g, dy, acc.fy);
  acc.fz = __ffma2_rn(g, dz, acc.fz);
}

template <bool ENERGY>
__global__ void __launch_bounds__(CW * 32) k2c_pairs_kernel(const CoulArgs A) {
  __shared__ float4 tile[CW][2][64];  // double buffer of 32 sources: hi parts, then lo parts
  const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
  const int pr = lane >> 3, ph = lane & 7;
  const int t0 = A.t_lo + 8 * (blockIdx.x * CW + wib);
  if (t0 >= A.t_hi) return;
  const int ta = t0 + 2 * pr, tb = ta + 1;
  bool mine[2];
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const int ts = ta + k;
    const int ow = ts < A.t_hi ? (A.owner ? __ldg(A.owner + ts) : ts) : -1;
    mine[k] = ow >= A.w_lo && ow < A.w_hi;
  }
  if (!__any_sync(0xffffffffu, mine[0] || mine[1])) return;  // another rank's targets
  const int ca = 2 * min(ta, A.Np - 1), cb = 2 * min(tb, A.Np - 1);
  const float4 pa = __ldg(A.cpos + ca), pb = __ldg(A.cpos + cb), qa = __ldg(A.cpos + ca + 1), qb = __ldg(A.cpos + cb + 1);
  CTargets t;
  t.hx = make_float2(-pa.x, -pb.x); t.hy = make_float2(-pa.y, -pb.y); t.hz = make_float2(-pa.z, -pb.z);
  t.lx = make_float2(-qa.x, -qb.x); t.ly = make_float2(-qa.y, -qb.y); t.lz = make_float2(-qa.z, -qb.z);
  CAcc acc;
  acc.fx = acc.fy = acc.fz = acc.e = make_float2(0.f, 0.f);
  const int ntile = (A.Np + 31) >> 5;
  const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
  float4 q = lane < A.Np ? __ldg(A.cpos + 2 * lane) : zero, ql = lane < A.Np ? __ldg(A.cpos + 2 * lane + 1) : zero;
#pragma unroll 1
  for (int i = 0; i < ntile; ++i) {
    const int o = i & 1;
    tile[wib][o][lane] = q;
    tile[wib][o][32 + lane] = ql;
    const int nxt = ((i + 1) << 5) + lane;
    q = nxt < A.Np ? __ldg(A.cpos + 2 * nxt) : zero;
    ql = nxt < A.Np ? __ldg(A.cpos + 2 * nxt + 1) : zero;
    __syncwarp();
#pragma unroll
    for (int j = 0; j < 4; ++j) coulomb_step<ENERGY>(tile[wib][o][ph + 8 * j], tile[wib][o][32 + ph + 8 * j], t, acc, A);
  }
  // the 8 phases of a target pair meet in FP64
  double v[8] = {(double)acc.fx.x, (double)acc.fy.x, (double)acc.fz.x, (double)acc.e.x,
                 (double)acc.fx.y, (double)acc.fy.y, (double)acc.fz.y, (double)acc.e.y};
#pragma unroll
  for (int k = 0; k < 8; ++k) {
#pragma unroll
    for (int w = 4; w >= 1; w >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], w);
  }
  if (ph == 0) {
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      const int ts = ta + k;
      if (mine[k]) {
        const int64_t i = __ldg(A.perm + ts);
        A.F[3 * i + 0] -= A.aL * v[4 * k + 0];  // du was u_j - u_i
        A.F[3 * i + 1] -= A.aL * v[4 * k + 1];
        A.F[3 * i + 2] -= A.aL * v[4 * k + 2];
        if (ENERGY) A.e[i] += 0.5 * A.aL * v[4 * k + 3];
      }
    }
  }
}

}  // namespace

// Adds the all-pairs nearest-image Coulomb term of the protons to F (and e) of the current sorted order.
int k2_coulomb_all_pairs(Sim* s, bool with_energy) {
  if (s->Np < 1) return PASTA_OK;
  if (s->sort_kind != 0 && s->sort_kind != 2) {
    set_error("coulomb_all_pairs: the proton slots of the chunk / list sort are needed");
    return PASTA_ESTATE;
  }
  PASTA_TRY(buffer_reserve(s, &s->cpos, 2 * sizeof(float4) * (size_t)s->Np));
  CoulArgs A;
  A.Np = (int32_t)s->Np;
  A.w_lo = s->shard.slot_lo;
  A.w_hi = s->shard.slot_hi;
  A.owner = s->sort_kind == 0 ? s->chunk_first.as<int32_t>() : nullptr;
  // list path: a target is owned through its own slot, so the launch covers the window only; chunk path: every
  // proton group looks its owner up and the others' return at once
  A.t_lo = A.owner ? 0 : (s->shard.slot_lo < 0 ? 0 : s->shard.slot_lo);
  A.t_hi = A.owner ? A.Np : (s->shard.slot_hi > A.Np ? A.Np : s->shard.slot_hi);
  A.cpos = s->cpos.as<float4>();
  A.perm = s->perm.as<int32_t>();
  A.F = s->F.as<double>();
  A.e = s->e.as<double>();
  A.kL = (float)(1.4426950408889634074 * s->L / s->prm.lambda);
  A.invL = (float)(1.0 / s->L);
  A.invlam = (float)(1.0 / s->prm.lambda);
  A.aL = s->prm.alpha_hbarc / s->L;
  k2c_fractions_kernel<<<grid_for(s->Np, 256), 256, 0, s->stream>>>(A.Np, s->x.as<double>(), A.perm, 1.0 / s->L,
                                                                    s->cpos.as<float4>());
  s->launches += 1;
  if (A.t_hi > A.t_lo) {
    const int groups = (A.t_hi - A.t_lo + 7) / 8;
    const int grid = (groups + CW - 1) / CW;
    if (with_energy) k2c_pairs_kernel<true><<<grid, CW * 32, 0, s->stream>>>(A);
    else k2c_pairs_kernel<false><<<grid, CW * 32, 0, s->stream>>>(A);
    s->launches += 1;
  }
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

}  // namespace pasta
