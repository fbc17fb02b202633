// K2 -- pair force and energy (Eq. 1a-c; cut-off and nearest image,
// PAPER.md:98, readings D1-D3).
//
// FP32 pair arithmetic in pre-scaled coordinates x' = sigma x with sigma^2 = log2(e)/(2 Lambda), so that
//   u = exp(-r^2 / 2 Lambda) = exp2(-r'^2)                      one MUFU.EX2, no multiply
//   V = u (a u + B)                                               B = b+c (like) / b-c (unlike)
//   g' = -(1/r) dV/dr / sigma = u (g2a u + gB)                    F_i = sum g' d'   (d' = sigma d)
//   pp: 1/r' = rsqrt(r'^2); ex = exp2(-kappa r'); t = ex / r'
//       V += alpha_s t;  g' += alpha_s2 t (1/r' + inv_lam_s) / r'
// Positions are cell-relative (|x'| < sigma w) plus an exact integer cell offset times w', which keeps
// the FP32 ulp of a coordinate below 1e-6 fm even in a 690 fm box (hard part 1).
// Partial sums run in FP32 over short runs and are flushed into FP64 accumulators.
#include "pasta_internal.cuh"

namespace pasta {

PairConsts make_pair_consts(const pasta_params& p) {
  const double log2e = 1.4426950408889634074;
  const double sigma = sqrt(log2e / (2.0 * p.Lambda));
  PairConsts c;
  c.sigma = (float)sigma;
  c.inv_sigma = (float)(1.0 / sigma);
  c.rc2s = (float)(sigma * sigma * p.r_c * p.r_c);
  {
    const double rn = p.r_nuc > 0.0 ? p.r_nuc : p.r_c;
    c.rn2s = (float)(sigma * sigma * rn * rn);
  }
  c.a = (float)p.a;
  c.g2a = (float)(2.0 * p.a / (p.Lambda * sigma));
  c.B_like = (float)(p.b + p.c);
  c.B_unlike = (float)(p.b - p.c);
  c.gB_like = (float)((p.b + p.c) / (p.Lambda * sigma));
  c.gB_unlike = (float)((p.b - p.c) / (p.Lambda * sigma));
  c.kappa = (float)(log2e / (sigma * p.lambda));
  c.alpha_s = (float)(p.alpha_hbarc * sigma);
  c.alpha_s2 = (float)(p.alpha_hbarc * sigma * sigma);
  c.inv_lam_s = (float)(1.0 / (p.lambda * sigma));
  c.v_self = (float)(p.a + p.b + p.c);
  return c;
}

__device__ __forceinline__ float fast_ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float fast_rsqrt(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// One pair in scaled units.  COUL: both protons.  Accumulates into (fx, fy, fz, e); e gets V (not V/2).
template <bool COUL, bool ENERGY>
__device__ __forceinline__ void pair_accumulate(float dx, float dy, float dz, float r2, float B, float gB,
                                                const PairConsts& c, float& fx, float& fy, float& fz, float& e) {
  const float u = r2 < c.rn2s ? fast_ex2(-r2) : 0.f;  // nuclear terms: strict r < r_n
  float g = u * fmaf(c.g2a, u, gB);
  float V = 0.f;
  if (ENERGY) V = u * fmaf(c.a, u, B);
  if (COUL) {
    if (r2 > 0.f) {  // D2: the divergent Coulomb term of coincident protons is skipped
      const float rinv = fast_rsqrt(r2);
      const float r = r2 * rinv;
      const float t = fast_ex2(-c.kappa * r) * rinv;
      if (ENERGY) V = fmaf(c.alpha_s, t, V);
      g = fmaf(c.alpha_s2 * t, (rinv + c.inv_lam_s) * rinv, g);
    }
  }
  fx = fmaf(g, dx, fx);
  fy = fmaf(g, dy, fy);
  fz = fmaf(g, dz, fz);
  if (ENERGY) e += V;
}

// ---------------------------------------------------------------------------------------------------
// Variant 1 ("v0", reference GPU kernel): one thread per target in sorted order, walks the (2k+1)^3
// cell stencil of its own cell for both species segments, reading sources through L1.  Falls back to
// "all sources, per-pair nearest image" when the grid has fewer than 2k+1 cells per side (small boxes,
// e.g. config 1), where a stencil would visit a cell twice.  Simple and slow; kept as the in-library
// cross-check of the tiled kernel and as the pair counter.
// ---------------------------------------------------------------------------------------------------
struct V0Args {
  int64_t N;
  int32_t Np;
  int32_t ncell, nc3, k;
  float wS;      // sigma * cell width
  float LS;      // sigma * L
  float inv_LS;  // 1 / (sigma L)
  const float4* pos4;
  const int32_t* cxyz;
  const int32_t* bin_start;
  const int32_t* perm;
  double* F;
  double* e;
  unsigned long long* pair_counter;
};

template <bool ENERGY, bool COUNT_ONLY>
__global__ void __launch_bounds__(128) k2_v0_kernel(V0Args A, PairConsts c) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= A.N) return;
  const float4 pi = A.pos4[t];
  const int ci = A.cxyz[t];
  const int cix = PASTA_CX(ci), ciy = PASTA_CY(ci), ciz = PASTA_CZ(ci);
  const bool ip = t < A.Np;
  double Fx = 0.0, Fy = 0.0, Fz = 0.0, E = 0.0;
  unsigned long long count = 0, count_nz = 0;  // in range; in range with a term that is not exactly 0 in FP32
  const bool stencil = A.ncell >= 2 * A.k + 1;

  for (int sj = 0; sj < 2; ++sj) {  // source species: 0 = protons, 1 = neutrons
    const bool like = (ip == (sj == 0));
    const float B = like ? c.B_like : c.B_unlike;
    const float gB = like ? c.gB_like : c.gB_unlike;
    const bool coul = ip && sj == 0;
    if (stencil) {
      for (int dz = -A.k; dz <= A.k; ++dz)
        for (int dy = -A.k; dy <= A.k; ++dy)
          for (int dx = -A.k; dx <= A.k; ++dx) {
            int jx = cix + dx, jy = ciy + dy, jz = ciz + dz;
            jx += jx < 0 ? A.ncell : (jx >= A.ncell ? -A.ncell : 0);
            jy += jy < 0 ? A.ncell : (jy >= A.ncell ? -A.ncell : 0);
            jz += jz < 0 ? A.ncell : (jz >= A.ncell ? -A.ncell : 0);
            const int bin = sj * A.nc3 + (jz * A.ncell + jy) * A.ncell + jx;
            const int lo = A.bin_start[bin], hi = A.bin_start[bin + 1];
            // target position expressed in the source cell's frame
            const float xi = pi.x - (float)dx * A.wS, yi = pi.y - (float)dy * A.wS, zi = pi.z - (float)dz * A.wS;
            float fx = 0.f, fy = 0.f, fz = 0.f, e = 0.f;
            for (int j = lo; j < hi; ++j) {
              if (j == t) continue;
              const float4 pj = A.pos4[j];
              const float ddx = xi - pj.x, ddy = yi - pj.y, ddz = zi - pj.z;
              const float r2 = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx));
              if (r2 < c.rc2s) {
                if (COUNT_ONLY) {
                  ++count;
                  count_nz += (coul || (r2 < 126.0f && r2 < c.rn2s)) ? 1 : 0;
                } else if (coul) {
                  pair_accumulate<true, ENERGY>(ddx, ddy, ddz, r2, B, gB, c, fx, fy, fz, e);
                } else {
                  pair_accumulate<false, ENERGY>(ddx, ddy, ddz, r2, B, gB, c, fx, fy, fz, e);
                }
              }
            }
            Fx += fx; Fy += fy; Fz += fz; E += e;
          }
    } else {
      const int lo = sj == 0 ? 0 : A.Np, hi = sj == 0 ? A.Np : (int)A.N;
      float fx = 0.f, fy = 0.f, fz = 0.f, e = 0.f;
      for (int j = lo; j < hi; ++j) {
        if (j != t) {
          const float4 pj = A.pos4[j];
          const int cj = A.cxyz[j];
          float ddx = fmaf((float)(cix - PASTA_CX(cj)), A.wS, pi.x - pj.x);
          float ddy = fmaf((float)(ciy - PASTA_CY(cj)), A.wS, pi.y - pj.y);
          float ddz = fmaf((float)(ciz - PASTA_CZ(cj)), A.wS, pi.z - pj.z);
          ddx -= A.LS * rintf(ddx * A.inv_LS);  // nearest periodic image
          ddy -= A.LS * rintf(ddy * A.inv_LS);
          ddz -= A.LS * rintf(ddz * A.inv_LS);
          const float r2 = fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx));
          if (r2 < c.rc2s) {
            if (COUNT_ONLY) {
              ++count;
              count_nz += (coul || (r2 < 126.0f && r2 < c.rn2s)) ? 1 : 0;
            } else if (coul) {
              pair_accumulate<true, ENERGY>(ddx, ddy, ddz, r2, B, gB, c, fx, fy, fz, e);
            } else {
              pair_accumulate<false, ENERGY>(ddx, ddy, ddz, r2, B, gB, c, fx, fy, fz, e);
            }
          }
        }
        if (((j - lo) & 63) == 63 || j == hi - 1) {
          Fx += fx; Fy += fy; Fz += fz; E += e;
          fx = fy = fz = e = 0.f;
        }
      }
    }
  }
  if (COUNT_ONLY) {
    if (count) atomicAdd(A.pair_counter, count);
    if (count_nz) atomicAdd(A.pair_counter + 1, count_nz);
  } else {
    const int i = A.perm[t];
    A.F[3 * (int64_t)i + 0] = Fx;
    A.F[3 * (int64_t)i + 1] = Fy;
    A.F[3 * (int64_t)i + 2] = Fz;
    if (ENERGY) A.e[i] = 0.5 * E;
  }
}

static V0Args make_v0_args(Sim* s) {
  const PairConsts c = make_pair_consts(s->prm);
  const double sigma = sqrt(1.4426950408889634074 / (2.0 * s->prm.Lambda));
  V0Args A;
  A.N = s->N;
  A.Np = (int32_t)s->Np;
  A.ncell = s->grid_sp[0].ncell;  // both species share one grid for this kernel (k1_build uniform)
  A.nc3 = (int32_t)s->grid_sp[0].nc3;
  A.k = s->prm.cell_subdiv;
  A.wS = (float)(sigma * s->grid_sp[0].w);
  A.LS = (float)(sigma * s->L);
  A.inv_LS = (float)(1.0 / (sigma * s->L));
  A.pos4 = s->pos4.as<float4>();
  A.cxyz = s->cxyz.as<int32_t>();
  A.bin_start = s->bin_start.as<int32_t>();
  A.perm = s->perm.as<int32_t>();
  A.F = s->F.as<double>();
  A.e = s->e.as<double>();
  A.pair_counter = s->counters.as<unsigned long long>();
  (void)c;
  return A;
}

int k2_forces(Sim* s, bool with_energy, double kick) {
  // force_variant: 0 = library default (chunk kernel), 1 = thread-per-target reference, 2 = chunk kernel
  if (s->tune.force_variant == 1) {
    if (kick != 0.0) {
      set_error("the thread-per-target kernel has no fused kick");
      return PASTA_ESTATE;
    }
    return k2_reference_forces(s, with_energy);
  }
  return k2_chunk_forces(s, with_energy, false, kick);
}

int k2_reference_forces(Sim* s, bool with_energy) {
  const PairConsts c = make_pair_consts(s->prm);
  V0Args A = make_v0_args(s);
  const int B = 128;
  if (with_energy)
    k2_v0_kernel<true, false><<<grid_for(s->N, B), B, 0, s->stream>>>(A, c);
  else
    k2_v0_kernel<false, false><<<grid_for(s->N, B), B, 0, s->stream>>>(A, c);
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

int k2_pair_count(Sim* s, int64_t* ordered_pairs_host, int64_t* nonzero_pairs_host) {
  const PairConsts c = make_pair_consts(s->prm);
  V0Args A = make_v0_args(s);
  PASTA_CUDA_OK(cudaMemsetAsync(A.pair_counter, 0, 2 * sizeof(unsigned long long), s->stream));
  const int B = 128;
  k2_v0_kernel<false, true><<<grid_for(s->N, B), B, 0, s->stream>>>(A, c);
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  unsigned long long h[2] = {0, 0};
  PASTA_CUDA_OK(cudaMemcpyAsync(h, A.pair_counter, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
  PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  if (ordered_pairs_host) *ordered_pairs_host = (int64_t)h[0];
  if (nonzero_pairs_host) *nonzero_pairs_host = (int64_t)h[1];
  return PASTA_OK;
}

}  // namespace pasta
