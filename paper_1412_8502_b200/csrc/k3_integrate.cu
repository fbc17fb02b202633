// K3 -- velocity Verlet, isokinetic rescale and uniform box/position scaling in FP64
// (readings D6-D11), plus the seeded initial state (D15)
// and the deterministic FP64 reductions (KE, PE).
#include <string.h>

#include "pasta_internal.cuh"

namespace pasta {

// x <- x - L floor(x/L), mapped into [0, L).
__device__ __forceinline__ double wrap_coord(double x, double L, double invL) {
  double w = x - L * floor(x * invL);
  if (w >= L) w -= L;
  if (w < 0.0) w += L;
  if (w >= L || w < 0.0) w = 0.0;
  return w;
}

// First half kick, drift, scale and wrap (O2 steps 1-2):  v += h F;  x = wrap(s (x + dt v)) -- and, fused with it,
// the first step of the cell list of the new positions (K1 a1): the particle's (species, cell) bin on its
// species' force grid and the histogram of the bins.  One thread per particle.
__global__ void k3_kick_drift_count_kernel(int64_t N, double* __restrict__ x, double* __restrict__ v,
                                           const double* __restrict__ F, const uint8_t* __restrict__ is_p, double h,
                                           double dt, double scale, double L, double invL, const GridPair g,
                                           int32_t* __restrict__ pbin, int32_t* __restrict__ bin_count) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  double xn[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const double vk = v[3 * i + k] + h * F[3 * i + k];
    v[3 * i + k] = vk;
    xn[k] = wrap_coord(scale * (x[3 * i + k] + dt * vk), L, invL);
    x[3 * i + k] = xn[k];
  }
  if (bin_count == nullptr) return;  // list mode: the sorted order is frozen (or about to be rebuilt on another grid)
  const int bin = force_bin(g, is_p[i] ? 0 : 1, xn[0], xn[1], xn[2]);
  pbin[i] = bin;
  atomicAdd(&bin_count[bin], 1);
}

// List mode: the same kick and drift, and fused with it the refresh of the frozen sorted order (k1_refresh_kernel): the
// particle's slot gets its new cell-relative coordinates and the launch reports the largest displacement since the build.
__global__ void __launch_bounds__(128) k3_kick_drift_refresh_kernel(int64_t N, double* __restrict__ x, double* __restrict__ v,
                                                                    const double* __restrict__ F, double h, double dt,
                                                                    double scale, double L, double invL,
                                                                    const int32_t* __restrict__ slot_of, const RefreshArgs R) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  float d2 = 0.f;
  if (i < N) {
    double xn[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const double vk = v[3 * i + k] + h * F[3 * i + k];
      v[3 * i + k] = vk;
      xn[k] = wrap_coord(scale * (x[3 * i + k] + dt * vk), L, invL);
      x[3 * i + k] = xn[k];
    }
    d2 = refresh_slot(R, slot_of[i], i, xn);
  }
  refresh_post(R, d2);
}

constexpr int RED_T = 256;
__device__ __forceinline__ double block_sum(double s) {
  __shared__ double ws[RED_T / 32];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = s;
  __syncthreads();
  double t = 0.0;
  if (threadIdx.x < 32) {
    t = threadIdx.x < RED_T / 32 ? ws[threadIdx.x] : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  }
  __syncthreads();
  return t;  // valid in thread 0
}

// Second half kick (O2 step 4) and per-block kinetic-energy partials: v += h F; partial = sum 1/2 M v^2.
__global__ void __launch_bounds__(RED_T) k3_kick_ke_kernel(int64_t n3, double* __restrict__ v,
                                                           const double* __restrict__ F, double h, double half_m,
                                                           double* __restrict__ partials) {
  double s = 0.0;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n3; k += (int64_t)gridDim.x * blockDim.x) {
    const double vk = v[k] + h * F[k];
    v[k] = vk;
    s += half_m * vk * vk;
  }
  s = block_sum(s);
  if (threadIdx.x == 0) partials[blockIdx.x] = s;
}

// Fixed-order final sum of the partials into scalars[slot]; optionally the rescale factor
// sqrt(1.5 N T / KE) into scalars[2] (1 if KE == 0, D8).
__global__ void __launch_bounds__(RED_T) k3_final_sum_kernel(const double* __restrict__ partials, int n,
                                                             double* __restrict__ scalars, int slot,
                                                             double target_ke, int want_factor) {
  double s = 0.0;
  for (int k = threadIdx.x; k < n; k += RED_T) s += partials[k];
  s = block_sum(s);
  if (threadIdx.x == 0) {
    scalars[slot] = s;
    if (want_factor) scalars[2] = s > 0.0 ? sqrt(target_ke / s) : 1.0;
  }
}

__global__ void k3_scale_v_kernel(int64_t n3, double* __restrict__ v, const double* __restrict__ scalars) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n3) return;
  v[k] *= scalars[2];
}

__global__ void __launch_bounds__(RED_T) k3_partial_sum_kernel(const double* __restrict__ in, int64_t n,
                                                               double* __restrict__ partials, double mul,
                                                               int square) {
  double s = 0.0;
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
    const double a = in[k];
    s += square ? mul * a * a : mul * a;
  }
  s = block_sum(s);
  if (threadIdx.x == 0) partials[blockIdx.x] = s;
}

__global__ void k3_wrap_scale_kernel(int64_t n3, double* __restrict__ x, double scale, double L, double invL) {
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n3) return;
  x[k] = wrap_coord(scale * x[k], L, invL);
}

static int red_blocks(int64_t n) {
  int64_t b = (n + RED_T - 1) / RED_T;
  return (int)(b < 1 ? 1 : (b > 1184 ? 1184 : b));  // 148 SMs x 8 resident blocks
}

// The caller has set s->L to the box the forces will be evaluated in; L_wrap = the box the drifted positions are
// wrapped into (the same, except under the linear box-only expansion, where it is the box before it grew).
int k3_kick_drift_count(Sim* s, double dt, double scale, double L_wrap, bool count) {
  GridPair g;
  memset(&g, 0, sizeof(g));
  if (count) PASTA_TRY(k1_setup(s, false, &g));
  k3_kick_drift_count_kernel<<<grid_for(s->N, 128), 128, 0, s->stream>>>(
      s->N, s->x.as<double>(), s->v.as<double>(), s->F.as<double>(), s->is_p.as<uint8_t>(), dt / (2.0 * s->prm.mass),
      dt, scale, L_wrap, 1.0 / L_wrap, g, s->cell_id.as<int32_t>(), count ? s->bin_count.as<int32_t>() : nullptr);
  s->launches += 1;
  s->hist_valid = count;
  s->hist_uniform = s->tune.force_variant == 1;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

int k3_kick_drift_refresh(Sim* s, double dt, double scale, double L_wrap) {
  RefreshArgs R;
  k1_refresh_args(s, &R);
  k3_kick_drift_refresh_kernel<<<grid_for(s->N, 128), 128, 0, s->stream>>>(
      s->N, s->x.as<double>(), s->v.as<double>(), s->F.as<double>(), dt / (2.0 * s->prm.mass), dt, scale, L_wrap,
      1.0 / L_wrap, s->slot_of.as<int32_t>(), R);
  s->launches += 1;
  s->hist_valid = false;
  s->list.pending = true;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

int k3_kick_ke(Sim* s, double dt, bool rescale) {
  const int64_t n3 = 3 * s->N;
  const int nb = red_blocks(n3);
  double* part = s->partials.as<double>();
  double* sc = s->scalars.as<double>();
  k3_kick_ke_kernel<<<nb, RED_T, 0, s->stream>>>(n3, s->v.as<double>(), s->F.as<double>(), dt / (2.0 * s->prm.mass),
                                                 0.5 * s->prm.mass, part);
  s->launches += 1;
  if (rescale) {
    k3_final_sum_kernel<<<1, RED_T, 0, s->stream>>>(part, nb, sc, 0, 1.5 * (double)s->N * s->T, 1);
    k3_scale_v_kernel<<<grid_for(n3, 256), 256, 0, s->stream>>>(n3, s->v.as<double>(), sc);
    s->launches += 2;
  }
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

int k3_wrap_scale(Sim* s, double scale, double L_new) {
  const int64_t n3 = 3 * s->N;
  s->hist_valid = false;
  k3_wrap_scale_kernel<<<grid_for(n3, 256), 256, 0, s->stream>>>(n3, s->x.as<double>(), scale, L_new, 1.0 / L_new);
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

int k3_sum(Sim* s, const double* in, int64_t n, int slot) {
  const int nb = red_blocks(n);
  k3_partial_sum_kernel<<<nb, RED_T, 0, s->stream>>>(in, n, s->partials.as<double>(), 1.0, 0);
  k3_final_sum_kernel<<<1, RED_T, 0, s->stream>>>(s->partials.as<double>(), nb, s->scalars.as<double>(), slot, 0.0, 0);
  s->launches += 2;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

int k3_kinetic(Sim* s, double* ke_host) {
  const int64_t n3 = 3 * s->N;
  const int nb = red_blocks(n3);
  k3_partial_sum_kernel<<<nb, RED_T, 0, s->stream>>>(s->v.as<double>(), n3, s->partials.as<double>(),
                                                     0.5 * s->prm.mass, 1);
  k3_final_sum_kernel<<<1, RED_T, 0, s->stream>>>(s->partials.as<double>(), nb, s->scalars.as<double>(), 0, 0.0, 0);
  s->launches += 2;
  PASTA_CUDA_OK(cudaGetLastError());
  if (ke_host) {
    PASTA_CUDA_OK(cudaMemcpyAsync(ke_host, s->scalars.as<double>(), sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  }
  return PASTA_OK;
}

// ---- seeded initial state (D15): counter-based, one hash chain per (particle, component) ---------------
__device__ __forceinline__ uint64_t splitmix64(uint64_t z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
__device__ __forceinline__ double u01(uint64_t bits) {  // (0,1): 53 random bits, never exactly 0 or 1
  return ((double)(bits >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

__global__ void k3_init_kernel(int64_t N, int64_t Np, double L, double sigma_v, uint64_t seed, double* __restrict__ x,
                               double* __restrict__ v, uint8_t* __restrict__ is_p) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const uint64_t key = splitmix64(seed ^ 0x70617374615F6232ull);
  is_p[i] = i < Np ? 1 : 0;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const uint64_t ctr = (uint64_t)i * 16 + (uint64_t)a * 4;
    double ux = u01(splitmix64(key + splitmix64(ctr + 2)));
    double xa = ux * L;
    x[3 * i + a] = xa < L ? xa : 0.0;
    // Box-Muller: one normal deviate per component
    const double u1 = u01(splitmix64(key + splitmix64(ctr)));
    const double u2 = u01(splitmix64(key + splitmix64(ctr + 1)));
    v[3 * i + a] = sigma_v * sqrt(-2.0 * log(u1)) * cospi(2.0 * u2);
  }
}

__global__ void k3_count_protons_kernel(int64_t N, const uint8_t* __restrict__ is_p, unsigned long long* __restrict__ out) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned m = __ballot_sync(0xffffffffu, i < N && is_p[i] != 0);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(out, (unsigned long long)__popc(m));
}

int k3_count_protons(Sim* s) {
  unsigned long long* c = s->counters.as<unsigned long long>() + 8;
  PASTA_CUDA_OK(cudaMemsetAsync(c, 0, sizeof(unsigned long long), s->stream));
  k3_count_protons_kernel<<<grid_for(s->N, 256), 256, 0, s->stream>>>(s->N, s->is_p.as<uint8_t>(), c);
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  unsigned long long h = 0;
  PASTA_CUDA_OK(cudaMemcpyAsync(&h, c, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
  PASTA_CUDA_OK(cudaStreamSynchronize(s->stream));
  s->Np = (int64_t)h;
  return PASTA_OK;
}

int k3_init_state(Sim* s, uint64_t seed) {
  k3_init_kernel<<<grid_for(s->N, 256), 256, 0, s->stream>>>(s->N, s->Np, s->L, sqrt(s->T / s->prm.mass), seed,
                                                             s->x.as<double>(), s->v.as<double>(),
                                                             s->is_p.as<uint8_t>());
  s->launches += 1;
  PASTA_CUDA_OK(cudaGetLastError());
  return PASTA_OK;
}

}  // namespace pasta
