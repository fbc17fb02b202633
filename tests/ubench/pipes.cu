// Issue/pipe microbenchmark behind the K2 roofline denominators (profiles/r1_pipe_microbench.md).
// One block per SM, W warps per SM sub-partition (SMSP), unrolled loops of independent dependency chains, timed
// with clock64 inside the kernel.  Prints one line per experiment: "<name> W=<w> <SMSP-cycles per warp instruction>".
// Built and run by tests/test_pipe_peaks.py (nvcc -gencode arch=compute_100a,code=sm_100a).
#include <cstdio>
#include <cuda_runtime.h>
#define ITERS 8192
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float2 dup(float a) { return make_float2(a, a); }
__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }

// MODE 0: scalar FFMA (one varying operand); 1: MUFU.EX2; 2: FFMA2 p += q*q' (three distinct register pairs);
// 3: FFMA2 p += q*q (two); 4: FADD2 p += scalar broadcast; 5: FMUL2 p *= m
template <int MODE>
__global__ void __launch_bounds__(1024) k_ops(float* out, long long* cyc, float seed) {
  float2 p[8], q[8];
  float a[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { p[i] = make_float2(seed + i, seed - i); q[i] = make_float2(seed * i, seed + 2 * i + threadIdx.x); a[i] = seed + i; }
  const float2 m = make_float2(seed * 0.5f, seed * 0.25f);
  const float ms = seed * 0.999f;
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < ITERS; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (MODE == 0) a[i] = fmaf(a[i], ms, seed);
        if (MODE == 1) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(a[i]));
        if (MODE == 2) p[i] = __ffma2_rn(q[i], q[(i + 1) & 7], p[i]);
        if (MODE == 3) p[i] = __ffma2_rn(q[i], q[i], p[i]);
        if (MODE == 4) p[i] = __fadd2_rn(make_float2(a[i], a[i]), p[i]);
        if (MODE == 5) p[i] = __fmul2_rn(p[i], m);
      }
    }
  }
  const long long t1 = clock64();
  float s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += a[i] + p[i].x + p[i].y + q[i].x;
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
  if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// The evaluation step of k2_chunk.cu (one source against a packed pair of targets: 13 packed instructions + 2
// MUFU.EX2) from registers, 4 steps per trip.
struct Acc { float2 fx, fy, fz, e; };
__device__ __forceinline__ void evaluate(float sx, float sy, float sz, float2 ntx, float2 nty, float2 ntz, Acc& acc,
                                         float g2a, float gB, float a, float B) {
  const float2 dx = __fadd2_rn(dup(sx), ntx), dy = __fadd2_rn(dup(sy), nty), dz = __fadd2_rn(dup(sz), ntz);
  float2 nr2 = __fmul2_rn(neg2(dx), dx);
  nr2 = __ffma2_rn(neg2(dy), dy, nr2);
  nr2 = __ffma2_rn(neg2(dz), dz, nr2);
  const float2 u = make_float2(ex2_approx(nr2.x), ex2_approx(nr2.y));
  const float2 g = __fmul2_rn(u, __ffma2_rn(dup(g2a), u, dup(gB)));
  acc.e = __ffma2_rn(u, __ffma2_rn(dup(a), u, dup(B)), acc.e);
  acc.fx = __ffma2_rn(g, dx, acc.fx);
  acc.fy = __ffma2_rn(g, dy, acc.fy);
  acc.fz = __ffma2_rn(g, dz, acc.fz);
}
__global__ void __launch_bounds__(1024) k_step(float* out, long long* cyc, float seed) {
  Acc acc; acc.fx = acc.fy = acc.fz = acc.e = make_float2(0.f, 0.f);
  const float2 ntx = make_float2(seed + threadIdx.x, seed * 2), nty = make_float2(seed * 3, seed * 4), ntz = make_float2(seed * 5, seed * 6);
  float s[12];
#pragma unroll
  for (int i = 0; i < 12; ++i) s[i] = seed * (i + 1) + 0.001f * threadIdx.x;
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < ITERS; ++it) {
#pragma unroll
    for (int j = 0; j < 4; ++j) evaluate(s[3 * j], s[3 * j + 1], s[3 * j + 2], ntx, nty, ntz, acc, seed, seed * .5f, seed * .25f, seed * .125f);
#pragma unroll
    for (int i = 0; i < 12; ++i) s[i] = __int_as_float(__float_as_int(s[i]) ^ (it & 64));  // loop-variant sources (ALU pipe)
  }
  const long long t1 = clock64();
  out[blockIdx.x * blockDim.x + threadIdx.x] = acc.fx.x + acc.fx.y + acc.fy.x + acc.fy.y + acc.fz.x + acc.fz.y + acc.e.x + acc.e.y;
  if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

// Do other pipes' instructions issue in the shadow of packed FP32?  16 independent 2-operand FFMA2 per trip (32 pipe
// cycles) interleaved with M integer ALU instructions (LOP3, 8 independent chains) or M shared-memory loads: if a packed
// instruction kept only the FMA pipe for its second cycle the trip would cost max(32, 16 + M) cycles; if it keeps the
// DISPATCH port it costs 32 + M.
template <int M, bool LOADS>
__global__ void __launch_bounds__(1024) k_mix(float* out, long long* cyc, float seed) {
  __shared__ int sm[1024];
  float2 p[8], q[8];
  unsigned x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { p[i] = make_float2(seed + i, seed - i); q[i] = make_float2(seed * i, seed + 2 * i + threadIdx.x); x[i] = threadIdx.x * 2654435761u + i; }
  sm[threadIdx.x] = threadIdx.x;
  __syncthreads();
  const unsigned key = (unsigned)__float_as_int(seed) | 1u;
  const unsigned a0 = (unsigned)__cvta_generic_to_shared(&sm[threadIdx.x & ~31]);
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < ITERS; ++it) {
#pragma unroll
    for (int r = 0; r < 2; ++r) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        p[i] = __ffma2_rn(q[i], q[i], p[i]);
#pragma unroll
        for (int m = 0; m < (M >= 16 ? M / 16 : ((i + 8 * r) % (16 / (M > 0 ? M : 16)) == 0 && M > 0 ? 1 : 0)); ++m) {
          if (LOADS) { int v; asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(a0 + 4 * ((i + m + r) & 31)) : "memory"); x[i] ^= (unsigned)v; }
          else if ((m + r) & 1) asm volatile("add.u32 %0, %0, %1;" : "+r"(x[i]) : "r"(key));   // (xor / add alternate: nothing to fold)
          else asm volatile("xor.b32 %0, %0, %1;" : "+r"(x[i]) : "r"(key));
        }
      }
    }
  }
  const long long t1 = clock64();
  float s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += p[i].x + p[i].y + q[i].x + (float)x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
  if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}

static float* g_out; static long long* g_cyc; static int g_sms;
template <class F> static void run(const char* name, int w, double per_trip, F launch) {
  launch(w); launch(w);
  cudaDeviceSynchronize();
  static long long h[1024];
  cudaMemcpy(h, g_cyc, g_sms * sizeof(long long), cudaMemcpyDeviceToHost);
  double avg = 0; for (int i = 0; i < g_sms; ++i) avg += h[i]; avg /= g_sms;
  printf("%s W=%d %.4f\n", name, w, avg / ((double)ITERS * per_trip * w));
}
int main() {
  cudaDeviceProp prop; if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { printf("no device\n"); return 1; }
  g_sms = prop.multiProcessorCount;
  cudaMalloc(&g_out, (size_t)g_sms * 1024 * 4); cudaMalloc(&g_cyc, g_sms * 8);
  printf("sms %d\n", g_sms);
  for (int w : {2, 4, 8}) {
    run("ffma", w, 32, [](int w_) { k_ops<0><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mufu_ex2", w, 32, [](int w_) { k_ops<1><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("ffma2_3op", w, 32, [](int w_) { k_ops<2><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("ffma2_2op", w, 32, [](int w_) { k_ops<3><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("fadd2_bcast", w, 32, [](int w_) { k_ops<4><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("fmul2", w, 32, [](int w_) { k_ops<5><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("eval_step", w, 4, [](int w_) { k_step<<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    // SMSP-cycles per TRIP of 16 packed FFMA2 + M other instructions
    run("mix16_alu0", w, 1, [](int w_) { k_mix<0, false><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mix16_alu4", w, 1, [](int w_) { k_mix<4, false><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mix16_alu8", w, 1, [](int w_) { k_mix<8, false><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mix16_lds4", w, 1, [](int w_) { k_mix<4, true><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mix16_lds8", w, 1, [](int w_) { k_mix<8, true><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mix16_alu16", w, 1, [](int w_) { k_mix<16, false><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mix16_alu32", w, 1, [](int w_) { k_mix<32, false><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mix16_alu64", w, 1, [](int w_) { k_mix<64, false><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
    run("mix16_lds16", w, 1, [](int w_) { k_mix<16, true><<<g_sms, 128 * w_>>>(g_out, g_cyc, 1.0001f); });
  }
  return 0;
}
