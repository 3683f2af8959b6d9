// Instruction-throughput microbenchmark behind the FP32 roofline denominator of bench.py / DESIGN.md 5:
// warp instructions per clock per SM for the instruction classes of the particle-interaction kernels
// (FFMA, FFMA2 = fma.rn.f32x2, HFMA2, FMNMX, MUFU, HMMA m16n8k8).  Stand-alone program (not part of the library):
//   python -m paper_2104_00537_b200.fp32_peak      compiles and runs it, prints the table.
// One CTA of 1024 threads per SM; every thread runs NCHAIN independent dependency chains for NITER iterations;
// the rate is (warps x instructions) / (clock64 cycles of the CTA), median over the CTAs.
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <algorithm>
#include <cstdio>
#include <vector>

constexpr int NCHAIN = 8, NITER = 4096, NT = 1024;

typedef unsigned long long f2;
__device__ __forceinline__ f2 pack(float a, float b) { f2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }

enum { K_FFMA_REUSE, K_FFMA_3OP, K_FFMA2, K_HFMA2, K_FMNMX, K_MUFU_RCP, K_MUFU_SQRT, K_HMMA, K_FFMA_MUFU, K_COUNT };
static const char* k_names[K_COUNT] = {"FFMA  d = a*d + a (2 register operands)", "FFMA  d = a*b + d (3 distinct registers)",
                                       "FFMA2 fma.rn.f32x2", "HFMA2", "FMNMX", "MUFU.RSQ", "MUFU.SQRT",
                                       "HMMA m16n8k8 f16", "FFMA + MUFU.RSQ 8:1 interleaved (FFMA rate)"};

template <int KIND>
__global__ void __launch_bounds__(NT, 1) k_rate(float* out, long long* cycles, float seed) {
  float x[NCHAIN], b = seed * 1.0001f, a = seed * 0.9999f;
  f2 p[NCHAIN];
  __half2 h[NCHAIN];
  unsigned m0[NCHAIN], m1[NCHAIN];
#pragma unroll
  for (int i = 0; i < NCHAIN; i++) {
    x[i] = seed + (float)(threadIdx.x + i) * 1e-6f;
    p[i] = pack(x[i], x[i] + 1e-6f);
    h[i] = __floats2half2_rn(x[i], x[i]);
    m0[i] = m1[i] = 0u;
  }
  const f2 pa = pack(a, a), pb = pack(b * 1e-3f, b * 1e-3f);
  const __half2 ha = __floats2half2_rn(a, a), hb = __floats2half2_rn(1e-3f, 1e-3f);
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 16
  for (int it = 0; it < NITER; it++) {
#pragma unroll
    for (int i = 0; i < NCHAIN; i++) {
      if (KIND == K_FFMA_REUSE) asm volatile("fma.rn.f32 %0, %1, %0, %1;" : "+f"(x[i]) : "f"(a));
      if (KIND == K_FFMA_3OP) asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(x[i]) : "f"(a), "f"(b));
      if (KIND == K_FFMA2) asm volatile("fma.rn.f32x2 %0, %1, %0, %2;" : "+l"(p[i]) : "l"(pa), "l"(pb));
      if (KIND == K_HFMA2) asm volatile("fma.rn.f16x2 %0, %1, %0, %2;" : "+r"(*reinterpret_cast<unsigned*>(&h[i])) : "r"(*reinterpret_cast<const unsigned*>(&ha)), "r"(*reinterpret_cast<const unsigned*>(&hb)));
      if (KIND == K_FMNMX) asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
      if (KIND == K_MUFU_RCP) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
      if (KIND == K_MUFU_SQRT) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
      if (KIND == K_HMMA)
        asm volatile("mma.sync.aligned.m16n8k8.row.col.f16.f16.f16.f16 {%0, %1}, {%2, %3}, {%4}, {%0, %1};"
                     : "+r"(m0[i]), "+r"(m1[i]) : "r"(0x3c003c00u), "r"(0x3c003c00u), "r"(0x00000000u));
      if (KIND == K_FFMA_MUFU) {
        asm volatile("fma.rn.f32 %0, %1, %0, %1;" : "+f"(x[i]) : "f"(a));
        if (i == 0) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(b));
      }
    }
  }
  const long long t1 = clock64();
  float s = b;
#pragma unroll
  for (int i = 0; i < NCHAIN; i++) s += x[i] + __low2float(h[i]) + (float)(p[i] & 0xff) + (float)((m0[i] ^ m1[i]) & 0xff);
  if (s == 123.456f) out[0] = s;
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template <int KIND>
static double run(int n_sm, float* d_out, long long* d_cyc) {
  k_rate<KIND><<<n_sm, NT>>>(d_out, d_cyc, 1.0f);   // warm-up
  k_rate<KIND><<<n_sm, NT>>>(d_out, d_cyc, 1.0f);
  std::vector<long long> c(n_sm);
  cudaMemcpy(c.data(), d_cyc, sizeof(long long) * n_sm, cudaMemcpyDeviceToHost);
  std::sort(c.begin(), c.end());
  return (double)(NT / 32) * NCHAIN * NITER / (double)c[n_sm / 2];
}

int main() {
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { fprintf(stderr, "no CUDA device\n"); return 1; }
  const int n_sm = prop.multiProcessorCount;
  float* d_out; long long* d_cyc;
  cudaMalloc(&d_out, 4); cudaMalloc(&d_cyc, sizeof(long long) * n_sm);
  double r[K_COUNT];
  r[K_FFMA_REUSE] = run<K_FFMA_REUSE>(n_sm, d_out, d_cyc);
  r[K_FFMA_3OP] = run<K_FFMA_3OP>(n_sm, d_out, d_cyc);
  r[K_FFMA2] = run<K_FFMA2>(n_sm, d_out, d_cyc);
  r[K_HFMA2] = run<K_HFMA2>(n_sm, d_out, d_cyc);
  r[K_FMNMX] = run<K_FMNMX>(n_sm, d_out, d_cyc);
  r[K_MUFU_RCP] = run<K_MUFU_RCP>(n_sm, d_out, d_cyc);
  r[K_MUFU_SQRT] = run<K_MUFU_SQRT>(n_sm, d_out, d_cyc);
  r[K_HMMA] = run<K_HMMA>(n_sm, d_out, d_cyc);
  r[K_FFMA_MUFU] = run<K_FFMA_MUFU>(n_sm, d_out, d_cyc);
  if (cudaDeviceSynchronize() != cudaSuccess) { fprintf(stderr, "CUDA error: %s\n", cudaGetErrorString(cudaGetLastError())); return 1; }
  int clk_khz = 0;
  cudaDeviceGetAttribute(&clk_khz, cudaDevAttrClockRate, 0);
  printf("device: %s, %d SMs, max SM clock %d MHz\n", prop.name, n_sm, clk_khz / 1000);
  printf("| instruction | warp instructions / clk / SM | thread results / clk / SM |\n|---|---|---|\n");
  for (int k = 0; k < K_COUNT; k++) {
    const double per = (k == K_FFMA2 || k == K_HFMA2) ? 64.0 : 32.0;
    printf("| %s | %.3f | %.1f |\n", k_names[k], r[k], r[k] * per);
  }
  const double ffma = r[K_FFMA_REUSE];
  printf("FP32 peak from the FFMA rate: %d SM x %.3f x 32 lanes x 2 flop x %.3f GHz = %.2f TFLOP/s (nominal 4/clk/SM: %.2f)\n", n_sm, ffma,
         clk_khz * 1e-6, n_sm * ffma * 64.0 * clk_khz * 1e-6 * 1e-3, n_sm * 4.0 * 64.0 * clk_khz * 1e-6 * 1e-3);
  return 0;
}
