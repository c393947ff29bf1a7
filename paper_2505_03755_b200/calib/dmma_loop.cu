// Calibration microbenchmark (not on the product path): the bare consumer loop of the DMMA kernels --
// fragment loads from shared memory + mma.sync.m8n8k4.f64 for a warp tile of TM x TN MMA tiles, 8
// consumer warps with setmaxnreg 232, no pipeline -- to tell what the instruction mix alone allows.
#include <cstdio>
#include <cuda_runtime.h>
#include <stdint.h>
__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
template <int TM, int TN, int VEC>
__global__ void __launch_bounds__(384, 1) k(double* out, int iters, int ld) {
  extern __shared__ __align__(16) double sm[];
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31, r = l >> 2, j = l & 3;
  for (int i = tid; i < 20 * 1024; i += blockDim.x) sm[i] = 1e-3 * (i % 97);
  __syncthreads();
  if (w >= 8) { asm volatile("setmaxnreg.dec.sync.aligned.u32 40;"); return; }
  asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
  double acc[TM][TN][2];
#pragma unroll
  for (int t = 0; t < TM; t++)
#pragma unroll
    for (int u = 0; u < TN; u++) acc[t][u][0] = acc[t][u][1] = 0.0;
  for (int it = 0; it < iters; it++) {
    const double* ap = sm + ((it & 1) * 128 + (w & 3) * 8 * TM % 96 + r) * ld;
    const double* bp = sm + 10240 + ((it & 1) * 128 + r) * ld;
    if (VEC == 1) {
#pragma unroll
      for (int kk = 0; kk < 4; kk++) {
        double a[TM], b[TN];
#pragma unroll
        for (int t = 0; t < TM; t++) a[t] = ap[(t * 8 % 32) * ld + j + 4 * kk];
#pragma unroll
        for (int u = 0; u < TN; u++) b[u] = bp[(u * 8 % 96) * ld + j + 4 * kk];
#pragma unroll
        for (int u = 0; u < TN; u++)
#pragma unroll
          for (int t = 0; t < TM; t++) dmma(acc[t][u][0], acc[t][u][1], a[t], b[u]);
      }
    } else {
#pragma unroll
      for (int kk = 0; kk < 4; kk += 2) {
        double2 a[TM], b[TN];
#pragma unroll
        for (int t = 0; t < TM; t++) a[t] = *reinterpret_cast<const double2*>(ap + (t * 8 % 32) * ld + 2 * j + 4 * kk);
#pragma unroll
        for (int u = 0; u < TN; u++) b[u] = *reinterpret_cast<const double2*>(bp + (u * 8 % 96) * ld + 2 * j + 4 * kk);
#pragma unroll
        for (int u = 0; u < TN; u++)
#pragma unroll
          for (int t = 0; t < TM; t++) dmma(acc[t][u][0], acc[t][u][1], a[t].x, b[u].x);
#pragma unroll
        for (int u = 0; u < TN; u++)
#pragma unroll
          for (int t = 0; t < TM; t++) dmma(acc[t][u][0], acc[t][u][1], a[t].y, b[u].y);
      }
    }
  }
  double s = 0;
#pragma unroll
  for (int t = 0; t < TM; t++)
#pragma unroll
    for (int u = 0; u < TN; u++) s += acc[t][u][0] + acc[t][u][1];
  if (s == 12345.678) out[0] = s;
}
template <int TM, int TN, int VEC>
void run(int ld) {
  double* out; cudaMalloc(&out, 8);
  const int iters = 20000, smem = 20 * 1024 * 8;
  cudaFuncSetAttribute(k<TM, TN, VEC>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  k<TM, TN, VEC><<<148, 384, smem>>>(out, 200, ld);
  cudaEventRecord(e0);
  k<TM, TN, VEC><<<148, 384, smem>>>(out, iters, ld);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  double flops = 148.0 * 8 * iters * 4.0 * TM * TN * 512;
  printf("warp tile %dx%d MMA tiles, %s ld=%d: LDS/DMMA = %.2f  %8.3f ms %6.2f TFLOP/s (%s)\n", TM, TN, VEC == 1 ? "LDS.64 " : "LDS.128", ld,
         (TM + TN) / (double)(TM * TN) / VEC, ms, flops / ms * 1e-9, cudaGetErrorString(cudaGetLastError()));
  cudaFree(out);
}
int main() {
  run<2, 19, 1>(20); run<2, 19, 2>(24);
  run<4, 10, 1>(20); run<4, 10, 2>(24);
  run<4, 9, 1>(20);  run<4, 9, 2>(24);
  run<5, 5, 1>(36);  run<5, 5, 2>(40);
  run<5, 3, 1>(36);  run<5, 2, 1>(36);
  run<6, 6, 1>(36);  run<6, 6, 2>(40);
  run<2, 8, 1>(20);  run<2, 4, 1>(20);
  return 0;
}
