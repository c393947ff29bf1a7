// Calibration microbenchmark (not on the product path): the consumer loop of k_half_transform<19>
// (64 x 304 CTA tile) inside its full/empty mbarrier ring, fed by bulk copies only or with the A tile
// gathered by 8-byte cp.async, one CTA of 8+4 warps or two of 4+4 per SM, operands re-read from L2.
#include <cstdio>
#include "../csrc/common.cuh"
#include "../csrc/pipeline.cuh"
using namespace dfjk;
constexpr int WN = 19, NT = 16 * WN;
// KS = k4 steps per chunk (4 -> k-chunk 16, 8 -> k-chunk 32); PROD 0: bulk only (A and B), 1: cp.async8 gather for A
// SKEW: second warpgroup starts half a chunk late. STAGES pipeline depth.
template <int KS, int PROD, int SKEW, int STAGES>
__global__ void __launch_bounds__(384, 1) k(const double* __restrict__ src, double* out, int nchunks) {
  constexpr int LD = 4 * KS + 4;                   // 20 or 36
  constexpr int ATILE = 64 * LD, BTILE = NT * LD;
  constexpr uint32_t ABYTES = ATILE * 8, BBYTES = BTILE * 8;
  extern __shared__ __align__(128) double smem[];
  double* sA = smem; double* sB = smem + STAGES * ATILE;
  __shared__ __align__(8) unsigned long long bars[2 * STAGES + 1];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[STAGES]), skewbar = smem_u32(&bars[2 * STAGES]);
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
  if (tid == 0) {
    for (int s = 0; s < STAGES; s++) { mbar_init(full0 + 8 * s, PROD ? 129 : 1); mbar_init(empty0 + 8 * s, 8); }
    mbar_init(skewbar, 4);
    mbar_fence_init();
  }
  __syncthreads();
  if (w >= 8) {
    reg_dec<40>();
    const int tp = tid - 256;
    const uint32_t sA_u = smem_u32(sA), sB_u = smem_u32(sB);
    for (int c = 0; c < nchunks; c++) {
      const int stage = c % STAGES;
      const uint32_t fullb = full0 + 8 * stage;
      mbar_wait(empty0 + 8 * stage, ((c / STAGES) & 1) ^ 1);
      const double* g = src + (size_t)((c * 7 + blockIdx.x) % 64) * (ATILE + BTILE);
      if (tp == 0) {
        mbar_arrive_expect_tx(fullb, PROD ? BBYTES : ABYTES + BBYTES);
        bulk_g2s(sB_u + stage * BBYTES, g + ATILE, BBYTES, fullb);
        if (!PROD) bulk_g2s(sA_u + stage * ABYTES, g, ABYTES, fullb);
      }
      if (PROD) {
        for (int e = tp; e < 64 * 4 * KS; e += 128) {
          const int m = e / (4 * KS), kx = e % (4 * KS);
          cp_async8(sA_u + stage * ABYTES + (m * LD + kx) * 8, g + m * 1201 % ATILE + kx, true);
        }
        cp_async_mbar_arrive_noinc(fullb);
      }
    }
    return;
  }
  reg_inc<232>();
  const int r = l >> 2, j = l & 3, wm = w & 3, wn = w >> 2;
  double acc[2][WN][2];
#pragma unroll
  for (int t = 0; t < 2; t++)
#pragma unroll
    for (int u = 0; u < WN; u++) acc[t][u][0] = acc[t][u][1] = 0.0;
  if (SKEW && wn == 1) mbar_wait(skewbar, 0);
  for (int c = 0; c < nchunks; c++) {
    const int stage = c % STAGES;
    mbar_wait(full0 + 8 * stage, (c / STAGES) & 1);
    const double* a_ptr = sA + stage * ATILE + (wm * 16 + r) * LD + j;
    const double* b_ptr = sB + stage * BTILE + (wn * 8 * WN + r) * LD + j;
#pragma unroll
    for (int kk = 0; kk < KS; kk++) {
      const double a0 = a_ptr[4 * kk], a1 = a_ptr[8 * LD + 4 * kk];
      double b[WN];
#pragma unroll
      for (int u = 0; u < WN; u++) b[u] = b_ptr[u * 8 * LD + 4 * kk];
#pragma unroll
      for (int u = 0; u < WN; u++) { dmma884(acc[0][u][0], acc[0][u][1], a0, b[u]); dmma884(acc[1][u][0], acc[1][u][1], a1, b[u]); }
      if (SKEW && c == 0 && wn == 0 && kk == KS / 2 - 1) { __syncwarp(); if (l == 0) mbar_arrive(skewbar); }
    }
    __syncwarp();
    if (l == 0) mbar_arrive(empty0 + 8 * stage);
  }
  double s = 0;
#pragma unroll
  for (int t = 0; t < 2; t++)
#pragma unroll
    for (int u = 0; u < WN; u++) s += acc[t][u][0] + acc[t][u][1];
  if (s == 12345.678) out[0] = s;
}
template <int KS, int PROD, int SKEW, int STAGES>
void run(const double* src, double* out) {
  constexpr int LD = 4 * KS + 4;
  const size_t smem = (size_t)STAGES * (64 + NT) * LD * 8;
  const int nchunks = 60000 * 4 / KS;
  cudaFuncSetAttribute(k<KS, PROD, SKEW, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  k<KS, PROD, SKEW, STAGES><<<148, 384, smem>>>(src, out, 100);
  cudaEventRecord(e0);
  k<KS, PROD, SKEW, STAGES><<<148, 384, smem>>>(src, out, nchunks);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  const double flops = 148.0 * 8 * (double)nchunks * KS * 2 * WN * 512;
  printf("k-chunk %2d, %s, skew %d, %d stages (%zu KB smem): %8.3f ms %6.2f TFLOP/s (%s)\n", 4 * KS,
         PROD ? "cp.async8 A + bulk B" : "bulk A + bulk B     ", SKEW, STAGES, smem >> 10, ms, flops / ms * 1e-9,
         cudaGetErrorString(cudaGetLastError()));
}

// Two independent 256-thread CTAs per SM: 4 consumer warps (64 x 152 tile) + 4 producer warps each.
template <int KS, int PROD, int STAGES>
__global__ void __launch_bounds__(256, 2) k2(const double* __restrict__ src, double* out, int nchunks) {
  constexpr int NTH = 8 * WN;
  constexpr int LD = 4 * KS + 4;
  constexpr int ATILE = 64 * LD, BTILE = NTH * LD;
  constexpr uint32_t ABYTES = ATILE * 8, BBYTES = BTILE * 8;
  extern __shared__ __align__(128) double smem[];
  double* sA = smem; double* sB = smem + STAGES * ATILE;
  __shared__ __align__(8) unsigned long long bars[2 * STAGES];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[STAGES]);
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
  if (tid == 0) {
    for (int s = 0; s < STAGES; s++) { mbar_init(full0 + 8 * s, PROD ? 129 : 1); mbar_init(empty0 + 8 * s, 4); }
    mbar_fence_init();
  }
  __syncthreads();
  if (w >= 4) {
    reg_dec<32>();
    const int tp = tid - 128;
    const uint32_t sA_u = smem_u32(sA), sB_u = smem_u32(sB);
    for (int c = 0; c < nchunks; c++) {
      const int stage = c % STAGES;
      const uint32_t fullb = full0 + 8 * stage;
      mbar_wait(empty0 + 8 * stage, ((c / STAGES) & 1) ^ 1);
      const double* g = src + (size_t)((c * 7 + blockIdx.x) % 64) * (ATILE + 2 * BTILE);
      if (tp == 0) {
        mbar_arrive_expect_tx(fullb, PROD ? BBYTES : ABYTES + BBYTES);
        bulk_g2s(sB_u + stage * BBYTES, g + ATILE, BBYTES, fullb);
        if (!PROD) bulk_g2s(sA_u + stage * ABYTES, g, ABYTES, fullb);
      }
      if (PROD) {
        for (int e = tp; e < 64 * 4 * KS; e += 128) {
          const int m = e / (4 * KS), kx = e % (4 * KS);
          cp_async8(sA_u + stage * ABYTES + (m * LD + kx) * 8, g + m * 1201 % ATILE + kx, true);
        }
        cp_async_mbar_arrive_noinc(fullb);
      }
    }
    return;
  }
  reg_inc<224>();
  const int r = l >> 2, j = l & 3, wm = w & 3;
  double acc[2][WN][2];
#pragma unroll
  for (int t = 0; t < 2; t++)
#pragma unroll
    for (int u = 0; u < WN; u++) acc[t][u][0] = acc[t][u][1] = 0.0;
  for (int c = 0; c < nchunks; c++) {
    const int stage = c % STAGES;
    mbar_wait(full0 + 8 * stage, (c / STAGES) & 1);
    const double* a_ptr = sA + stage * ATILE + (wm * 16 + r) * LD + j;
    const double* b_ptr = sB + stage * BTILE + r * LD + j;
#pragma unroll
    for (int kk = 0; kk < KS; kk++) {
      const double a0 = a_ptr[4 * kk], a1 = a_ptr[8 * LD + 4 * kk];
      double b[WN];
#pragma unroll
      for (int u = 0; u < WN; u++) b[u] = b_ptr[u * 8 * LD + 4 * kk];
#pragma unroll
      for (int u = 0; u < WN; u++) { dmma884(acc[0][u][0], acc[0][u][1], a0, b[u]); dmma884(acc[1][u][0], acc[1][u][1], a1, b[u]); }
    }
    __syncwarp();
    if (l == 0) mbar_arrive(empty0 + 8 * stage);
  }
  double s = 0;
#pragma unroll
  for (int t = 0; t < 2; t++)
#pragma unroll
    for (int u = 0; u < WN; u++) s += acc[t][u][0] + acc[t][u][1];
  if (s == 12345.678) out[0] = s;
}
template <int KS, int PROD, int STAGES>
void run2(const double* src, double* out) {
  constexpr int LD = 4 * KS + 4;
  const size_t smem = (size_t)STAGES * (64 + 8 * WN) * LD * 8;
  const int nchunks = 60000 * 4 / KS;
  cudaFuncSetAttribute(k2<KS, PROD, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  int nb = 0; cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k2<KS, PROD, STAGES>, 256, smem);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  k2<KS, PROD, STAGES><<<296, 256, smem>>>(src, out, 100);
  cudaEventRecord(e0);
  k2<KS, PROD, STAGES><<<296, 256, smem>>>(src, out, nchunks);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  const double flops = 296.0 * 4 * (double)nchunks * KS * 2 * WN * 512;
  printf("2 CTAs/SM (occupancy %d): k-chunk %2d, %s, %d stages (%zu KB smem/CTA): %8.3f ms %6.2f TFLOP/s (%s)\n", nb, 4 * KS,
         PROD ? "cp.async8 A + bulk B" : "bulk A + bulk B     ", STAGES, smem >> 10, ms, flops / ms * 1e-9,
         cudaGetErrorString(cudaGetLastError()));
}
int main() {
  double *src, *out;
  const size_t n = 64 * (size_t)(64 + NT) * 36 * 2 + 4096;
  cudaMalloc(&src, n * 8); cudaMemset(src, 0, n * 8); cudaMalloc(&out, 8);
  run<4, 0, 0, 3>(src, out); run<4, 0, 1, 3>(src, out);
  run<4, 1, 0, 3>(src, out); run<4, 1, 1, 3>(src, out);
  run<8, 0, 0, 2>(src, out); run<8, 0, 1, 2>(src, out);
  run<8, 1, 0, 2>(src, out);
  run<2, 0, 0, 6>(src, out); run<2, 1, 0, 6>(src, out);
  run2<4, 0, 3>(src, out); run2<4, 1, 3>(src, out); run2<8, 0, 2>(src, out); run2<8, 1, 2>(src, out); run2<2, 1, 6>(src, out);
  return 0;
}
