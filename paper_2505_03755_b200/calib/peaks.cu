// Calibration microbenchmark (not on the product path): the roofline denominators that
// MEASURED_PEAKS.json does not carry -- FP64 tensor (DMMA.8x8x4) and vector (DFMA) issue peaks and
// the read-only HBM stream -- measured with CUDA events on one B200.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o peaks peaks.cu && ./peaks
#include <cstdio>
#include <cuda_runtime.h>

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int NACC>
__global__ void k_dmma(double* out, int iters) {
  double acc[NACC][2];
#pragma unroll
  for (int i = 0; i < NACC; i++) acc[i][0] = acc[i][1] = 0.0;
  const double a = 1.0 + threadIdx.x * 1e-3, b = 0.5;
  for (int it = 0; it < iters; it++)
#pragma unroll
    for (int i = 0; i < NACC; i++) dmma(acc[i][0], acc[i][1], a, b);
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < NACC; i++) s += acc[i][0] + acc[i][1];
  if (s == 123.456) out[0] = s;
}

template <int NACC>
__global__ void k_dfma(double* out, int iters) {
  double acc[NACC];
#pragma unroll
  for (int i = 0; i < NACC; i++) acc[i] = i;
  const double a = 1.0 + threadIdx.x * 1e-9, b = 1e-9;
#pragma unroll 8
  for (int it = 0; it < iters; it++)
#pragma unroll
    for (int i = 0; i < NACC; i++) acc[i] = fma(acc[i], a, b);
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < NACC; i++) s += acc[i];
  if (s == 123.456) out[0] = s;
}

// Issue rate of ONE warp per SM sub-partition as a function of operand reuse: 16 accumulators, DMMA i reads
// a[i % NA] and b[(i / 2) % NB] (NA = NB = 1: both operands reused; NA = 16, NB = 8: every DMMA reads fresh registers)
template <int NA, int NB>
__global__ void k_dmma_ops(double* out, int iters) {
  double acc[16][2], a[NA], b[NB];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i][0] = acc[i][1] = 0.0;
#pragma unroll
  for (int i = 0; i < NA; i++) a[i] = 1.0 + threadIdx.x * 1e-3 + i;
#pragma unroll
  for (int i = 0; i < NB; i++) b[i] = 0.5 + i * 0.25 + threadIdx.x;
  for (int it = 0; it < iters; it++)
#pragma unroll
    for (int i = 0; i < 16; i++) dmma(acc[i][0], acc[i][1], a[i % NA], b[(i / 2) % NB]);
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += acc[i][0] + acc[i][1];
  if (s == 123.456) out[0] = s;
}

// Do DMMA (tensor pipe) and DFMA (fp64 pipe) add up?  Even warps run the DMMA loop, odd warps the DFMA loop.
__global__ void k_mixed(double* out, int iters) {
  double acc[8][2], f[16];
#pragma unroll
  for (int i = 0; i < 8; i++) acc[i][0] = acc[i][1] = 0.0;
#pragma unroll
  for (int i = 0; i < 16; i++) f[i] = i;
  const double a = 1.0 + threadIdx.x * 1e-3, b = 0.5, c = 1e-9;
  if (((threadIdx.x >> 5) & 1) == 0) {
    for (int it = 0; it < iters; it++)
#pragma unroll
      for (int i = 0; i < 8; i++) dmma(acc[i][0], acc[i][1], a, b);       // 8 x 512 flop per warp and iteration
  } else {
    for (int it = 0; it < iters; it++)
#pragma unroll
      for (int i = 0; i < 64; i++) f[i & 15] = fma(f[i & 15], a, c);      // 64 x 64 flop per warp and iteration
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; i++) s += acc[i][0] + acc[i][1];
#pragma unroll
  for (int i = 0; i < 16; i++) s += f[i];
  if (s == 123.456) out[0] = s;
}

template <int U>
__global__ void k_read(const double2* __restrict__ p, size_t n, double* out) {
  double s = 0.0;
  const size_t stride = (size_t)gridDim.x * blockDim.x;
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (; i + (U - 1) * stride < n; i += U * stride) {
    double2 v[U];
#pragma unroll
    for (int u = 0; u < U; u++)
      asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v[u].x), "=d"(v[u].y) : "l"(p + i + u * stride));
#pragma unroll
    for (int u = 0; u < U; u++) s += v[u].x + v[u].y;
  }
  if (s == 123.456) out[0] = s;
}

static float time_ms(void (*launch)(void*), void* ctx) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  launch(ctx);
  cudaEventRecord(e0);
  launch(ctx);
  cudaEventRecord(e1);
  cudaEventSynchronize(e1);
  float ms;
  cudaEventElapsedTime(&ms, e0, e1);
  return ms;
}

struct Ctx { double* out; int warps; int iters; const double2* p; size_t n; int ctas; int threads; };
template <int NACC> void l_dmma(void* c) { Ctx* x = (Ctx*)c; k_dmma<NACC><<<148, 32 * x->warps>>>(x->out, x->iters); }
template <int NACC> void l_dfma(void* c) { Ctx* x = (Ctx*)c; k_dfma<NACC><<<148, 32 * x->warps>>>(x->out, x->iters); }
template <int NA, int NB> void l_ops(void* c) { Ctx* x = (Ctx*)c; k_dmma_ops<NA, NB><<<148, 32 * x->warps>>>(x->out, x->iters); }
void l_mixed(void* c) { Ctx* x = (Ctx*)c; k_mixed<<<148, 32 * x->warps>>>(x->out, x->iters); }
template <int U> void l_read(void* c) { Ctx* x = (Ctx*)c; k_read<U><<<148 * x->ctas, x->threads>>>(x->p, x->n, x->out); }

int main() {
  cudaDeviceProp prop;
  cudaGetDeviceProperties(&prop, 0);
  printf("%s, %d SMs, %.0f MHz\n", prop.name, prop.multiProcessorCount, prop.clockRate * 1e-3);
  Ctx c{};
  cudaMalloc(&c.out, 8);
  const int iters = 40000;
  c.iters = iters;
  for (int warps : {4, 8, 16, 32}) {
    c.warps = warps;
    float ms = time_ms(l_dmma<8>, &c);
    printf("dmma nacc=8  warps/SM=%2d  %7.3f ms  %6.2f TFLOP/s\n", warps, ms, 148.0 * warps * iters * 8 * 512 / ms * 1e-9);
    if (warps <= 16) {                                                 // 32 warps x 16 accumulator pairs do not fit the register file
      ms = time_ms(l_dmma<16>, &c);
      printf("dmma nacc=16 warps/SM=%2d  %7.3f ms  %6.2f TFLOP/s\n", warps, ms, 148.0 * warps * iters * 16 * 512 / ms * 1e-9);
    }
    ms = time_ms(l_dfma<16>, &c);
    printf("dfma nacc=16 warps/SM=%2d  %7.3f ms  %6.2f TFLOP/s\n", warps, ms, 148.0 * warps * 32 * iters * 16 * 2.0 / ms * 1e-9);
  }
  for (int warps : {4, 8}) {                                            // operand reuse: one / two warps per sub-partition
    c.warps = warps;
    const double f = 148.0 * warps * iters * 16 * 512 * 1e-9;
    printf("dmma operands warps/SM=%d  A,B reused %6.2f  A reused %6.2f  B reused %6.2f  none reused %6.2f TFLOP/s\n", warps,
           f / time_ms(l_ops<1, 1>, &c), f / time_ms(l_ops<1, 8>, &c), f / time_ms(l_ops<16, 1>, &c), f / time_ms(l_ops<16, 8>, &c));
  }
  for (int warps : {8, 16}) {                                           // half of the warps DMMA, the other half DFMA
    c.warps = warps;
    const float ms = time_ms(l_mixed, &c);
    const double tm = 148.0 * (warps / 2) * iters * 8 * 512 / ms * 1e-9, tf = 148.0 * (warps / 2) * iters * 64 * 64 / ms * 1e-9;
    printf("mixed warps/SM=%2d  %7.3f ms  dmma %6.2f + dfma %6.2f = %6.2f TFLOP/s\n", warps, ms, tm, tf, tm + tf);
  }
  c.warps = 16; c.iters = 40000 * 240;                                  // ~2.5 s: sustained
  float ms = time_ms(l_dmma<8>, &c);
  printf("dmma sustained %.1f ms per launch  %6.2f TFLOP/s\n", ms, 148.0 * 16 * (double)c.iters * 8 * 512 / ms * 1e-9);
  const size_t bytes = (size_t)8 << 30;
  double2* buf;
  cudaMalloc(&buf, bytes);
  cudaMemset(buf, 0, bytes);
  c.p = buf; c.n = bytes / 16;
  const int cfg[][2] = {{1, 256}, {1, 1024}, {2, 512}, {4, 256}, {8, 1024}};
  for (auto& f : cfg) {
    c.ctas = f[0]; c.threads = f[1];
    const float m4 = time_ms(l_read<4>, &c), m8 = time_ms(l_read<8>, &c), m16 = time_ms(l_read<16>, &c);
    printf("read ctas/SM=%d threads=%4d  U4 %7.1f  U8 %7.1f  U16 %7.1f GB/s\n", f[0], f[1], bytes / m4 * 1e-6, bytes / m8 * 1e-6,
           bytes / m16 * 1e-6);
  }
  printf("%s\n", cudaGetErrorString(cudaGetLastError()));
  return 0;
}
