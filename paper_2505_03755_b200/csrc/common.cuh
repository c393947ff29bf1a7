// Shared device helpers for the DF-JK kernels (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "dfjk kernels are written for sm_100a only"
#endif

namespace dfjk {

// packed lower-triangle offset of row mu: idx(mu,nu) = mu(mu+1)/2 + nu, mu >= nu
__host__ __device__ __forceinline__ size_t tri(int mu) { return (size_t)mu * (size_t)(mu + 1) / 2; }

__host__ __device__ __forceinline__ int cdiv(int a, int b) { return (a + b - 1) / b; }
__host__ __device__ __forceinline__ int round_up(int a, int b) { return cdiv(a, b) * b; }

// FP64 tensor-core MMA, D(8x8) += A(8x4) * B(4x8).  SASS: DMMA.8x8x4 (the only native FP64 tensor
// shape on sm_100a; tcgen05/TMEM have no f64 kind).  Lane l holds
//   A[row = l/4][k = l%4],  B[k = l%4][col = l/4],  C/D[row = l/4][col = 2*(l%4) + {0,1}].
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(d0), "+d"(d1)
               : "d"(a), "d"(b));
}

// x with its sign bit flipped when m = 0x80000000 (m = 0: unchanged); an integer op on the high word
__device__ __forceinline__ double flip_sign(double x, unsigned int m) {
  return __hiloint2double(__double2hiint(x) ^ (int)m, __double2loint(x));
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}

// Ampere-style async copies (SASS LDGSTS).  src_bytes < cp-size zero-fills the rest.
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src, bool pred) {
  const int n = pred ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(n) : "memory");
}
// streaming 128-bit read of B: read-only path, do not keep in L1
__device__ __forceinline__ double2 ldg_stream2(const double* p) {
  double2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ double ldg_stream1(const double* p) {
  double v;
  asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}

}  // namespace dfjk
