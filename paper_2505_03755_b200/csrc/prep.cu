// Step a1, density prep (Eq. 14 needs D; Eq. 16 needs gamma = C n C^T):
//   Ct[i][lam]  = sqrt(|n_i|) C[lam][i] all sets concatenated, each set padded to 8 columns with
//                                       zeros, lam padded to a multiple of 16 with zeros; stored
//                                       k-tiled as Ct[(lam/16 * ct_rows + i) * 20 + lam%16] so that
//                                       the half-transform fetches a whole k-chunk of its B operand
//                                       with one bulk copy, already in the padded smem layout;
//   sgnbits     bit i%32 of word i/32 is set iff n_i < 0: D = C' diag(sign n) C'^T exactly, so signed
//               occupations (differences of densities) cost what unsigned ones do;
//               the SYRK, the fused rho and Dw apply the sign as a flip of the fp64 sign bit;
//   Dw_s[pair]  = (2 - delta_{mu nu}) sum_i sign(n_i) Ct[i][mu] Ct[i][nu]   packed, off-diagonal
//                 weight 2, so that the packed dot product with B_P equals the full-square sum of Eq. 14.
#include "common.cuh"
#include "ctx.h"

namespace dfjk {

__global__ void __launch_bounds__(256)
k_prep_ct(const __grid_constant__ SetInfo si, const double* __restrict__ C, const double* __restrict__ occ,
          double* __restrict__ Ct, unsigned int* __restrict__ sgnbits, int nao, int nk_pad, int ct_rows) {
  __shared__ double t[32][33];
  const int tx = threadIdx.x, ty = threadIdx.y;
  const int lam0 = blockIdx.x * 32, ip0 = blockIdx.y * 32;
  const int ip = ip0 + tx;
  // which set owns padded column ip (uniform per thread over the row loop)
  int s = -1, il = 0;
  if (ip < si.nocc_pad) {
    for (int q = 0; q < si.nset; q++)
      if (ip >= si.col0[q] && ip < si.col0[q + 1]) s = q;
    il = ip - si.col0[s];
    if (il >= si.nocc[s]) s = -1;  // padding column
  }
  double scale = 0.0;
  bool neg = false;
  if (s >= 0) {
    const double n = occ ? occ[si.ooff[s] + il] : 1.0;          // occ == nullptr: plain coefficients (AO2MO)
    scale = sqrt(fabs(n));
    neg = n < 0.0;
  }
  if (blockIdx.x == 0 && ty == 0) {                             // this block's 32 padded columns = one sign word
    const unsigned int word = __ballot_sync(0xffffffffu, neg);
    if (tx == 0) sgnbits[blockIdx.y] = word;
  }
  for (int r = ty; r < 32; r += 8) {
    const int lam = lam0 + r;
    double v = 0.0;
    if (s >= 0 && lam < nao) v = scale * C[si.coff[s] + (long long)lam * si.nocc[s] + il];
    t[r][tx] = v;
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int ipw = ip0 + r, lam = lam0 + tx;
    if (ipw < si.nocc_pad && lam < nk_pad)
      Ct[((size_t)(lam >> 4) * ct_rows + ipw) * kHtLd + (lam & 15)] = t[tx][r];
  }
}

// 64x64 tile of D_s per CTA, 4x4 per thread, plain DFMA (0.4 GFLOP at nao=1200: negligible).
__global__ void __launch_bounds__(256)
k_prep_dw(const __grid_constant__ SetInfo si, const double* __restrict__ Ct, const unsigned int* __restrict__ sgnbits,
          double* __restrict__ Dw, int nao, int nk_pad, int ct_rows, size_t npair) {
  const int bi = blockIdx.x, bj = blockIdx.y, s = blockIdx.z;
  if (bj > bi) return;
  __shared__ double As[16][64], Bs[16][64];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  double acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; a++)
#pragma unroll
    for (int b = 0; b < 4; b++) acc[a][b] = 0.0;
  const int c0 = si.col0[s], c1 = si.col0[s + 1];
  for (int i0 = c0; i0 < c1; i0 += 16) {
    for (int e = tid; e < 16 * 64; e += 256) {
      const int ii = e >> 6, m = e & 63, i = i0 + ii;
      const int la = bi * 64 + m, lb = bj * 64 + m;
      As[ii][m] = (i < c1 && la < nk_pad) ? Ct[((size_t)(la >> 4) * ct_rows + i) * kHtLd + (la & 15)] : 0.0;
      double bv = (i < c1 && lb < nk_pad) ? Ct[((size_t)(lb >> 4) * ct_rows + i) * kHtLd + (lb & 15)] : 0.0;
      if (i < c1 && ((sgnbits[i >> 5] >> (i & 31)) & 1u)) bv = -bv;
      Bs[ii][m] = bv;
    }
    __syncthreads();
#pragma unroll
    for (int ii = 0; ii < 16; ii++) {
      double av[4], bv[4];
#pragma unroll
      for (int a = 0; a < 4; a++) av[a] = As[ii][ty * 4 + a];
#pragma unroll
      for (int b = 0; b < 4; b++) bv[b] = Bs[ii][tx * 4 + b];
#pragma unroll
      for (int a = 0; a < 4; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) acc[a][b] = fma(av[a], bv[b], acc[a][b]);
    }
    __syncthreads();
  }
  double* out = Dw + (size_t)s * npair;
#pragma unroll
  for (int a = 0; a < 4; a++) {
    const int mu = bi * 64 + ty * 4 + a;
    if (mu >= nao) continue;
#pragma unroll
    for (int b = 0; b < 4; b++) {
      const int nu = bj * 64 + tx * 4 + b;
      if (nu <= mu) out[tri(mu) + nu] = (mu == nu ? 1.0 : 2.0) * acc[a][b];
    }
  }
}

int launch_prep_ct(dfjk_ctx* h, const SetInfo& si, const double* C, const double* occ, cudaStream_t st) {
  if (si.nocc_pad == 0) return 0;
  prof_mark(h, DFJK_PHASE_PREP, st);
  dim3 grid(cdiv(h->nck * kHtBK, 32), cdiv(si.nocc_pad, 32)), block(32, 8);
  k_prep_ct<<<grid, block, 0, st>>>(si, C, occ, h->Ct, h->sgnbits, h->nao, h->nck * kHtBK, h->ct_rows);
  return 1;
}

int launch_prep_dw(dfjk_ctx* h, const SetInfo& si, cudaStream_t st) {
  prof_mark(h, DFJK_PHASE_PREP, st);
  const int nb = cdiv(h->nao, 64);
  dim3 grid(nb, nb, si.nset);
  k_prep_dw<<<grid, 256, 0, st>>>(si, h->Ct, h->sgnbits, h->Dw, h->nao, h->nck * kHtBK, h->ct_rows, h->npair);
  return 1;
}

}  // namespace dfjk
