// Steps a5-a9, the exchange build (Eq. 16-17) on the FP64 tensor pipe:
//   a5/a6  half-transform  X[P][mu][i] = sum_lam B_P[mu][lam] C'[lam][i]   (k_half_transform)
//          the A operand is read straight from the packed triangle: chunks below the diagonal
//          as stored, chunks above it as the transpose of the stored tile (only the shared-memory
//          read pattern changes), chunks crossing it element by element.
//   a7     SYRK            K_s[mu>=nu] += sum_{P,i in s} X[P][mu][i] X[P][nu][i]   (k_syrk)
//          lower-triangle 128x128 tiles, split-K over the aux rows of the block, partials
//          read-modify-written by exactly one CTA each (no atomics: deterministic).
//   a9     epilogue        fixed-order sum of the split-K partials, mirrored to both triangles.
// Both GEMMs run DMMA.8x8x4 (mma.sync m8n8k4 f64) from shared-memory tiles whose row stride is
// 4 mod 16 doubles, which makes both the [row][k] and the [k][row] fragment reads conflict-free.
#include "common.cuh"
#include "ctx.h"

namespace dfjk {

constexpr int kStages = 3;
constexpr int kLdT = kBK + 4;        // 36: row stride of a [rows][kBK] tile
constexpr int kLdTT = 128 + 4;       // 132: row stride of a transposed [kBK][128] tile
constexpr int kTileDoubles = 128 * kLdT;  // 4608 >= kBK * kLdTT = 4224

// ------------------------------------------------------------------ half-transform
// CTA: 128 rows (mu) of one aux slice x NT = 8*WN columns; 8 warps stacked along M (16 rows each).
template <int WN>
__global__ void __launch_bounds__(256, 1)
k_half_transform(const double* __restrict__ Bp, size_t npair, int nao, int nao_k,
                 const double* __restrict__ Ct, int nocc_pad, double* __restrict__ X, int p_first) {
  extern __shared__ __align__(16) double smem[];
  constexpr int NT = 8 * WN;
  double* sA = smem;                               // kStages x kTileDoubles
  double* sB = smem + kStages * kTileDoubles;      // kStages x NT*kLdT
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31, r = l >> 2, j = l & 3;
  const int n0 = blockIdx.x * NT, m0 = blockIdx.y * 128, pl = blockIdx.z;
  const double* BpP = Bp + (size_t)(p_first + pl) * npair;
  const int nchunks = nao_k / kBK;

  auto chunk_mode = [&](int c) -> int {  // 0 = stored rows (direct), 1 = transposed, 2 = crossing
    const int l0 = c * kBK;
    if (l0 + kBK - 1 <= m0) return 0;
    if (l0 >= m0 + 127) return 1;
    return 2;
  };
  auto load_chunk = [&](int c, int stage) {
    const int l0 = c * kBK, mode = chunk_mode(c);
    const uint32_t a_base = smem_u32(sA + stage * kTileDoubles);
    if (mode == 1) {
      const int m = tid & 127, mu = m0 + m;
#pragma unroll
      for (int q = 0; q < 16; q++) {
        const int k = (tid >> 7) + 2 * q, lam = l0 + k;
        const bool ok = mu < nao && lam < nao;
        const double* src = BpP + (ok ? tri(lam) + mu : 0);
        cp_async8(a_base + (uint32_t)(k * kLdTT + m) * 8u, src, ok);
      }
    } else {
      const int k = tid & 31, lam = l0 + k;
#pragma unroll
      for (int q = 0; q < 16; q++) {
        const int m = (tid >> 5) + 8 * q, mu = m0 + m;
        const bool ok = mu < nao && lam < nao;
        size_t off = 0;
        if (ok) off = (lam <= mu) ? tri(mu) + lam : tri(lam) + mu;
        cp_async8(a_base + (uint32_t)(m * kLdT + k) * 8u, BpP + off, ok);
      }
    }
    const uint32_t b_base = smem_u32(sB + stage * NT * kLdT);
    for (int e = tid; e < NT * (kBK / 2); e += 256) {
      const int n = e >> 4, k2 = (e & 15) * 2;
      const bool ok = n0 + n < nocc_pad;
      const double* src = Ct + (ok ? (size_t)(n0 + n) * nao_k + l0 + k2 : 0);
      cp_async16(b_base + (uint32_t)(n * kLdT + k2) * 8u, src, ok);
    }
  };

  double acc[2][WN][2];
#pragma unroll
  for (int t = 0; t < 2; t++)
#pragma unroll
    for (int u = 0; u < WN; u++) acc[t][u][0] = acc[t][u][1] = 0.0;

  for (int s = 0; s < kStages - 1; s++) {
    if (s < nchunks) load_chunk(s, s);
    cp_async_commit();
  }
  for (int c = 0; c < nchunks; c++) {
    cp_async_wait<kStages - 2>();
    __syncthreads();
    if (c + kStages - 1 < nchunks) load_chunk(c + kStages - 1, (c + kStages - 1) % kStages);
    cp_async_commit();
    const int stage = c % kStages;
    const bool tr = chunk_mode(c) == 1;
    const int sM = tr ? 1 : kLdT, sK = tr ? kLdTT : 1;
    const double* a_ptr = sA + stage * kTileDoubles + (w * 16 + r) * sM + j * sK;
    const double* b_ptr = sB + stage * NT * kLdT + r * kLdT + j;
#pragma unroll
    for (int kk = 0; kk < kBK / 4; kk++) {
      const double a0 = a_ptr[4 * kk * sK], a1 = a_ptr[8 * sM + 4 * kk * sK];
      double b[WN];
#pragma unroll
      for (int u = 0; u < WN; u++) b[u] = b_ptr[u * 8 * kLdT + 4 * kk];
#pragma unroll
      for (int u = 0; u < WN; u++) {
        dmma884(acc[0][u][0], acc[0][u][1], a0, b[u]);
        dmma884(acc[1][u][0], acc[1][u][1], a1, b[u]);
      }
    }
  }
  cp_async_wait<0>();
  // epilogue: lane owns X[mu][n], X[mu][n+1] with mu = m0 + 16w + 8t + r, n = n0 + 8u + 2j
  double* Xp = X + (size_t)pl * nao * nocc_pad;
#pragma unroll
  for (int t = 0; t < 2; t++) {
    const int mu = m0 + w * 16 + 8 * t + r;
    if (mu >= nao) continue;
#pragma unroll
    for (int u = 0; u < WN; u++) {
      const int n = n0 + 8 * u + 2 * j;
      if (n < nocc_pad)
        *reinterpret_cast<double2*>(Xp + (size_t)mu * nocc_pad + n) = make_double2(acc[t][u][0], acc[t][u][1]);
    }
  }
}

// ------------------------------------------------------------------ SYRK
// CTA: one lower-triangle 128x128 tile (ta >= tb) of K_s, one split of the block's aux rows.
// 8 warps as 2 (M) x 4 (N), warp tile 64x32 = 8x4 MMA tiles.  The reduction runs over chunks
// (P, 32 columns of set s); both operands are [row][k] tiles of X, the diagonal tile loads one.
__global__ void __launch_bounds__(256, 1)
k_syrk(const double* __restrict__ X, int nao, int ldx, int c0, int c1, int nrows_blk, int rows_per_split,
       int ntiles_m, double* __restrict__ Kpart_s, size_t split_stride, int first) {
  extern __shared__ __align__(16) double smem[];
  double* sA = smem;
  double* sB = smem + kStages * kTileDoubles;
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31, r = l >> 2, j = l & 3;
  const int wm = w >> 2, wn = w & 3;
  // tile index -> (ta, tb), ta >= tb
  const int ntiles = ntiles_m * (ntiles_m + 1) / 2;
  const int t = blockIdx.x % ntiles, g = blockIdx.x / ntiles;
  int ta = (int)((sqrt(8.0 * t + 1.0) - 1.0) * 0.5);
  while ((ta + 1) * (ta + 2) / 2 <= t) ta++;
  while (ta * (ta + 1) / 2 > t) ta--;
  const int tb = t - ta * (ta + 1) / 2;
  const bool diag = ta == tb;
  const int a0 = ta * 128, b0 = tb * 128;
  const int p_beg = g * rows_per_split;
  int p_end = p_beg + rows_per_split;
  if (p_end > nrows_blk) p_end = nrows_blk;
  const int np = p_end > p_beg ? p_end - p_beg : 0;
  const int cps = (c1 - c0 + kBK - 1) / kBK;   // chunks per aux row
  const int nchunks = np * cps;

  auto load_chunk = [&](int c, int stage) {
    const int P = p_beg + c / cps, i0 = c0 + (c % cps) * kBK;
    const int klen = min(kBK, c1 - i0);          // multiple of 8
    const double* Xp = X + (size_t)P * nao * ldx + i0;
    const uint32_t a_base = smem_u32(sA + stage * kTileDoubles);
    const uint32_t b_base = smem_u32(sB + stage * kTileDoubles);
    const int k2 = (tid & 15) * 2;
    if (k2 < klen) {
#pragma unroll
      for (int q = 0; q < 8; q++) {
        const int m = (tid >> 4) + 16 * q;
        const bool oka = a0 + m < nao;
        cp_async16(a_base + (uint32_t)(m * kLdT + k2) * 8u, Xp + (oka ? (size_t)(a0 + m) * ldx + k2 : 0), oka);
        if (!diag) {
          const bool okb = b0 + m < nao;
          cp_async16(b_base + (uint32_t)(m * kLdT + k2) * 8u, Xp + (okb ? (size_t)(b0 + m) * ldx + k2 : 0), okb);
        }
      }
    }
  };

  double acc[8][4][2];
#pragma unroll
  for (int tt = 0; tt < 8; tt++)
#pragma unroll
    for (int u = 0; u < 4; u++) acc[tt][u][0] = acc[tt][u][1] = 0.0;

  for (int s = 0; s < kStages - 1; s++) {
    if (s < nchunks) load_chunk(s, s);
    cp_async_commit();
  }
  for (int c = 0; c < nchunks; c++) {
    cp_async_wait<kStages - 2>();
    __syncthreads();
    if (c + kStages - 1 < nchunks) load_chunk(c + kStages - 1, (c + kStages - 1) % kStages);
    cp_async_commit();
    const int stage = c % kStages;
    const int i0 = c0 + (c % cps) * kBK;
    const int ksteps = min(kBK, c1 - i0) / 4;
    const double* a_ptr = sA + stage * kTileDoubles + (wm * 64 + r) * kLdT + j;
    const double* b_ptr = (diag ? sA : sB) + stage * kTileDoubles + (wn * 32 + r) * kLdT + j;
#pragma unroll 2
    for (int kk = 0; kk < ksteps; kk++) {
      double a[8], b[4];
#pragma unroll
      for (int tt = 0; tt < 8; tt++) a[tt] = a_ptr[tt * 8 * kLdT + 4 * kk];
#pragma unroll
      for (int u = 0; u < 4; u++) b[u] = b_ptr[u * 8 * kLdT + 4 * kk];
#pragma unroll
      for (int tt = 0; tt < 8; tt++)
#pragma unroll
        for (int u = 0; u < 4; u++) dmma884(acc[tt][u][0], acc[tt][u][1], a[tt], b[u]);
    }
  }
  cp_async_wait<0>();
  // read-modify-write this CTA's private partial tile (full 128x128, also above the diagonal of
  // a diagonal tile; the epilogue reads mu >= nu only)
  double* Kp = Kpart_s + (size_t)g * split_stride;
#pragma unroll
  for (int tt = 0; tt < 8; tt++) {
    const int mu = a0 + wm * 64 + 8 * tt + r;
    if (mu >= nao) continue;
#pragma unroll
    for (int u = 0; u < 4; u++) {
      const int nu = b0 + wn * 32 + 8 * u + 2 * j;
      double* p = Kp + (size_t)mu * nao + nu;
      if (nu < nao) p[0] = first ? acc[tt][u][0] : p[0] + acc[tt][u][0];
      if (nu + 1 < nao) p[1] = first ? acc[tt][u][1] : p[1] + acc[tt][u][1];
    }
  }
}

// Step a9: K_s[mu][nu] = K_s[nu][mu] = sum_g Kpart[g][s][mu][nu] for mu >= nu, g ascending.
__global__ void __launch_bounds__(256)
k_k_epilogue(const double* __restrict__ Kpart, int nsplit, size_t split_stride, int nao, double* __restrict__ K) {
  const int bi = blockIdx.x, bj = blockIdx.y, s = blockIdx.z;
  if (bj > bi) return;
  __shared__ double t[32][33];
  const int tx = threadIdx.x, ty = threadIdx.y;
  const double* src = Kpart + (size_t)s * nao * nao;
  for (int r = ty; r < 32; r += 8) {
    const int mu = bi * 32 + r, nu = bj * 32 + tx;
    double v = 0.0;
    if (mu < nao && nu <= mu)
      for (int g = 0; g < nsplit; g++) v += src[(size_t)g * split_stride + (size_t)mu * nao + nu];
    t[r][tx] = v;
  }
  __syncthreads();
  double* Ks = K + (size_t)s * nao * nao;
  for (int r = ty; r < 32; r += 8) {
    const int mu = bi * 32 + r, nu = bj * 32 + tx;
    if (mu < nao && nu < nao) {
      if (bi != bj) Ks[(size_t)mu * nao + nu] = t[r][tx];
      else Ks[(size_t)mu * nao + nu] = (nu <= mu) ? t[r][tx] : t[tx][r];
    }
    if (bi != bj) {
      const int row = bj * 32 + r, colm = bi * 32 + tx;
      if (row < nao && colm < nao) Ks[(size_t)row * nao + colm] = t[tx][r];
    }
  }
}

__global__ void k_zero(double* p, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = 0.0;
}

// ------------------------------------------------------------------ launchers (step a8)
static size_t ht_smem_bytes(int wn) { return (size_t)kStages * (kTileDoubles + 8 * wn * kLdT) * sizeof(double); }
static size_t syrk_smem_bytes() { return (size_t)kStages * 2 * kTileDoubles * sizeof(double); }

template <int WN>
static cudaError_t launch_ht(dim3 grid, cudaStream_t st, const double* Bp, size_t npair, int nao, int nao_k,
                             const double* Ct, int nocc_pad, double* X, int p_first) {
  static bool attr_set = false;  // per-process, per-instantiation; the attribute is per-function
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(k_half_transform<WN>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)ht_smem_bytes(WN));
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  k_half_transform<WN><<<grid, 256, ht_smem_bytes(WN), st>>>(Bp, npair, nao, nao_k, Ct, nocc_pad, X, p_first);
  return cudaSuccess;
}

static cudaError_t dispatch_ht(int wn, dim3 grid, cudaStream_t st, const double* Bp, size_t npair, int nao,
                               int nao_k, const double* Ct, int nocc_pad, double* X, int p_first) {
  switch (wn) {
#define DFJK_HT_CASE(N) \
  case N: return launch_ht<N>(grid, st, Bp, npair, nao, nao_k, Ct, nocc_pad, X, p_first);
    DFJK_HT_CASE(1) DFJK_HT_CASE(2) DFJK_HT_CASE(3) DFJK_HT_CASE(4) DFJK_HT_CASE(5) DFJK_HT_CASE(6)
    DFJK_HT_CASE(7) DFJK_HT_CASE(8) DFJK_HT_CASE(9) DFJK_HT_CASE(10) DFJK_HT_CASE(11) DFJK_HT_CASE(12)
    DFJK_HT_CASE(13) DFJK_HT_CASE(14) DFJK_HT_CASE(15) DFJK_HT_CASE(16)
#undef DFJK_HT_CASE
    default: return cudaErrorInvalidValue;
  }
}

// Aux-block scheduler: cap the X workspace, pick the split-K factor, enqueue
// half-transform and SYRK block after block on one stream.  No allocation, no host sync.
int launch_k_path(dfjk_ctx* h, const SetInfo& si, double* K_out, cudaStream_t st) {
  int launches = 0;
  const int nao = h->nao, naux = h->naux;
  const size_t n2 = (size_t)nao * nao;
  const int nb32 = cdiv(nao, 32);
  const int ldx = si.nocc_pad;
  // sets without columns (or no aux rows at all): K_s = 0
  prof_mark(h, DFJK_PHASE_K_EPILOGUE, st);
  for (int s = 0; s < si.nset; s++)
    if (naux == 0 || si.col0[s + 1] == si.col0[s]) {
      k_zero<<<148, 256, 0, st>>>(K_out + n2 * s, n2);
      launches++;
    }
  if (naux == 0 || ldx == 0) return launches;

  // plan: aux block size from the workspace, N tiling of the half-transform, split-K of the SYRK
  const size_t row_bytes = (size_t)nao * ldx * sizeof(double);
  long long nblk = (long long)(h->X_doubles * sizeof(double) / row_bytes);
  if (h->nblk_forced > 0 && nblk > h->nblk_forced) nblk = h->nblk_forced;
  if (nblk > naux) nblk = naux;
  if (nblk > 32768) nblk = 32768;
  if (nblk < 1) nblk = 1;
  const int n8 = ldx / 8;
  const int ntn = cdiv(n8, 16), wn = cdiv(n8, ntn);
  const int ntm = h->n_mtiles, ntiles = ntm * (ntm + 1) / 2;
  int ksplit = h->ksplit_forced;
  if (ksplit <= 0) {
    // fill the 148 SMs (one SYRK CTA each) about three times over with the heaviest set
    ksplit = cdiv(3 * 148, ntiles);
    if (ksplit > h->ksplit) ksplit = h->ksplit;
  }
  if (ksplit > nblk) ksplit = (int)nblk;
  if (ksplit < 1) ksplit = 1;
  const size_t split_stride = (size_t)h->max_nset * n2;

  static bool syrk_attr = false;
  if (!syrk_attr) {
    if (cudaFuncSetAttribute(k_syrk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)syrk_smem_bytes()) != cudaSuccess)
      return -1;
    syrk_attr = true;
  }
  int nblocks = 0;
  for (int p0 = 0; p0 < naux; p0 += (int)nblk, nblocks++) {
    const int nb = (int)(naux - p0 < nblk ? naux - p0 : nblk);
    dim3 gh(ntn, ntm, nb);
    prof_mark(h, DFJK_PHASE_HALF_TRANSFORM, st);
    if (dispatch_ht(wn, gh, st, h->B, h->npair, nao, h->nao_k, h->Ct, ldx, h->X, p0) != cudaSuccess) return -1;
    launches++;
    const int rps = cdiv(nb, ksplit);
    prof_mark(h, DFJK_PHASE_SYRK, st);
    for (int s = 0; s < si.nset; s++) {
      if (si.col0[s + 1] == si.col0[s]) continue;
      k_syrk<<<ntiles * ksplit, 256, syrk_smem_bytes(), st>>>(h->X, nao, ldx, si.col0[s], si.col0[s + 1], nb, rps,
                                                            ntm, h->Kpart + n2 * s, split_stride, p0 == 0 ? 1 : 0);
      launches++;
    }
  }
  prof_mark(h, DFJK_PHASE_K_EPILOGUE, st);
  for (int s = 0; s < si.nset; s++) {
    if (si.col0[s + 1] == si.col0[s]) continue;
    dim3 ge(nb32, nb32, 1), be(32, 8);
    k_k_epilogue<<<ge, be, 0, st>>>(h->Kpart + n2 * s, ksplit, split_stride, nao, K_out + n2 * s);
    launches++;
  }
  h->plan_nblk = (int)nblk;
  h->plan_ksplit = ksplit;
  h->plan_nblocks = nblocks;
  return launches;
}

// ------------------------------------------------------------------ DMMA fragment self-test
__global__ void k_dmma_selftest(int* bad) {
  __shared__ double A[8][4], Bm[4][8], Cm[8][8];
  const int l = threadIdx.x;
  for (int e = l; e < 32; e += 32) {
    A[e / 4][e % 4] = 1.0 + 0.37 * e - 0.011 * e * e;
    Bm[e / 8][e % 8] = -2.0 + 0.53 * e + 0.007 * e * e;
  }
  for (int e = l; e < 64; e += 32) Cm[e / 8][e % 8] = 0.25 * e - 3.0;
  __syncwarp();
  double d0 = Cm[l >> 2][2 * (l & 3)], d1 = Cm[l >> 2][2 * (l & 3) + 1];
  dmma884(d0, d1, A[l >> 2][l & 3], Bm[l & 3][l >> 2]);
  int nb = 0;
  for (int c = 0; c < 2; c++) {
    const int row = l >> 2, col = 2 * (l & 3) + c;
    double ref = Cm[row][col];
    for (int k = 0; k < 4; k++) ref = fma(A[row][k], Bm[k][col], ref);
    const double got = c ? d1 : d0;
    if (fabs(got - ref) > 1e-12 * (1.0 + fabs(ref))) nb++;
  }
  if (nb) atomicAdd(bad, nb);
}

int run_dmma_selftest() {
  int* d = nullptr;
  int hbad = -1;
  if (cudaMalloc(&d, sizeof(int)) != cudaSuccess) return -1;
  cudaMemset(d, 0, sizeof(int));
  k_dmma_selftest<<<1, 32>>>(d);
  cudaError_t e = cudaMemcpy(&hbad, d, sizeof(int), cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return -1;
  return hbad;
}

}  // namespace dfjk
