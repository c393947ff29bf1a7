// AO2MO, the paper's second GPU kernel (Eq. 18-21):
//   Eq. 18  X^P[e2][p1]   = sum_{e1} b^P[e1][e2] M[e1][p1]        the half-transform of the JK path
//                                                                 (k_half_transform, row-major epilogue)
//   Eq. 19  bmo^P[p1][p2] = sum_{e2} X^P[e2][p1] M[e2][p2]
//   Eq. 20  ppaa[p1][p2][a1][a2] = sum_P bmo^P[p1][p2] bmo^P[a0+a1][a0+a2]
//   Eq. 21  papa[p1][a1][p2][a2] = sum_P bpa[P][p1][a1] bpa[P][p2][a2],   bpa[P][p][a] = bmo^P[p][a0+a]
// Eq. 19-21 are all of the form C (M x N) (+)= A^T B with both operands stored k-major
// (A is [K][M], B is [K][N]): one warp-specialised DMMA kernel, k_gemm_tn, serves the three.
// Aux blocks of N_blk rows bound the workspace (X block + bmo block, "2 N_blk N_emb^2").
#include "common.cuh"
#include "ctx.h"
#include "pipeline.cuh"

namespace dfjk {

constexpr int kGStages = 4;
constexpr int kGKC = 16;                  // k-chunk of the pipeline (4 k4 steps)
constexpr int kGThreads = 384;            // 8 consumer warps + 4 producer warps

struct GemmTN {
  const double* A; const double* B; double* C;
  int M, N, K;
  long long lda, ldb, ldc;                // row strides (doubles) of the k-major operands and of C
  long long sA, sB, sC;                   // batch strides (blockIdx.z)
  int accumulate;                         // 0: C = A^T B, 1: C += A^T B (one CTA owns each C tile)
  // grouped M index of A (0 = plain): column m of A lives at (m / a_group) * a_gstride + k * lda +
  // m % a_group -- the aux rows of a block stacked along M (Eq. 19 for the whole block as ONE
  // GEMM of nb * nmo rows, so that only the N dimension pays tile padding)
  int a_group = 0;
  long long a_gstride = 0;
  // grouped row index of C (0 = plain): element (m, n) is stored at (m / c_group) * c_gstride +
  // n * c_nstride + m % c_group -- the transposed per-aux-row blocks bpa[P][p][a] written by a GEMM
  // whose rows are (P, a) and whose columns are p
  int c_group = 0;
  long long c_gstride = 0, c_nstride = 0;
  // 1: C is known to be symmetric (Eq. 21: A == B): tiles that lie entirely above the diagonal are skipped and
  // k_mirror_lower fills the upper triangle from the lower one afterwards
  int lower_only = 0;
};

// CTA tile (8 WTM WGM) x (8 WTN WGN), WGM x WGN = 8 consumer warps, warp tile WTM x WTN MMA tiles.  WGM = 2:
// 2 (M) x 4 (N) warps, 64 or 128 rows x up to 352 columns; WGM = 8: all warps along M, 128 rows x 8 WTN columns
// for tall and narrow products whose N is not a multiple of 32 (W of the active-first route, N = 36).
// Shared-memory tiles are k-major, [16][TM + 4] and [16][TN + 4]: the row stride is 4 mod 16
// doubles, so the fragment reads tile[k = l%4][row = l/4] hit 16 distinct banks per half-warp.
// Producers: BULK = true -- both operands are plain k-major matrices whose rows start 16-byte aligned
// (even leading dimensions and tile origins, K a multiple of 4): every k row of a tile is one
// contiguous run, fetched by a bulk async copy (TMA engine, UBLKCP); sixteen lanes of one producer
// warp issue the 32 row copies of a stage, completion is counted in bytes.  Columns past M or N are
// never stored, so tails need no zero fill.  BULK = false -- 8-byte cp.async gathers (any alignment,
// grouped A rows, zero-fill past M, N, K).
template <int WTM, int WTN, bool BULK, int WGM = 2>
__global__ void __launch_bounds__(kGThreads, 1)
k_gemm_tn(const __grid_constant__ GemmTN g) {
  constexpr int WGN = 8 / WGM;
  constexpr int TM = 8 * WTM * WGM, TN = 8 * WTN * WGN, LA = TM + 4, LB = TN + 4;
  static_assert(LA % 16 == 4 || LA % 16 == 12, "A tile row stride must be +-4 mod 16 doubles");
  static_assert(LB % 16 == 4 || LB % 16 == 12, "B tile row stride must be +-4 mod 16 doubles");
  constexpr int kStageDoubles = kGKC * (LA + LB);
  extern __shared__ __align__(128) double smem[];
  __shared__ __align__(8) unsigned long long bars[2 * kGStages];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kGStages]);
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
  const int m0 = blockIdx.x * TM, n0 = blockIdx.y * TN;
  if (g.lower_only && n0 >= m0 + TM) return;          // every element of this tile has n > m
  const double* A = g.A + (size_t)blockIdx.z * g.sA;
  const double* B = g.B + (size_t)blockIdx.z * g.sB;
  double* C = g.C + (size_t)blockIdx.z * g.sC;
  const int nchunks = (g.K + kGKC - 1) / kGKC;

  if (tid == 0) {
    for (int s = 0; s < kGStages; s++) {
      mbar_init(full0 + 8 * s, BULK ? 1 : 128);   // the expect_tx arrival / one cp.async-completion arrival per producer thread
      mbar_init(empty0 + 8 * s, 8);        // one arrival per consumer warp
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (w >= 8) {
    // ===================== producer warpgroup =====================
    reg_dec<kProducerRegs>();
    const int tp = tid - 256;
    if constexpr (BULK) {
      if (tp >= kGKC) return;               // lane k of the first producer warp owns k row k of every stage
      const int mrows = min(TM, g.M - m0), ncols = min(TN, g.N - n0);
      const uint32_t a_bytes = (uint32_t)mrows * 8u, b_bytes = (uint32_t)ncols * 8u;
      const double* Ak = A + (size_t)m0 + (size_t)tp * g.lda;
      const double* Bk = B + (size_t)n0 + (size_t)tp * g.ldb;
      for (int c = 0; c < nchunks; c++) {
        const int stage = c % kGStages;
        const uint32_t fullb = full0 + 8 * stage;
        mbar_wait(empty0 + 8 * stage, ((c / kGStages) & 1) ^ 1);
        const int krows = min(kGKC, g.K - c * kGKC);             // a multiple of 4
        if (tp == 0) mbar_arrive_expect_tx(fullb, (uint32_t)krows * (a_bytes + b_bytes));
        __syncwarp(0x0000ffffu);                                  // the barrier is armed before any byte lands
        if (tp < krows) {
          const uint32_t sa = smem_u32(smem + stage * kStageDoubles), sb = sa + kGKC * LA * 8;
          bulk_g2s(sa + (uint32_t)(tp * LA) * 8u, Ak + (size_t)c * kGKC * g.lda, a_bytes, fullb);
          bulk_g2s(sb + (uint32_t)(tp * LB) * 8u, Bk + (size_t)c * kGKC * g.ldb, b_bytes, fullb);
        }
      }
      return;
    } else {
    // a thread keeps its columns for the whole kernel: one column m of the A tile (k rows tp / TM,
    // + 128 / TM, ...) and the columns tp, tp + 128, ... of the B tile; only k moves per chunk
    static_assert(128 % TM == 0 || TM % 128 == 0, "A tile width must divide or be a multiple of 128");
    constexpr int kAColsPerThread = TM > 128 ? TM / 128 : 1, kAKStep = TM > 128 ? 1 : 128 / TM;
    constexpr int kBColsPerThread = (TN + 127) / 128;
    size_t a_off[kAColsPerThread];
    bool a_ok[kAColsPerThread];
    const int a_k0 = TM > 128 ? 0 : tp / TM;
#pragma unroll
    for (int q = 0; q < kAColsPerThread; q++) {
      const int m = (TM > 128 ? tp + 128 * q : tp % TM), mg = m0 + m;
      a_ok[q] = mg < g.M;
      a_off[q] = mg;
      if (g.a_group > 0) {
        const int grp = mg / g.a_group;
        a_off[q] = (size_t)grp * g.a_gstride + (mg - grp * g.a_group);
      }
    }
    for (int c = 0; c < nchunks; c++) {
      const int stage = c % kGStages;
      mbar_wait(empty0 + 8 * stage, ((c / kGStages) & 1) ^ 1);
      const uint32_t sa = smem_u32(smem + stage * kStageDoubles), sb = sa + kGKC * LA * 8;
      const int k0 = c * kGKC;
#pragma unroll
      for (int q = 0; q < kAColsPerThread; q++) {
        const int m = (TM > 128 ? tp + 128 * q : tp % TM);
#pragma unroll
        for (int k = a_k0; k < kGKC; k += kAKStep) {
          const bool ok = a_ok[q] && (k0 + k < g.K);
          cp_async8(sa + (uint32_t)(k * LA + m) * 8u, A + (ok ? a_off[q] + (size_t)(k0 + k) * g.lda : 0), ok);
        }
      }
#pragma unroll
      for (int q = 0; q < kBColsPerThread; q++) {
        const int n = tp + 128 * q;
        if (n < TN) {
          const bool okn = n0 + n < g.N;
          const double* bp = B + (okn ? (size_t)(n0 + n) : 0);
#pragma unroll 4
          for (int k = 0; k < kGKC; k++) {
            const bool ok = okn && (k0 + k < g.K);
            cp_async8(sb + (uint32_t)(k * LB + n) * 8u, bp + (ok ? (size_t)(k0 + k) * g.ldb : 0), ok);
          }
        }
      }
      cp_async_mbar_arrive_noinc(full0 + 8 * stage);
    }
    return;
    }
  }

  // ===================== consumer warpgroups =====================
  reg_inc<kConsumerRegs>();
  const int r = l >> 2, j = l & 3;
  const int wm = w % WGM, wn = w / WGM;
  double acc[WTM][WTN][2];
#pragma unroll
  for (int t = 0; t < WTM; t++)
#pragma unroll
    for (int u = 0; u < WTN; u++) acc[t][u][0] = acc[t][u][1] = 0.0;
  const int nk4 = (g.K + 3) >> 2;
  for (int c = 0; c < nchunks; c++) {
    const int stage = c % kGStages;
    const int ksteps = min(4, nk4 - c * 4);
    mbar_wait(full0 + 8 * stage, (c / kGStages) & 1);
    const double* a_ptr = smem + stage * kStageDoubles + j * LA + wm * 8 * WTM + r;
    const double* b_ptr = smem + stage * kStageDoubles + kGKC * LA + j * LB + wn * 8 * WTN + r;
#pragma unroll
    for (int kk = 0; kk < 4; kk++) {
      if (kk < ksteps) {
        double a[WTM], b[WTN];
#pragma unroll
        for (int t = 0; t < WTM; t++) a[t] = a_ptr[4 * kk * LA + 8 * t];
#pragma unroll
        for (int u = 0; u < WTN; u++) b[u] = b_ptr[4 * kk * LB + 8 * u];
#pragma unroll
        for (int t = 0; t < WTM; t++)
#pragma unroll
          for (int u = 0; u < WTN; u++) dmma884(acc[t][u][0], acc[t][u][1], a[t], b[u]);
      }
    }
    __syncwarp();
    if (l == 0) mbar_arrive(empty0 + 8 * stage);
  }
  // epilogue: lane owns C[m][n], C[m][n+1], m = m0 + 8 (wm WTM + t) + r, n = n0 + 8 (wn WTN + u) + 2j
#pragma unroll
  for (int t = 0; t < WTM; t++) {
    const int m = m0 + 8 * (wm * WTM + t) + r;
    if (m >= g.M) continue;
#pragma unroll
    for (int u = 0; u < WTN; u++) {
      const int n = n0 + 8 * (wn * WTN + u) + 2 * j;
      if (g.c_group > 0) {
        double* p = C + (size_t)(m / g.c_group) * g.c_gstride + (size_t)n * g.c_nstride + m % g.c_group;
        if (n < g.N) p[0] = g.accumulate ? p[0] + acc[t][u][0] : acc[t][u][0];
        if (n + 1 < g.N) p[g.c_nstride] = g.accumulate ? p[g.c_nstride] + acc[t][u][1] : acc[t][u][1];
        continue;
      }
      double* p = C + (size_t)m * g.ldc + n;
      if (n < g.N) p[0] = g.accumulate ? p[0] + acc[t][u][0] : acc[t][u][0];
      if (n + 1 < g.N) p[1] = g.accumulate ? p[1] + acc[t][u][1] : acc[t][u][1];
    }
  }
}

__global__ void k_zero_ao(double* p, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = 0.0;
}

template <int WTM, int WTN, bool BULK, int WGM = 2>
static cudaError_t launch_gemm_tn_b(int device, const GemmTN& g, int batch, cudaStream_t st) {
  constexpr int TM = 8 * WTM * WGM, TN = 8 * WTN * (8 / WGM);
  constexpr size_t smem = (size_t)kGStages * kGKC * (TM + 4 + TN + 4) * sizeof(double);
  static std::atomic<unsigned long long> attr_done{0};
  cudaError_t e = ensure_dyn_smem(k_gemm_tn<WTM, WTN, BULK, WGM>, smem, device, attr_done);
  if (e != cudaSuccess) return e;
  if (g.M <= 0 || g.N <= 0 || batch <= 0) return cudaSuccess;
  dim3 grid(cdiv(g.M, TM), cdiv(g.N, TN), batch);
  k_gemm_tn<WTM, WTN, BULK, WGM><<<grid, kGThreads, smem, st>>>(g);
  return cudaSuccess;
}

// bulk copies need 16-byte aligned k rows of both operands for every tile and batch, and whole k4 steps
static bool gemm_tn_bulk_ok(const GemmTN& g) {
  auto even = [](long long v) { return (v & 1) == 0; };
  return g.a_group == 0 && ((uintptr_t)g.A & 15u) == 0 && ((uintptr_t)g.B & 15u) == 0 && even(g.lda) && even(g.ldb) &&
         even(g.sA) && even(g.sB) && even(g.M) && even(g.N) && (g.K & 3) == 0;
}

template <int WTM, int WTN, int WGM = 2>
static cudaError_t launch_gemm_tn(int device, const GemmTN& g, int batch, cudaStream_t st) {
  return gemm_tn_bulk_ok(g) ? launch_gemm_tn_b<WTM, WTN, true, WGM>(device, g, batch, st)
                            : launch_gemm_tn_b<WTM, WTN, false, WGM>(device, g, batch, st);
}

// CTA tile 64 x (32 WTN): the N tile is fitted to the problem (at most 352 columns per tile, the
// fewest tiles that cover N, then the narrowest WTN that does), so that e.g. N = 340 pays 352.
static cudaError_t gemm_tn(int device, const GemmTN& g, int batch, cudaStream_t st) {
  if (g.lower_only) return launch_gemm_tn<8, 4>(device, g, batch, st);     // square 128 x 128 tiles: half of them run
  const int n8 = cdiv(g.N > 0 ? g.N : 1, 8);
  const int ntn = cdiv(n8, 44), wtn = cdiv(n8, 4 * ntn);
  if (g.N > 32 && g.N <= 40 && g.M >= 128 * 148)   // 36 packed (a1 >= a2) pairs of 8 active orbitals: 128 x 40 tiles
    return launch_gemm_tn<2, 5, 8>(device, g, batch, st);
  if (wtn <= 2 && g.M >= 128 * 148) {       // narrow and tall (W of the active-first route): 128-row tiles
    return wtn == 1 ? launch_gemm_tn<8, 1>(device, g, batch, st) : launch_gemm_tn<8, 2>(device, g, batch, st);
  }
  switch (wtn) {
#define DFJK_GEMM_CASE(N) \
  case N: return launch_gemm_tn<4, N>(device, g, batch, st);
    DFJK_GEMM_CASE(1) DFJK_GEMM_CASE(2) DFJK_GEMM_CASE(3) DFJK_GEMM_CASE(4) DFJK_GEMM_CASE(5) DFJK_GEMM_CASE(6)
    DFJK_GEMM_CASE(7) DFJK_GEMM_CASE(8) DFJK_GEMM_CASE(9) DFJK_GEMM_CASE(10) DFJK_GEMM_CASE(11)
#undef DFJK_GEMM_CASE
    default: return cudaErrorInvalidValue;
  }
}

// C[m][n] = C[n][m] for n > m (n x n, row stride ldc): completes a product computed on its lower tiles
__global__ void k_mirror_lower(double* __restrict__ C, int n, long long ldc) {
  __shared__ double t[32][33];
  const int bi = blockIdx.x, bj = blockIdx.y;
  if (bj > bi) return;
  const int tx = threadIdx.x, ty = threadIdx.y;
  for (int r = ty; r < 32; r += 8) {
    const int m = bi * 32 + r, c = bj * 32 + tx;
    t[r][tx] = (m < n && c < n) ? C[(size_t)m * ldc + c] : 0.0;
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int row = bj * 32 + r, col = bi * 32 + tx;             // the mirrored tile (bj, bi): element (row, col) = lower (col, row)
    if (row < n && col < n && col > row) C[(size_t)row * ldc + col] = t[tx][r];
  }
}

// bpa[P][p][a] = bmo[P][p][a0 + a]  (pulled back by the caller) and
// baa[P][a1][a2] = bmo[P][a0 + a1][a0 + a2]  (the B operand of Eq. 20)
__global__ void k_ao2mo_gather(const double* __restrict__ bmo, int nb, int nmo, int a0, int nact,
                               double* __restrict__ bpa, double* __restrict__ baa) {
  const int P = blockIdx.y;
  const double* src = bmo + (size_t)P * nmo * nmo;
  const int npa = nmo * nact, naa = nact * nact;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < npa + naa; e += gridDim.x * blockDim.x) {
    if (e < npa) {
      const int p = e / nact, a = e - p * nact;
      bpa[(size_t)P * npa + e] = src[(size_t)p * nmo + a0 + a];
    } else {
      const int f = e - npa, a1 = f / nact, a2 = f - a1 * nact;
      baa[(size_t)P * naa + f] = src[(size_t)(a0 + a1) * nmo + a0 + a2];
    }
  }
}

// Route 1: Eq. 18-21 as printed, block after block.  Workspace: the X buffer of the handle holds,
// per aux row of the block, the half-transformed slice (nao x ldx), bmo (nmo x nmo) and baa (nact x nact).
static int launch_ao2mo_as_printed(dfjk_ctx* h, int nmo, int a0, int nact, const double* M, double* bpa_out,
                                   double* ppaa_out, double* papa_out, cudaStream_t st) {
  int launches = 0;
  const int nao = h->nao, naux = h->naux;
  const size_t n2 = (size_t)nmo * nmo, npa = (size_t)nmo * nact, naa = (size_t)nact * nact;
  SetInfo si;
  si.nset = 1; si.col0[0] = 0; si.nocc[0] = nmo; si.coff[0] = 0; si.ooff[0] = 0;
  si.col0[1] = si.nocc_pad = round_up(nmo, 8);
  prof_mark(h, DFJK_PHASE_PREP, st);
  launches += launch_prep_ct(h, si, M, nullptr, st);          // C' = M (no occupations)
  const int ldx = si.nocc_pad;
  const size_t row_doubles = (size_t)nao * ldx + n2 + naa;
  long long nblk = (long long)(h->X_doubles / row_doubles);
  if (h->nblk_forced > 0 && nblk > h->nblk_forced) nblk = h->nblk_forced;
  if (nblk > naux) nblk = naux;
  if (nblk > 32768) nblk = 32768;
  if (nmo > 0 && nblk > (1LL << 30) / nmo) nblk = (1LL << 30) / nmo;   // nb * nmo is an int in Eq. 19
  if (nblk < 1) return -2;                                    // workspace too small for one aux row
  double* Xb = h->X;
  double* bmo = Xb + (size_t)nblk * nao * ldx;
  double* baa = bmo + (size_t)nblk * n2;
  for (int p0 = 0; p0 < naux; p0 += (int)nblk) {
    const int nb = (int)(naux - p0 < nblk ? naux - p0 : nblk);
    prof_mark(h, DFJK_PHASE_HALF_TRANSFORM, st);
    if (launch_half_transform_rowmajor(h, si, p0, nb, Xb, ldx, st) != 0) return -1;      // Eq. 18
    launches++;
    prof_mark(h, DFJK_PHASE_SYRK, st);
    // Eq. 19 for the whole block as one GEMM: rows (P, p1) stacked along M, bmo[P][p1][p2] = C[(P p1)][p2]
    GemmTN g19{Xb, M, bmo, nb * nmo, nmo, nao, ldx, nmo, nmo, 0, 0, 0, 0, nmo, (long long)nao * ldx};
    if (gemm_tn(h->device, g19, 1, st) != cudaSuccess) return -1;
    launches++;
    if (nact > 0) {
      dim3 gg(cdiv((int)(npa + naa), 256) < 64 ? cdiv((int)(npa + naa), 256) : 64, nb);
      k_ao2mo_gather<<<gg, 256, 0, st>>>(bmo, nb, nmo, a0, nact, bpa_out + (size_t)p0 * npa, baa);
      launches++;
      if (ppaa_out) {
        GemmTN g20{bmo, baa, ppaa_out, (int)n2, (int)naa, nb, (long long)n2, (long long)naa, (long long)naa,
                   0, 0, 0, p0 > 0 ? 1 : 0};
        if (gemm_tn(h->device, g20, 1, st) != cudaSuccess) return -1;                                // Eq. 20
        launches++;
      }
    }
  }
  if (papa_out && nact > 0) {
    prof_mark(h, DFJK_PHASE_SYRK, st);
    GemmTN g21{bpa_out, bpa_out, papa_out, (int)npa, (int)npa, naux, (long long)npa, (long long)npa,
               (long long)npa, 0, 0, 0, 0};
    g21.lower_only = 1;                                                                              // (p1 a1|p2 a2) = (p2 a2|p1 a1)
    if (gemm_tn(h->device, g21, 1, st) != cudaSuccess) return -1;                                    // Eq. 21
    {
      const int nb32 = cdiv((int)npa, 32);
      dim3 gm(nb32, nb32), bm(32, 8);
      k_mirror_lower<<<gm, bm, 0, st>>>(papa_out, (int)npa, (long long)npa);
    }
    launches += 2;
  }
  return launches;
}

// Mact[e][a] = M[e][a0 + a], contiguous
__global__ void k_copy_cols(const double* __restrict__ M, int nao, int nmo, int a0, int nact, double* __restrict__ dst) {
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < nao * nact; e += gridDim.x * blockDim.x) {
    const int r = e / nact, a = e - r * nact;
    dst[e] = M[(size_t)r * nmo + a0 + a];
  }
}

// baat[P][tri(a1) + a2] = bpa[P][a0 + a1][a2], a1 >= a2: the active-active block of bmo^P is symmetric, so the
// W contraction only needs its nact (nact + 1) / 2 distinct columns (zero padded to ldt)
__global__ void k_pack_baa(const double* __restrict__ bpa, int naux, size_t npa, int a0, int nact, int ldt,
                           double* __restrict__ baat) {
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < (size_t)naux * ldt; e += (size_t)gridDim.x * blockDim.x) {
    const size_t P = e / ldt;
    const int t = (int)(e - P * ldt);
    int a1 = 0;
    while ((a1 + 1) * (a1 + 2) / 2 <= t) a1++;
    const int a2 = t - a1 * (a1 + 1) / 2;
    baat[e] = a1 < nact ? bpa[P * npa + (size_t)(a0 + a1) * nact + a2] : 0.0;
  }
}

// Wsq[e1][e2][t] = W[tri(max(e1,e2)) + min(e1,e2)][t], t < ldt (the packed active pairs a1 >= a2); W element (pair, t)
// sits at pair * pstride + t * tstride (either orientation of the W product)
__global__ void k_unpack_w(const double* __restrict__ W, int nao, int ldt, long long pstride, long long tstride,
                           double* __restrict__ Wsq) {
  const size_t n = (size_t)nao * nao * ldt;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
    const int t = (int)(e % ldt);
    const size_t ee = e / ldt;
    const int e1 = (int)(ee / nao), e2 = (int)(ee % nao);
    Wsq[e] = W[(e1 >= e2 ? tri(e1) + e2 : tri(e2) + e1) * pstride + t * tstride];
  }
}

// ppaa[p1][p2][a1][a2] = Pt[p1][p2][tri(max(a1,a2)) + min(a1,a2)]
__global__ void k_expand_ppaa(const double* __restrict__ Pt, size_t n2, int nact, int ldt, double* __restrict__ ppaa) {
  const int naa = nact * nact;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n2 * naa; e += (size_t)gridDim.x * blockDim.x) {
    const size_t pp = e / naa;
    const int a = (int)(e - pp * naa), a1 = a / nact, a2 = a - a1 * nact;
    ppaa[e] = Pt[pp * ldt + (a1 >= a2 ? a1 * (a1 + 1) / 2 + a2 : a2 * (a2 + 1) / 2 + a1)];
  }
}

// Route 2, "active first": the same bpa, ppaa, papa without ever forming bmo^P (nmo x nmo per aux
// row).  Eq. 18-19 are only evaluated for the active columns,
//      Z^P = b^P M_act (nao x nact),   bpa^P = M^T Z^P,
// and Eq. 20 is contracted over P in the AO basis first (a Coulomb-like build with the nact^2
// "densities" baa^P, Eq. 15's pattern), then transformed:
//      W[e1 e2][a1 a2] = sum_P b^P[e1][e2] bpa^P[a0+a1][a2]      (only the a1 >= a2 columns: baa^P is symmetric),
//      ppaa[p1][p2][a1 a2] = sum_{e1 e2} M[e1][p1] W[e1 e2][a1 a2] M[e2][p2]    (packed pairs a1 >= a2 throughout).
// Work 2 naux nao^2 nact + naux nao^2 nact^2 + small, against 2 naux nao nmo (nao + nmo) for the
// printed order: 5x less at nmo = 340, nact = 8; the printed order wins for large active spaces.
static int launch_ao2mo_active_first(dfjk_ctx* h, int nmo, int a0, int nact, const double* M, double* bpa_out,
                                     double* ppaa_out, double* papa_out, cudaStream_t st) {
  int launches = 0;
  const int nao = h->nao, naux = h->naux;
  const size_t npa = (size_t)nmo * nact;
  const int ldz = round_up(nact, 8);
  double* Mact = h->X;
  double* Z = h->X + round_up(nao * nact, 2);
  long long nbz = (long long)((h->X_doubles - round_up(nao * nact, 2)) / ((size_t)nao * ldz));
  if (h->nblk_forced > 0 && nbz > h->nblk_forced) nbz = h->nblk_forced;
  if (nbz > naux) nbz = naux;
  if (nbz > 32768) nbz = 32768;
  prof_mark(h, DFJK_PHASE_PREP, st);
  k_copy_cols<<<64, 256, 0, st>>>(M, nao, nmo, a0, nact, Mact);
  SetInfo si;
  si.nset = 1; si.col0[0] = 0; si.nocc[0] = nact; si.coff[0] = 0; si.ooff[0] = 0;
  si.col0[1] = si.nocc_pad = ldz;
  // at most 8 active columns: one pass over the packed triangle, every stored element used twice (symm.cu)
  // (9 to 16 columns were measured both as two passes of the thin kernel, 10.5 ms, and as two column groups on the
  // same fragments, 10.2 ms, against 9.8 ms tiled at nact = 10: the thin kernel is bound by its DMMA issue)
  const bool thin = symm_thin_ok(h, nact) && ldz == 8;
  launches += 1;
  if (!thin) launches += launch_prep_ct(h, si, Mact, nullptr, st);
  for (int p0 = 0; p0 < naux; p0 += (int)nbz) {
    const int nb = (int)(naux - p0 < nbz ? naux - p0 : nbz);
    prof_mark(h, DFJK_PHASE_HALF_TRANSFORM, st);
    if (thin) {
      if (launch_symm_thin(h, Mact, nact, nact, p0, nb, Z, ldz, st) != 0) return -1;       // Z^P = b^P M_act
    } else if (launch_half_transform_rowmajor(h, si, p0, nb, Z, ldz, st) != 0) {
      return -1;
    }
    prof_mark(h, DFJK_PHASE_SYRK, st);
    // bpa^P = M^T Z^P for the whole block as one GEMM with rows (P, a) and columns p:
    // C[(P a)][p] = sum_mu Z^P[mu][a] M[mu][p], stored transposed into bpa[P][p][a]
    GemmTN gb{Z, M, bpa_out + (size_t)p0 * npa, nb * nact, nmo, nao, ldz, nmo, 0, 0, 0, 0, 0,
              nact, (long long)nao * ldz, nact, (long long)npa, nact};
    if (gemm_tn(h->device, gb, 1, st) != cudaSuccess) return -1;
    launches += 2;
  }
  prof_mark(h, DFJK_PHASE_SYRK, st);
  if (ppaa_out) {
    const int ldt = round_up(nact * (nact + 1) / 2, 2);
    double* W = h->X;
    double* Wsq = W + h->npair * ldt;                        // [e1][e2][t]
    double* T = Wsq + (size_t)nao * nao * ldt;               // [p1][e2][t]
    double* baat = T + (size_t)nmo * nao * ldt;              // [P][t]
    double* Pt = baat + (size_t)naux * ldt;                  // [p1][p2][t]
    k_pack_baa<<<148, 256, 0, st>>>(bpa_out, naux, npa, a0, nact, ldt, baat);
    // W = sum_P b^P (x) baa^P.  With bulk-copyable operands the product runs transposed, Wt[t][pair] = baat^T B
    // (40..64 x 256 tiles, 20 to 32 accumulator tiles per warp); otherwise as W[pair][t] = B^T baat
    GemmTN gwt{baat, h->B, W, ldt, (int)h->npair, naux, (long long)ldt, (long long)h->npair, (long long)h->npair, 0, 0, 0, 0};
    const bool wt = ldt > 32 && ldt <= 64 && gemm_tn_bulk_ok(gwt);         // 8 to 11 active orbitals: 36 to 66 pairs
    if (wt) {
      cudaError_t e = cudaErrorInvalidValue;
      switch (cdiv(ldt, 8)) {
        case 5: e = launch_gemm_tn_b<5, 4, true, 1>(h->device, gwt, 1, st); break;
        case 6: e = launch_gemm_tn_b<6, 4, true, 1>(h->device, gwt, 1, st); break;
        case 7: e = launch_gemm_tn_b<7, 4, true, 1>(h->device, gwt, 1, st); break;
        case 8: e = launch_gemm_tn_b<8, 4, true, 1>(h->device, gwt, 1, st); break;
        default: break;
      }
      if (e != cudaSuccess) return -1;
    } else {
      GemmTN gw{h->B, baat, W, (int)h->npair, ldt, naux, (long long)h->npair, (long long)ldt, (long long)ldt, 0, 0, 0, 0};
      if (gemm_tn(h->device, gw, 1, st) != cudaSuccess) return -1;
    }
    k_unpack_w<<<1184, 256, 0, st>>>(W, nao, ldt, wt ? 1 : ldt, wt ? (long long)h->npair : 1LL, Wsq);
    // the two index transformations keep the packed active pairs: T[p1][e2 t] = M^T W, then ONE product over all
    // (p1, t) rows, Pt[(p1 t)][p2] = sum_e2 T[p1][e2][t] M[e2][p2], stored as Pt[p1][p2][t]
    GemmTN gt{M, Wsq, T, nmo, nao * ldt, nao, nmo, (long long)nao * ldt, (long long)nao * ldt, 0, 0, 0, 0};
    if (gemm_tn(h->device, gt, 1, st) != cudaSuccess) return -1;
    GemmTN gp{T, M, Pt, nmo * ldt, nmo, nao, ldt, nmo, 0, 0, 0, 0, 0,
              ldt, (long long)nao * ldt, ldt, (long long)nmo * ldt, ldt};
    if (gemm_tn(h->device, gp, 1, st) != cudaSuccess) return -1;
    k_expand_ppaa<<<1184, 256, 0, st>>>(Pt, (size_t)nmo * nmo, nact, ldt, ppaa_out);
    launches += 6;
  }
  if (papa_out) {
    GemmTN g21{bpa_out, bpa_out, papa_out, (int)npa, (int)npa, naux, (long long)npa, (long long)npa,
               (long long)npa, 0, 0, 0, 0};
    g21.lower_only = 1;                                                                               // (p1 a1|p2 a2) = (p2 a2|p1 a1)
    if (gemm_tn(h->device, g21, 1, st) != cudaSuccess) return -1;                                     // Eq. 21
    {
      const int nb32 = cdiv((int)npa, 32);
      dim3 gm(nb32, nb32), bm(32, 8);
      k_mirror_lower<<<gm, bm, 0, st>>>(papa_out, (int)npa, (long long)npa);
    }
    launches += 2;
  }
  return launches;
}

// Picks the cheaper route (h->ao2mo_route forces one: 1 as printed, 2 active first).
int launch_ao2mo(dfjk_ctx* h, int nmo, int a0, int nact, const double* M, double* bpa_out, double* ppaa_out,
                 double* papa_out, cudaStream_t st) {
  int launches = 0;
  const int nao = h->nao, naux = h->naux;
  const size_t n2 = (size_t)nmo * nmo, naa = (size_t)nact * nact;
  if (naux == 0 || nmo == 0 || nact == 0) {
    if (ppaa_out && n2 * naa) { k_zero_ao<<<148, 256, 0, st>>>(ppaa_out, n2 * naa); launches++; }
    if (papa_out && n2 * naa) { k_zero_ao<<<148, 256, 0, st>>>(papa_out, n2 * naa); launches++; }
    if (naux == 0 || nmo == 0) return launches;
  }
  const double dn = nao, dm = nmo, da = nact;
  const double cost_printed = 2.0 * dn * dm * (dn + dm) + 2.0 * dm * dm * da * da;          // per aux row
  const double cost_active = 2.0 * dn * dn * round_up(nact, 8) + 2.0 * dn * dm * 32.0 + dn * dn * da * (da + 1.0) * 0.5 +
                             2.0 * dn * dm * da * da * (dn + dm) / (naux > 0 ? naux : 1);
  const size_t ldt_ = (size_t)round_up(nact * (nact + 1) / 2, 2);
  const size_t need2 = (h->npair + (size_t)nao * nao + (size_t)nmo * nao + (size_t)naux + (size_t)nmo * nmo) * ldt_;  // W, Wsq, T, baat, Pt
  const size_t need1 = (size_t)round_up(nao * nact, 2) + (size_t)nao * round_up(nact, 8);   // Mact + one row of Z
  const bool fits = nact > 0 && need2 <= h->X_doubles && need1 <= h->X_doubles && (double)nao * ldt_ < 2e9 && (double)nmo * ldt_ < 2e9 &&
                    round_up(nact, 8) <= h->nocc_pad_cap;
  bool active = fits && cost_active < cost_printed;
  if (h->ao2mo_route == 1) active = false;
  if (h->ao2mo_route == 2 && fits) active = true;
  const int n = active ? launch_ao2mo_active_first(h, nmo, a0, nact, M, bpa_out, ppaa_out, papa_out, st)
                       : launch_ao2mo_as_printed(h, nmo, a0, nact, M, bpa_out, ppaa_out, papa_out, st);
  h->plan_ao2mo_route = active ? 2 : 1;
  prof_mark(h, -1, st);
  return n < 0 ? n : n + launches;
}

}  // namespace dfjk
