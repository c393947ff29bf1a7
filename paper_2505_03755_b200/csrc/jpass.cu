// Steps a2-a4, the Coulomb build (Eq. 14-15), HBM-bandwidth bound:
//   pass 1  rho[s][P]  = sum_pair B[P][pair] Dw_s[pair]        (one stream over packed B)
//   pass 2  Jp_s[pair] = sum_P rho[s][P] B[P][pair]            (second stream over packed B)
//   epilogue: fixed-order sum of the P-split partials and unpack to the full symmetric square.
// Pass 1 is a bulk-copy (TMA engine) pipeline when npair is even: k_j1_tma (DFMA) for one or two sets,
// k_j1_mma (DMMA, the weighted densities fetched once per 64 aux rows) for three to eight; for odd
// npair, where packed rows are only 8-byte aligned, k_j1 streams with plain loads: a (64 aux rows) x
// (<=8 sets) x (pairs) contraction per warp on DMMA.8x8x4, whose row x set accumulators fall out of
// the MMA fragments (no per-row shuffle reduction; one Dw fragment serves 8 row groups).
#include "common.cuh"
#include "ctx.h"
#include "pipeline.cuh"

namespace dfjk {

// two adjacent pairs of a packed row that is only 8-byte aligned (odd npair)
__device__ __forceinline__ double2 load_pair(const double* p) {
  double2 v;
  v.x = ldg_stream1(p);
  v.y = ldg_stream1(p + 1);
  return v;
}

// grid.x = pair chunk (kJ1Chunk pairs), grid.y = block of 64 aux rows; 8 warps, warp w streams
// pairs [chunk*kJ1Chunk + w*kJ1SubChunk, +kJ1SubChunk) of its 64 rows.
__global__ void __launch_bounds__(kJ1Warps * 32, 2)
k_j1(const double* __restrict__ B, size_t npair, int naux, const double* __restrict__ Dw, int nsetg,
     double* __restrict__ part, int naux_pad) {
  __shared__ double red[kJ1Warps][kJ1Rows][8];
  const int w = threadIdx.x >> 5, l = threadIdx.x & 31, r = l >> 2, j = l & 3;
  const int p0 = blockIdx.y * kJ1Rows;
  const size_t kbeg = (size_t)blockIdx.x * kJ1Chunk + (size_t)w * kJ1SubChunk;
  size_t kend = kbeg + kJ1SubChunk;
  if (kend > npair) kend = npair;

  const double* rowp[8];
#pragma unroll
  for (int g = 0; g < 8; g++) {
    int row = p0 + 8 * g + r;
    if (row > naux - 1) row = naux - 1;  // clamped rows land in accumulator rows nobody reads
    rowp[g] = B + (size_t)row * npair + 2 * j;
  }
  const bool dw_on = r < nsetg;          // lane's column of the MMA B operand = set index r
  const double* dwp = Dw + (size_t)(dw_on ? r : 0) * npair + 2 * j;

  double acc[8][2];
#pragma unroll
  for (int g = 0; g < 8; g++) acc[g][0] = acc[g][1] = 0.0;

  size_t kk = kbeg;
  for (; kk + 16 <= kend; kk += 16) {
    double2 b[2][8], d[2];
#pragma unroll
    for (int u = 0; u < 2; u++)
#pragma unroll
      for (int g = 0; g < 8; g++) b[u][g] = load_pair(rowp[g] + kk + 8 * u);
#pragma unroll
    for (int u = 0; u < 2; u++) {
      d[u] = make_double2(0.0, 0.0);
      if (dw_on) {
        d[u].x = dwp[kk + 8 * u];
        d[u].y = dwp[kk + 8 * u + 1];
      }
    }
#pragma unroll
    for (int u = 0; u < 2; u++)
#pragma unroll
      for (int g = 0; g < 8; g++) {
        dmma884(acc[g][0], acc[g][1], b[u][g].x, d[u].x);
        dmma884(acc[g][0], acc[g][1], b[u][g].y, d[u].y);
      }
  }
  for (; kk < kend; kk += 8) {  // guarded tail steps
    const bool ok0 = kk + 2 * j < kend, ok1 = kk + 2 * j + 1 < kend;
    double2 d = make_double2(0.0, 0.0);
    if (dw_on && ok0) d.x = dwp[kk];
    if (dw_on && ok1) d.y = dwp[kk + 1];
#pragma unroll
    for (int g = 0; g < 8; g++) {
      double2 b = make_double2(0.0, 0.0);
      if (ok0) b.x = ldg_stream1(rowp[g] + kk);
      if (ok1) b.y = ldg_stream1(rowp[g] + kk + 1);
      dmma884(acc[g][0], acc[g][1], b.x, d.x);
      dmma884(acc[g][0], acc[g][1], b.y, d.y);
    }
  }
  // fixed-order combine of the 8 warps, one partial per CTA
#pragma unroll
  for (int g = 0; g < 8; g++) {
    red[w][8 * g + r][2 * j] = acc[g][0];
    red[w][8 * g + r][2 * j + 1] = acc[g][1];
  }
  __syncthreads();
  for (int e = threadIdx.x; e < kJ1Rows * 8; e += kJ1Warps * 32) {
    const int s = e / kJ1Rows, row = e % kJ1Rows;
    double t = 0.0;
#pragma unroll
    for (int ww = 0; ww < kJ1Warps; ww++) t += red[ww][row][s];
    part[((size_t)blockIdx.x * 8 + s) * naux_pad + p0 + row] = t;
  }
}

// Pass 1 as a bulk-copy (TMA engine) pipeline, for npair even (every packed row and every Dw row
// then starts 16-byte aligned).  CTA = 64 aux rows x kJ1Chunk pairs, walked as 8 row groups of 8
// rows x 32 chunks of 512 pairs; a stage holds the chunk of the 8 rows (32 KB) and of the NS
// weighted densities (4 KB each), filled by one elected producer thread with 8 + NS bulk copies,
// so 100-190 KB per SM are in flight whatever the consumers do.  Consumer warp w owns pairs
// [64 w, 64 w + 64) of every chunk, a lane two adjacent pairs (one conflict-free LDS.128 per row):
// 8 x NS accumulators per lane, plain DFMA (the stream needs 3 DFMA/clk/SM per set), reduced by
// shuffles and a fixed-order sum over the 8 warps once per row group.
constexpr int kJ1tSC = 512;                       // pairs per stage
constexpr int kJ1tThreads = 288;                  // 8 consumer warps + 1 producer warp
__host__ __device__ constexpr int j1t_stages(int ns) { return ns <= 1 ? 6 : 5; }

template <int NS>
__global__ void __launch_bounds__(kJ1tThreads, 1)
k_j1_tma(const double* __restrict__ B, size_t npair, int naux, const double* __restrict__ Dw,
         double* __restrict__ part, int naux_pad, int rows_cta) {
  constexpr int STAGES = j1t_stages(NS);
  constexpr int kStageDoubles = (8 + NS) * kJ1tSC;
  extern __shared__ __align__(128) double smem[];
  __shared__ __align__(8) unsigned long long bars[2 * STAGES];
  __shared__ double red[8][8][NS];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[STAGES]);
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
  const int p0 = blockIdx.y * rows_cta;          // rows_cta = 8, 16, 32 or 64 aux rows per CTA (launch_j_passes)
  const size_t kbeg = (size_t)blockIdx.x * kJ1Chunk;
  const size_t kend = kbeg + kJ1Chunk < npair ? kbeg + kJ1Chunk : npair;
  const int nchunk = (int)((kend - kbeg + kJ1tSC - 1) / kJ1tSC);
  const int ngroups = min(rows_cta >> 3, (naux - p0 + 7) / 8);
  const int nstage = ngroups * nchunk;
  if (tid == 0) {
    for (int s = 0; s < STAGES; s++) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 8);
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (w == 8) {
    if (l == 0) {
      const uint32_t s_u32 = smem_u32(smem);
      int rg = 0, c = 0;
      for (int it = 0; it < nstage; it++) {
        const int stage = it % STAGES;
        const uint32_t fullb = full0 + 8 * stage;
        mbar_wait(empty0 + 8 * stage, ((it / STAGES) & 1) ^ 1);
        const size_t k0 = kbeg + (size_t)c * kJ1tSC;
        const uint32_t bytes = (uint32_t)((kend - k0 < (size_t)kJ1tSC ? kend - k0 : (size_t)kJ1tSC) * 8);
        const int nrows = min(8, naux - (p0 + 8 * rg));
        mbar_arrive_expect_tx(fullb, bytes * (uint32_t)(nrows + NS));
        const uint32_t dst = s_u32 + (uint32_t)(stage * kStageDoubles) * 8u;
        for (int g = 0; g < nrows; g++)
          bulk_g2s(dst + (uint32_t)(g * kJ1tSC) * 8u, B + (size_t)(p0 + 8 * rg + g) * npair + k0, bytes, fullb);
        for (int s = 0; s < NS; s++)
          bulk_g2s(dst + (uint32_t)((8 + s) * kJ1tSC) * 8u, Dw + (size_t)s * npair + k0, bytes, fullb);
        if (++c == nchunk) { c = 0; rg++; }
      }
    }
    return;
  }

  double acc[8][NS];
  int it = 0;
  for (int rg = 0; rg < ngroups; rg++) {
#pragma unroll
    for (int g = 0; g < 8; g++)
#pragma unroll
      for (int s = 0; s < NS; s++) acc[g][s] = 0.0;
    const int nrows = min(8, naux - (p0 + 8 * rg));
    for (int c = 0; c < nchunk; c++, it++) {
      const int stage = it % STAGES;
      const size_t k0 = kbeg + (size_t)c * kJ1tSC;
      const int nvalid = (int)(kend - k0 < (size_t)kJ1tSC ? kend - k0 : (size_t)kJ1tSC);
      mbar_wait(full0 + 8 * stage, (it / STAGES) & 1);
      const double* sp = smem + stage * kStageDoubles + w * 64 + 2 * l;
      if (w * 64 + 2 * l < nvalid) {          // nvalid is even: a lane's two pairs are both in or both out
        double2 d[NS];
#pragma unroll
        for (int s = 0; s < NS; s++) d[s] = *reinterpret_cast<const double2*>(sp + (8 + s) * kJ1tSC);
#pragma unroll
        for (int g = 0; g < 8; g++) {
          if (g < nrows) {
            const double2 b = *reinterpret_cast<const double2*>(sp + g * kJ1tSC);
#pragma unroll
            for (int s = 0; s < NS; s++) acc[g][s] = fma(b.y, d[s].y, fma(b.x, d[s].x, acc[g][s]));
          }
        }
      }
      __syncwarp();
      if (l == 0) mbar_arrive(empty0 + 8 * stage);
    }
    // row group done: lanes -> warp (xor shuffles), warps -> CTA (fixed order)
#pragma unroll
    for (int g = 0; g < 8; g++)
#pragma unroll
      for (int s = 0; s < NS; s++) {
        double v = acc[g][s];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (l == 0) red[w][g][s] = v;
      }
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (tid < 8 * NS) {
      const int g = tid / NS, s = tid % NS;
      double t = 0.0;
#pragma unroll
      for (int ww = 0; ww < 8; ww++) t += red[ww][g][s];
      part[((size_t)blockIdx.x * 8 + s) * naux_pad + p0 + 8 * rg + g] = t;
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");
  }
}

// Pass 1 for three and more sets, DMMA formulation of the same bulk-copy pipeline.  The DFMA kernel above
// re-reads the NS weighted densities from L2 once per 8 aux rows (NS * 4 KB per 32 KB of B: 1.75x the HBM stream
// at NS = 6, which then sits at the L2-to-SM rate) because its 8 x NS accumulators per lane only cover one row
// group.  Here rho[row][set] is a GEMM over the pairs on the FP64 tensor pipe: one DMMA.8x8x4 takes 8 rows x 4
// pairs x 8 sets, its accumulator tile is 2 registers per lane, so a warp keeps the tiles of all 8 row groups
// of the CTA (64 aux rows) and the loop runs chunk-outer: the Dw chunk is fetched ONCE per 64 rows and its 16
// B fragments stay in registers while the 8 row groups stream through the ring.  Rows land with a stride of
// 516 doubles (4 mod 16): the fragment reads are bank-conflict free.
constexpr int kJ1mLd = kJ1tSC + 4;                 // 516
constexpr int kJ1mStages = 4;
constexpr int kJ1mStageDoubles = 8 * kJ1mLd;       // 8 rows of one chunk
constexpr int kJ1mDwDoubles = 8 * kJ1mLd;          // up to 8 sets of one chunk

__global__ void __launch_bounds__(kJ1tThreads, 1)
k_j1_mma(const double* __restrict__ B, size_t npair, int naux, const double* __restrict__ Dw, int ns,
         double* __restrict__ part, int naux_pad) {
  extern __shared__ __align__(128) double smem[];
  double* ring = smem;                                          // kJ1mStages x 8 rows
  double* dws = smem + kJ1mStages * kJ1mStageDoubles;           // 2 x ns rows
  __shared__ __align__(8) unsigned long long bars[2 * kJ1mStages + 4];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kJ1mStages]);
  const uint32_t dfull0 = smem_u32(&bars[2 * kJ1mStages]), dempty0 = smem_u32(&bars[2 * kJ1mStages + 2]);
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
  const int p0 = blockIdx.y * kJ1Rows;
  const size_t kbeg = (size_t)blockIdx.x * kJ1Chunk;
  const size_t kend = kbeg + kJ1Chunk < npair ? kbeg + kJ1Chunk : npair;
  const int nchunk = (int)((kend - kbeg + kJ1tSC - 1) / kJ1tSC);
  const int ngroups = min(8, (naux - p0 + 7) / 8);
  for (int e = tid; e < kJ1mStages * kJ1mStageDoubles + 2 * kJ1mDwDoubles; e += kJ1tThreads) smem[e] = 0.0;   // stale slots stay finite
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  if (tid == 0) {
    for (int s = 0; s < kJ1mStages; s++) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 8);
    }
    for (int s = 0; s < 2; s++) {
      mbar_init(dfull0 + 8 * s, 1);
      mbar_init(dempty0 + 8 * s, 8);
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (w == 8) {
    if (l == 0) {
      const uint32_t ring_u32 = smem_u32(ring), dws_u32 = smem_u32(dws);
      int it = 0;
      for (int c = 0; c < nchunk; c++) {
        const size_t k0 = kbeg + (size_t)c * kJ1tSC;
        const uint32_t bytes = (uint32_t)((kend - k0 < (size_t)kJ1tSC ? kend - k0 : (size_t)kJ1tSC) * 8);
        const uint32_t dfull = dfull0 + 8 * (c & 1);
        mbar_wait(dempty0 + 8 * (c & 1), ((c >> 1) & 1) ^ 1);
        mbar_arrive_expect_tx(dfull, bytes * (uint32_t)ns);
        for (int s = 0; s < ns; s++)
          bulk_g2s(dws_u32 + (uint32_t)((c & 1) * kJ1mDwDoubles + s * kJ1mLd) * 8u, Dw + (size_t)s * npair + k0, bytes, dfull);
        for (int rg = 0; rg < ngroups; rg++, it++) {
          const int stage = it % kJ1mStages;
          const uint32_t fullb = full0 + 8 * stage;
          mbar_wait(empty0 + 8 * stage, ((it / kJ1mStages) & 1) ^ 1);
          const int nrows = min(8, naux - (p0 + 8 * rg));
          mbar_arrive_expect_tx(fullb, bytes * (uint32_t)nrows);
          for (int g = 0; g < nrows; g++)
            bulk_g2s(ring_u32 + (uint32_t)(stage * kJ1mStageDoubles + g * kJ1mLd) * 8u, B + (size_t)(p0 + 8 * rg + g) * npair + k0,
                     bytes, fullb);
        }
      }
    }
    return;
  }

  const int r = l >> 2, j = l & 3;
  double acc[8][2];
#pragma unroll
  for (int rg = 0; rg < 8; rg++) acc[rg][0] = acc[rg][1] = 0.0;
  int it = 0;
  for (int c = 0; c < nchunk; c++) {
    const size_t k0 = kbeg + (size_t)c * kJ1tSC;
    const int nvalid = (int)(kend - k0 < (size_t)kJ1tSC ? kend - k0 : (size_t)kJ1tSC);
    // B fragments of this chunk: Dw[set r][pair 64 w + 4 i + j], zero for sets past ns and pairs past the end
    double bf[16];
    mbar_wait(dfull0 + 8 * (c & 1), (c >> 1) & 1);
    const double* dp = dws + (c & 1) * kJ1mDwDoubles + r * kJ1mLd + 64 * w + j;
#pragma unroll
    for (int i = 0; i < 16; i++) bf[i] = (r < ns && 64 * w + 4 * i + j < nvalid) ? dp[4 * i] : 0.0;
    __syncwarp();
    if (l == 0) mbar_arrive(dempty0 + 8 * (c & 1));
#pragma unroll
    for (int rg = 0; rg < 8; rg++) {
      if (rg < ngroups) {
        const int stage = it % kJ1mStages;
        mbar_wait(full0 + 8 * stage, (it / kJ1mStages) & 1);
        const double* ap = ring + stage * kJ1mStageDoubles + r * kJ1mLd + 64 * w + j;
        double a[16];
#pragma unroll
        for (int i = 0; i < 16; i++) a[i] = ap[4 * i];
#pragma unroll
        for (int i = 0; i < 16; i++) dmma884(acc[rg][0], acc[rg][1], a[i], bf[i]);
        __syncwarp();
        if (l == 0) mbar_arrive(empty0 + 8 * stage);
        it++;
      }
    }
  }
  // warps -> CTA in warp order: lane (r, j) of warp w holds rho[row 8 rg + r][sets 2j, 2j + 1] over its pairs
  asm volatile("bar.sync 1, 256;" ::: "memory");            // every stage has been consumed: the ring is free
  double* red = ring;                                       // [8 warps][64 rows][8 sets]
#pragma unroll
  for (int rg = 0; rg < 8; rg++)
    *reinterpret_cast<double2*>(red + (w * 64 + 8 * rg + r) * 8 + 2 * j) = make_double2(acc[rg][0], acc[rg][1]);
  asm volatile("bar.sync 1, 256;" ::: "memory");
  for (int e = tid; e < kJ1Rows * 8; e += 256) {
    const int s = e / kJ1Rows, row = e % kJ1Rows;
    double t = 0.0;
#pragma unroll
    for (int ww = 0; ww < 8; ww++) t += red[(ww * 64 + row) * 8 + s];
    if (s < ns) part[((size_t)blockIdx.x * 8 + s) * naux_pad + p0 + row] = t;
  }
}

static cudaError_t launch_j1_mma(int device, dim3 grid, cudaStream_t st, const double* B, size_t npair, int naux,
                                 const double* Dw, int ns, double* part, int naux_pad) {
  constexpr size_t smem = (size_t)(kJ1mStages * kJ1mStageDoubles + 2 * kJ1mDwDoubles) * sizeof(double);
  static std::atomic<unsigned long long> attr_done{0};
  cudaError_t e = ensure_dyn_smem(k_j1_mma, smem, device, attr_done);
  if (e != cudaSuccess) return e;
  k_j1_mma<<<grid, kJ1tThreads, smem, st>>>(B, npair, naux, Dw, ns, part, naux_pad);
  return cudaSuccess;
}

template <int NS>
static cudaError_t launch_j1_tma(int device, dim3 grid, cudaStream_t st, const double* B, size_t npair, int naux,
                                 const double* Dw, double* part, int naux_pad, int rows_cta) {
  constexpr size_t smem = (size_t)j1t_stages(NS) * (8 + NS) * kJ1tSC * sizeof(double);
  static std::atomic<unsigned long long> attr_done{0};
  cudaError_t e = ensure_dyn_smem(k_j1_tma<NS>, smem, device, attr_done);
  if (e != cudaSuccess) return e;
  k_j1_tma<NS><<<grid, kJ1tThreads, smem, st>>>(B, npair, naux, Dw, part, naux_pad, rows_cta);
  return cudaSuccess;
}

static cudaError_t dispatch_j1_tma(int device, int ns, dim3 grid, cudaStream_t st, const double* B, size_t npair,
                                   int naux, const double* Dw, double* part, int naux_pad, int rows_cta) {
  switch (ns) {
#define DFJK_J1T_CASE(N) \
  case N: return launch_j1_tma<N>(device, grid, st, B, npair, naux, Dw, part, naux_pad, rows_cta);
    DFJK_J1T_CASE(1) DFJK_J1T_CASE(2)          // three and more sets take k_j1_mma
#undef DFJK_J1T_CASE
    default: return cudaErrorInvalidValue;
  }
}

// rho[s][P] = sum over chunks in ascending order
__global__ void k_j1_reduce(const double* __restrict__ part, int nchunks, int naux_pad, int naux, int nsetg,
                            double* __restrict__ rho) {
  const int P = blockIdx.x * blockDim.x + threadIdx.x, s = blockIdx.y;
  if (P >= naux || s >= nsetg) return;
  double t = 0.0;
  for (int c = 0; c < nchunks; c++) t += part[((size_t)c * 8 + s) * naux_pad + P];
  rho[(size_t)s * naux + P] = t;
}

// Pass 2: a thread owns two adjacent pairs and NS accumulators each; rows stream 8 at a time.
template <int NS, bool VEC>
__global__ void __launch_bounds__(kJ2Threads)
k_j2(const double* __restrict__ B, size_t npair, int naux, const double* __restrict__ rho,
     double* __restrict__ part, size_t split_stride, int rows_per_split) {
  __shared__ __align__(16) double rs[NS][128];
  const size_t col = ((size_t)blockIdx.x * kJ2Threads + threadIdx.x) * 2;
  const bool ok0 = col < npair, ok1 = col + 1 < npair;
  const int p_beg = blockIdx.y * rows_per_split;
  int p_end = p_beg + rows_per_split;
  if (p_end > naux) p_end = naux;
  double acc[NS][2];
#pragma unroll
  for (int s = 0; s < NS; s++) acc[s][0] = acc[s][1] = 0.0;

  for (int pt = p_beg; pt < p_end; pt += 128) {
    const int n = min(128, p_end - pt);
    for (int e = threadIdx.x; e < NS * 128; e += kJ2Threads) {
      const int s = e >> 7, q = e & 127;
      rs[s][q] = q < n ? rho[(size_t)s * naux + pt + q] : 0.0;
    }
    __syncthreads();
    if (ok0) {
      const double* bp = B + (size_t)pt * npair + col;
      int q0 = 0;
      for (; q0 + 8 <= n; q0 += 8) {
        double2 b[8];
#pragma unroll
        for (int u = 0; u < 8; u++) {
          const double* p = bp + (size_t)(q0 + u) * npair;
          if (VEC) b[u] = ldg_stream2(p);
          else { b[u].x = ldg_stream1(p); b[u].y = ok1 ? ldg_stream1(p + 1) : 0.0; }
        }
#pragma unroll
        for (int s = 0; s < NS; s++)
#pragma unroll
          for (int u = 0; u < 8; u += 2) {
            const double2 rr = *reinterpret_cast<const double2*>(&rs[s][q0 + u]);
            acc[s][0] = fma(rr.x, b[u].x, acc[s][0]);
            acc[s][1] = fma(rr.x, b[u].y, acc[s][1]);
            acc[s][0] = fma(rr.y, b[u + 1].x, acc[s][0]);
            acc[s][1] = fma(rr.y, b[u + 1].y, acc[s][1]);
          }
      }
      for (; q0 < n; q0++) {
        const double* p = bp + (size_t)q0 * npair;
        const double bx = ldg_stream1(p), by = ok1 ? ldg_stream1(p + 1) : 0.0;
#pragma unroll
        for (int s = 0; s < NS; s++) {
          acc[s][0] = fma(rs[s][q0], bx, acc[s][0]);
          acc[s][1] = fma(rs[s][q0], by, acc[s][1]);
        }
      }
    }
    __syncthreads();
  }
  if (ok0) {
    double* out = part + (size_t)blockIdx.y * split_stride + col;
#pragma unroll
    for (int s = 0; s < NS; s++) {
      out[(size_t)s * npair] = acc[s][0];
      if (ok1) out[(size_t)s * npair + 1] = acc[s][1];
    }
  }
}

// Pass 2 on the FP64 tensor pipe (16-byte aligned packed rows; k_j2 serves the rest): Jp[set][pair] = sum_P rho[set][P] B[P][pair] is a GEMM over the
// aux rows, one DMMA.8x8x4 takes 8 sets x 4 aux rows x 8 pairs.  CTA = one chunk of 512 pairs x one split of
// the aux rows; a stage of the bulk-copy ring holds 8 aux rows of the chunk (row stride 516 doubles: conflict-
// free fragments); warp w owns pairs [64 w, 64 w + 64) as 8 accumulator tiles (16 registers) for the whole
// split.  k_j2 (DFMA, 2 NS FMAs per loaded pair) falls from 7.2 to 4.9 TB/s between one and eight sets; this
// kernel does the same 16 LDS + 16 DMMA per stage and warp whatever the number of sets.
constexpr int kJ2mStages = 5;

__global__ void __launch_bounds__(kJ1tThreads, 1)
k_j2_mma(const double* __restrict__ B, size_t npair, int naux, const double* __restrict__ rho, int ns,
         double* __restrict__ part, size_t split_stride, int rows_per_split) {
  extern __shared__ __align__(128) double smem[];
  __shared__ __align__(8) unsigned long long bars[2 * kJ2mStages];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kJ2mStages]);
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
  const size_t k0 = (size_t)blockIdx.x * kJ1tSC;
  const int nvalid = (int)(npair - k0 < (size_t)kJ1tSC ? npair - k0 : (size_t)kJ1tSC);
  const int p_beg = blockIdx.y * rows_per_split;
  const int p_end = min(naux, p_beg + rows_per_split);
  const int nstage = p_end > p_beg ? (p_end - p_beg + 7) / 8 : 0;
  for (int e = tid; e < kJ2mStages * kJ1mStageDoubles; e += kJ1tThreads) smem[e] = 0.0;      // stale slots stay finite
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  if (tid == 0) {
    for (int s = 0; s < kJ2mStages; s++) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 8);
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (w == 8) {
    if (l == 0) {
      const uint32_t ring_u32 = smem_u32(smem);
      const uint32_t bytes = (uint32_t)nvalid * 8u;
      for (int it = 0; it < nstage; it++) {
        const int stage = it % kJ2mStages;
        const uint32_t fullb = full0 + 8 * stage;
        mbar_wait(empty0 + 8 * stage, ((it / kJ2mStages) & 1) ^ 1);
        const int nrows = min(8, p_end - (p_beg + 8 * it));
        mbar_arrive_expect_tx(fullb, bytes * (uint32_t)nrows);
        for (int g = 0; g < nrows; g++)
          bulk_g2s(ring_u32 + (uint32_t)(stage * kJ1mStageDoubles + g * kJ1mLd) * 8u, B + (size_t)(p_beg + 8 * it + g) * npair + k0,
                   bytes, fullb);
      }
    }
    return;
  }

  const int r = l >> 2, j = l & 3;
  double acc[8][2];
#pragma unroll
  for (int t = 0; t < 8; t++) acc[t][0] = acc[t][1] = 0.0;
  const double* rp = rho + (size_t)(r < ns ? r : 0) * naux;
  for (int it = 0; it < nstage; it++) {
    const int stage = it % kJ2mStages;
    // A fragments: rho[set r][P], P = p_beg + 8 it + 4 h + j (zero for sets past ns and rows past the split)
    const int P0 = p_beg + 8 * it + j;
    const double a0 = (r < ns && P0 < p_end) ? __ldg(rp + P0) : 0.0;
    const double a1 = (r < ns && P0 + 4 < p_end) ? __ldg(rp + P0 + 4) : 0.0;
    mbar_wait(full0 + 8 * stage, (it / kJ2mStages) & 1);
    const double* bp = smem + stage * kJ1mStageDoubles + j * kJ1mLd + 64 * w + r;
    double b0[8], b1[8];
#pragma unroll
    for (int t = 0; t < 8; t++) { b0[t] = bp[8 * t]; b1[t] = bp[4 * kJ1mLd + 8 * t]; }
#pragma unroll
    for (int t = 0; t < 8; t++) dmma884(acc[t][0], acc[t][1], a0, b0[t]);
#pragma unroll
    for (int t = 0; t < 8; t++) dmma884(acc[t][0], acc[t][1], a1, b1[t]);
    __syncwarp();
    if (l == 0) mbar_arrive(empty0 + 8 * stage);
  }
  // lane (r, j) holds Jp[set r][pairs 64 w + 8 t + 2 j, + 1]
  if (r < ns) {
    double* out = part + (size_t)blockIdx.y * split_stride + (size_t)r * npair + k0 + 64 * w + 2 * j;
#pragma unroll
    for (int t = 0; t < 8; t++)
      if (64 * w + 8 * t + 2 * j < nvalid) *reinterpret_cast<double2*>(out + 8 * t) = make_double2(acc[t][0], acc[t][1]);
  }
}

static cudaError_t launch_j2_mma(int device, dim3 grid, cudaStream_t st, const double* B, size_t npair, int naux,
                                 const double* rho, int ns, double* part, size_t split_stride, int rows_per_split) {
  constexpr size_t smem = (size_t)kJ2mStages * kJ1mStageDoubles * sizeof(double);
  static std::atomic<unsigned long long> attr_done{0};
  cudaError_t e = ensure_dyn_smem(k_j2_mma, smem, device, attr_done);
  if (e != cudaSuccess) return e;
  k_j2_mma<<<grid, kJ1tThreads, smem, st>>>(B, npair, naux, rho, ns, part, split_stride, rows_per_split);
  return cudaSuccess;
}

// Step a4: J_s[mu][nu] = J_s[nu][mu] = sum_g part[g][s][tri(mu)+nu] (g ascending), 32x32 tiles,
// the mirrored tile goes through shared memory so both global writes are row-contiguous.
__global__ void __launch_bounds__(256)
k_j_epilogue(const double* __restrict__ part, int nsplit, size_t split_stride, size_t npair, int nao,
             double* __restrict__ J) {
  const int bi = blockIdx.x, bj = blockIdx.y, s = blockIdx.z;
  if (bj > bi) return;
  __shared__ double t[32][33];
  const int tx = threadIdx.x, ty = threadIdx.y;
  const double* src = part + (size_t)s * npair;
  for (int r = ty; r < 32; r += 8) {
    const int mu = bi * 32 + r, nu = bj * 32 + tx;
    double v = 0.0;
    if (mu < nao && nu <= mu) {
      const size_t idx = tri(mu) + nu;
      for (int g = 0; g < nsplit; g++) v += src[(size_t)g * split_stride + idx];
    }
    t[r][tx] = v;
  }
  __syncthreads();
  double* Js = J + (size_t)s * nao * nao;
  for (int r = ty; r < 32; r += 8) {
    const int mu = bi * 32 + r, nu = bj * 32 + tx;  // lower tile (bi,bj)
    if (mu < nao && nu < nao) {
      if (bi != bj) Js[(size_t)mu * nao + nu] = t[r][tx];
      else Js[(size_t)mu * nao + nu] = (nu <= mu) ? t[r][tx] : t[tx][r];
    }
    if (bi != bj) {  // mirrored tile (bj,bi): row nu' = bj*32 + r, col mu' = bi*32 + tx
      const int row = bj * 32 + r, colm = bi * 32 + tx;
      if (row < nao && colm < nao) Js[(size_t)row * nao + colm] = t[tx][r];
    }
  }
}

template <bool VEC>
static cudaError_t launch_j2(int ns, dim3 grid, cudaStream_t st, const double* B, size_t npair, int naux,
                             const double* rho, double* part, size_t split_stride, int rows_per_split) {
  switch (ns) {
#define DFJK_J2_CASE(N)                                                                               \
  case N:                                                                                             \
    k_j2<N, VEC><<<grid, kJ2Threads, 0, st>>>(B, npair, naux, rho, part, split_stride, rows_per_split); \
    break;
    DFJK_J2_CASE(1) DFJK_J2_CASE(2) DFJK_J2_CASE(3) DFJK_J2_CASE(4)
    DFJK_J2_CASE(5) DFJK_J2_CASE(6) DFJK_J2_CASE(7) DFJK_J2_CASE(8)
#undef DFJK_J2_CASE
    default: return cudaErrorInvalidValue;
  }
  return cudaSuccess;
}

// rho_ready: rho was already produced by the fused half-transform; only pass 2 and the epilogue run.
// More than 8 sets are processed in groups of 8 (the accumulators of one pass), each group
// streaming B once per pass.  Returns the number of launches, -1 on a launch failure.
int launch_j_passes(dfjk_ctx* h, const SetInfo& si, double* J_out, bool rho_ready, cudaStream_t st) {
  int launches = 0;
  const int naux = h->naux, nao = h->nao;
  const size_t npair = h->npair;
  const bool vec = (npair % 2 == 0) && h->b_aligned16;   // 16-byte aligned packed rows: 128-bit loads, bulk copies
  const int naux_pad = round_up(naux > 0 ? naux : 1, kJ1Rows);
  const size_t split_stride = (size_t)h->max_nset * npair;
  const int rows_per_split = round_up(cdiv(naux > 0 ? naux : 1, h->j2_splits), 8);
  for (int s0 = 0; s0 < si.nset; s0 += 8) {
    const int ns = si.nset - s0 < 8 ? si.nset - s0 : 8;
    if (naux > 0 && !rho_ready) {
      prof_mark(h, DFJK_PHASE_J1, st);
      dim3 g1(h->j1_chunks, naux_pad / kJ1Rows);
      if (vec && ns >= h->j1_mma_min_sets) {
        if (launch_j1_mma(h->device, g1, st, h->B, npair, naux, h->Dw + (size_t)s0 * npair, ns, h->rho_part, naux_pad) != cudaSuccess)
          return -1;
      } else if (vec) {
        // aux rows per CTA: 64 on long streams; short ones (small: 48 CTAs of 64 rows, medium: 2.6 waves) take the
        // split that needs the least time in whole waves of one CTA per SM, a CTA costing its rows plus a fixed
        // set-up (ring fill; about one row's worth)
        int rows_cta = kJ1Rows;
        double best = 0.0;
        for (int rc = kJ1Rows; rc >= 8; rc >>= 1) {
          const long long ctas = (long long)h->j1_chunks * cdiv(naux, rc);
          const double cost = (double)((ctas + h->num_sms - 1) / h->num_sms) * (rc + 1.0);
          if (rc == kJ1Rows || cost < 0.97 * best) { best = cost; rows_cta = rc; }
        }
        dim3 g1t(h->j1_chunks, cdiv(naux, rows_cta));
        if (dispatch_j1_tma(h->device, ns, g1t, st, h->B, npair, naux, h->Dw + (size_t)s0 * npair, h->rho_part, naux_pad, rows_cta) != cudaSuccess)
          return -1;
      } else {
        k_j1<<<g1, kJ1Warps * 32, 0, st>>>(h->B, npair, naux, h->Dw + (size_t)s0 * npair, ns, h->rho_part, naux_pad);
      }
      dim3 gr(cdiv(naux, 128), ns);
      k_j1_reduce<<<gr, 128, 0, st>>>(h->rho_part, h->j1_chunks, naux_pad, naux, ns, h->rho + (size_t)s0 * naux);
      launches += 2;
    }
    prof_mark(h, DFJK_PHASE_J2, st);
    dim3 g2((unsigned)((npair + 2 * kJ2Threads - 1) / (2 * kJ2Threads)), h->j2_splits);
    // the tensor-pipe kernel wins on long streams (3.13 vs 3.18 ms at large) and whenever there are many sets; on
    // short ones (medium: 0.47 vs 0.42 ms) its per-CTA ring set-up shows, and k_j2 stays
    const bool long_stream = (double)naux * (double)npair * 8.0 >= 8e9;
    if (vec && ns >= (long_stream ? h->j2_mma_min_sets : 7)) {
      dim3 gm((unsigned)((npair + kJ1tSC - 1) / kJ1tSC), h->j2_splits);
      if (launch_j2_mma(h->device, gm, st, h->B, npair, naux, h->rho + (size_t)s0 * naux, ns, h->Jp_part + (size_t)s0 * npair,
                        split_stride, rows_per_split) != cudaSuccess)
        return -1;
      launches += 1;
      continue;
    }
    cudaError_t e2 = vec ? launch_j2<true>(ns, g2, st, h->B, npair, naux, h->rho + (size_t)s0 * naux, h->Jp_part + (size_t)s0 * npair, split_stride, rows_per_split)
                         : launch_j2<false>(ns, g2, st, h->B, npair, naux, h->rho + (size_t)s0 * naux, h->Jp_part + (size_t)s0 * npair, split_stride, rows_per_split);
    if (e2 != cudaSuccess) return -1;
    launches += 1;
  }
  prof_mark(h, DFJK_PHASE_J_EPILOGUE, st);
  const int nb = cdiv(nao, 32);
  dim3 ge(nb, nb, si.nset), be(32, 8);
  k_j_epilogue<<<ge, be, 0, st>>>(h->Jp_part, h->j2_splits, split_stride, npair, nao, J_out);
  return launches + 1;
}

}  // namespace dfjk
