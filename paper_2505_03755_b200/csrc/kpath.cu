// Steps a5-a9, the exchange build (Eq. 16-17) on the FP64 tensor pipe:
//   a5/a6  half-transform  X[P][mu][i] = sum_lam B_P[mu][lam] C'[lam][i]   (k_half_transform)
//          the A operand comes from the re-tiled copy Bt built once in dfjk_create (k_retile: the
//          64 x 16 tiles of the symmetric slice as ready shared-memory images, bulk copies only),
//          or, without it, straight from the packed triangle: chunks below the diagonal as
//          stored, chunks above it as the transpose of the stored tile (only the shared-memory
//          read pattern changes), chunks crossing it element by element.  Epilogues: k-tiled X,
//          k-tiled X + rho partials (step a2 fused), row-major X (AO2MO Eq. 18).
//   a7     SYRK            K_s[mu>=nu] += sum_{P,i in s} X[P][mu][i] X[P][nu][i]   (k_syrk2)
//          lower-triangle T x T tiles (T = 64..112), split-K over the aux rows of the block,
//          partials read-modify-written by exactly one CTA each (no atomics: deterministic);
//          two-operand form K += X X2^T for the density-matrix form (Eq. 16-17 as printed).
//   a8     scheduler       launch_k_path / launch_k_path_dm: aux blocks from the workspace cap,
//          tile size and split-K from a list-schedule model.
//   a9     epilogue        fixed-order sum of the split-K partials, mirrored to both triangles.
// Both GEMMs are warp-specialised: warpgroups 0-1 (8 warps) only issue LDS + DMMA.8x8x4
// (mma.sync m8n8k4 f64; FP64 has no tcgen05/TMEM kind), warpgroup 2 produces the shared-memory
// stages -- bulk async copies (TMA engine, SASS UBLKCP) for the pre-tiled operands C', Bt and X,
// 8-byte cp.async gathers for the packed triangle -- through a 3-stage full/empty mbarrier ring,
// with setmaxnreg moving registers from the producers to the consumers.  All tiles have a row
// stride of 4 mod 16 doubles, which makes both the [row][k] and the [k][row] fragment reads
// bank-conflict-free.
#include "common.cuh"
#include "ctx.h"
#include "pipeline.cuh"

#include <algorithm>
#include <functional>
#include <queue>
#include <vector>

namespace dfjk {

static inline long long cdiv_ll(long long a, long long b) { return (a + b - 1) / b; }

constexpr int kStages = 3;
// Pipeline depth of the half-transform by N tile width: 3 stages of 59 KB at 304 columns; a thin
// tile (AO2MO's active columns, small sets) is bandwidth-bound and keeps up to 8 stages in flight.
// Narrow tiles (at most 96 columns: the `small` config, fragment-sized sets) run TWO CTAs per SM: a tile is
// only nao/16 short chunks, so its epilogue (X stores, rho) is a sizeable share of it, and with a second
// resident CTA the tensor pipe has the other tile's chunks to work on meanwhile.  Register budget then:
// 80 per thread at launch, 40 for the producer warpgroup, 96 for the consumers.
__host__ __device__ constexpr int ht_ctas_per_sm(int wn) { return wn <= 6 ? 2 : 1; }
__host__ __device__ constexpr int ht_stages(int wn) {
  const int stage_bytes = (64 * kHtLd + 16 * wn * kHtLd) * 8;
  const int fit = ((ht_ctas_per_sm(wn) == 2 ? 100 : 200) * 1024) / stage_bytes;
  return fit < 3 ? 3 : (fit > 8 ? 8 : fit);
}
constexpr int kThreads = 384;             // 2 consumer warpgroups + 1 producer warpgroup

// ------------------------------------------------------------------ half-transform
// CTA: 64 rows (mu) of one aux slice x NT = 16*WN columns (normally ALL columns of C', so the
// packed tensor passes through the SM once per row block).  Consumers: 4 (M, 16 rows) x 2 (N
// halves); warps w and w+4 share an SM sub-partition.  k-chunks of 16 (kHtBK).
//   C' tiled:  Ct[(chunk * ct_rows + n) * 20 + k]                  (written by k_prep_ct)
//   X tiled:   X[((pl * nch + n/32) * mu_pad + mu) * 36 + n%32]    (read by k_syrk2 with bulk copies)
constexpr int kHtATile = 64 * kHtLd;       // 1280 doubles >= 16 * 68 = 1088
constexpr int kHtLdT = 64 + 4;             // 68: row stride of the transposed [16][64] A tile

// Launch parameters of the half-transform.  The kernel is persistent: gridDim.x CTAs (one per SM)
// walk the tiles (aux row, 64-row block, N tile) round-robin, and the mbarrier ring keeps running
// across tile boundaries, so the producer prefetches the next tile while the consumers write X.
struct HtParams {
  const double* Bp; size_t npair; int nao;
  const double* Ct; int ct_rows; int nocc_pad;
  double* X; int nch; int mu_pad;       // EPI 0/1: k-tiled X for the SYRK
  int p_first, nb, ntm, ntn;            // aux rows [p_first, p_first + nb), 64-row blocks, N tiles
  double* rho_ht; int nset; int col0[kMaxSets + 1];   // EPI 1: per-warp partials of rho (step a2 fused)
  const unsigned int* sgnbits;          // EPI 1: sign bits of the occupations (k_prep_ct)
  int ldx, xrows;                       // EPI 2: row-major X[(pl * xrows + mu) * ldx + n]
  // optional re-tiled copy of B (dfjk_create): per aux row the 64 x 16 tiles of the symmetric
  // slice at and below the diagonal blocks, each stored as the padded [64][20] shared-memory image
  // (tile (mb, c), c < 4 (mb + 1), at image 2 mb (mb + 1) + c), so that the A operand of every chunk
  // is one bulk copy (a stored or diagonal tile) or four (the transpose: 16 rows of four images)
  const double* Bt; size_t bt_pstride;
  // with Bt and 1 <= nao % 64 <= 48 the last 64-row block of an aux row holds v = pair_last < 4 pieces of 16 rows:
  // the nb * v pieces of the last blocks of consecutive aux rows are then packed four to a tile (piece k of the
  // block range is rows 16 (k % v).. of aux row k / v), scheduled after the full tiles.  0 = off
  int pair_last;
};

// tile index -> (aux row, 64-row block, N tile); paired: the tile holds the pieces pl .. pl + 3 of the last blocks
struct HtTile { int pl, mb, nt; bool paired; };
template <bool PAIR>
__device__ __forceinline__ int ht_num_tiles(const HtParams& q) {
  return PAIR ? q.nb * (q.ntm - 1) * q.ntn + ((q.nb * q.pair_last + 3) >> 2) * q.ntn : q.nb * q.ntm * q.ntn;
}
template <bool PAIR>
__device__ __forceinline__ HtTile ht_tile(const HtParams& q, int tile) {
  HtTile t;
  if (!PAIR) {
    const int tiles_per_p = q.ntm * q.ntn;
    t.pl = tile / tiles_per_p;
    const int rem = tile - t.pl * tiles_per_p;
    t.mb = rem / q.ntn; t.nt = rem % q.ntn; t.paired = false;
    return t;
  }
  const int per_p = (q.ntm - 1) * q.ntn, nfull = q.nb * per_p;
  if (tile < nfull) {
    t.pl = tile / per_p;
    const int rem = tile - t.pl * per_p;
    t.mb = rem / q.ntn; t.nt = rem - t.mb * q.ntn; t.paired = false;
  } else {
    const int t2 = tile - nfull;
    t.pl = 4 * (t2 / q.ntn); t.nt = t2 % q.ntn; t.mb = q.ntm - 1; t.paired = true;
  }
  return t;
}

// EPI = 0: X k-tiled for k_syrk2.  EPI = 1: the same, plus rho[s][P] = sum_{mu,i in s} X[mu][i] C'[mu][i]
// (= sum_{mu,lam} B_P[mu][lam] D_s[lam][mu], Eq. 14) as per-warp partials, so that a get_jk call that
// wants both J and K streams B twice instead of three times.  EPI = 2: X row-major (AO2MO, Eq. 18).
// PAIR (compile-time, so that the unpaired instances keep their register budget): HtParams::pair_last
template <int WN, int EPI, bool PAIR>
__global__ void __launch_bounds__(kThreads, ht_ctas_per_sm(WN))
k_half_transform(const __grid_constant__ HtParams q) {
  extern __shared__ __align__(128) double smem[];
  constexpr int NT = 16 * WN;
  constexpr int kS = ht_stages(WN);               // 3 for the wide tiles, up to 8 for thin ones
  constexpr uint32_t kBBytes = NT * kHtLd * 8;
  double* sA = smem;                               // kS x kHtATile
  double* sB = smem + kS * kHtATile;          // kS x NT*kHtLd
  __shared__ __align__(8) unsigned long long bars[2 * kS];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kS]);
  const int tid = threadIdx.x, l = tid & 31;
  // PAIR: the warp index read from lane 0, so that the compiler sees the per-warp row assignment (and the branch
  // that skips a piece past the last aux row) as warp-uniform
  const int w = PAIR ? __shfl_sync(0xffffffffu, tid >> 5, 0) : tid >> 5;
  const int nao = q.nao;
  const int nk4 = (nao + 3) >> 2;                  // k4 steps that carry data
  const int nchunks = (nk4 + 3) >> 2;
  const int tiles_per_p = q.ntm * q.ntn, ntiles = ht_num_tiles<PAIR>(q);

  if (tid == 0) {
    for (int s = 0; s < kS; s++) {
      mbar_init(full0 + 8 * s, q.Bt ? 1 : 128 + 1);   // the expect_tx arrival (+ 128 cp.async arrivals when gathering)
      mbar_init(empty0 + 8 * s, 8);        // one arrival per consumer warp
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (w >= 8) {
    // ===================== producer warpgroup =====================
    reg_dec<kProducerRegs>();
    const int tp = tid - 256;
    if (q.Bt) {
      // re-tiled B: one elected thread, bulk copies only
      if (tp != 0) return;
      const uint32_t sA_u32 = smem_u32(sA), sB_u32 = smem_u32(sB);
      constexpr uint32_t kImgBytes = 64 * kHtLd * 8, kPieceBytes = 16 * kHtLd * 8;
      int g = 0;
      for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const HtTile ht = ht_tile<PAIR>(q, tile);
        const int pl = ht.pl, mb = ht.mb, n0 = ht.nt * NT;
        const double* BtP = q.Bt + (size_t)(q.p_first + ((PAIR && ht.paired) ? 0 : pl)) * q.bt_pstride;
        // packed tile: number of pieces that exist, aux row and piece-in-block of the first one
        int npc = 0, pk0 = 0, ik0 = 0;
        if (PAIR && ht.paired) {
          npc = min(4, q.nb * q.pair_last - pl);
          pk0 = pl / q.pair_last;
          ik0 = pl - pk0 * q.pair_last;
        }
        for (int c = 0; c < nchunks; c++, g++) {
          const int stage = g % kS;
          const uint32_t fullb = full0 + 8 * stage;
          mbar_wait(empty0 + 8 * stage, ((g / kS) & 1) ^ 1);
          mbar_arrive_expect_tx(fullb, kBBytes + ((PAIR && ht.paired) ? (uint32_t)npc * kPieceBytes : kImgBytes));
          bulk_g2s(sB_u32 + (uint32_t)stage * kBBytes, q.Ct + ((size_t)c * q.ct_rows + n0) * kHtLd, kBBytes, fullb);
          const uint32_t a_base = sA_u32 + (uint32_t)(stage * kHtATile) * 8u;
          if ((PAIR && ht.paired)) {                           // 16-row pieces of the last block's image (always stored / diagonal)
            const size_t img = (size_t)(2 * mb * (mb + 1) + c) * (64 * kHtLd);
            // consecutive pieces of one aux row are contiguous on both sides: one copy per aux row in the tile
            const double* src = BtP + (size_t)pk0 * q.bt_pstride + img;
            for (int k = 0, ik = ik0; k < npc; ik = 0, src += q.bt_pstride) {
              const int run = min(q.pair_last - ik, npc - k);
              bulk_g2s(a_base + (uint32_t)k * kPieceBytes, src + (size_t)ik * 16 * kHtLd, (uint32_t)run * kPieceBytes, fullb);
              k += run;
            }
          } else if (c < 4 * (mb + 1)) {             // stored or diagonal tile: its image as it is
            bulk_g2s(a_base, BtP + (size_t)(2 * mb * (mb + 1) + c) * (64 * kHtLd), kImgBytes, fullb);
          } else {                                   // transpose: rows 16 (c % 4) .. + 15 of the images (c / 4, 4 mb + qq)
            const int mbl = c >> 2;
            const double* src = BtP + (size_t)(2 * mbl * (mbl + 1) + 4 * mb) * (64 * kHtLd) + (size_t)(c & 3) * 16 * kHtLd;
#pragma unroll
            for (int qq = 0; qq < 4; qq++)
              bulk_g2s(a_base + (uint32_t)qq * kPieceBytes, src + (size_t)qq * (64 * kHtLd), kPieceBytes, fullb);
          }
        }
      }
      return;
    }
    const int kd = tp & 15, md = tp >> 4;          // direct / crossing: element (md + 8q, kd)
    const int mt = tp & 63, kt = tp >> 6;          // transposed:        element (mt, kt + 2q)
    const uint32_t sA_u32 = smem_u32(sA), sB_u32 = smem_u32(sB);
    const uint32_t a_dst_d = (uint32_t)(md * kHtLd + kd) * 8u, a_dst_t = (uint32_t)(kt * kHtLdT + mt) * 8u;
    int g = 0;                                     // chunk counter across tiles
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
      const HtTile ht = ht_tile<PAIR>(q, tile);
      const int pl = ht.pl, m0 = ht.mb * 64, n0 = ht.nt * NT;
      const double* BpP = q.Bp + (size_t)(q.p_first + pl) * q.npair;
      const bool okt = m0 + mt < nao;
      for (int c = 0; c < nchunks; c++, g++) {
        const int stage = g % kS;
        const uint32_t fullb = full0 + 8 * stage;
        mbar_wait(empty0 + 8 * stage, ((g / kS) & 1) ^ 1);
        const int l0 = c * kHtBK;
        if (tp == 0) {
          mbar_arrive_expect_tx(fullb, kBBytes);
          bulk_g2s(sB_u32 + (uint32_t)stage * kBBytes, q.Ct + ((size_t)c * q.ct_rows + n0) * kHtLd, kBBytes, fullb);
        }
        const uint32_t a_base = sA_u32 + (uint32_t)(stage * kHtATile) * 8u;
        if (l0 + kHtBK - 1 <= m0) {                  // stored rows, all lam <= mu
#pragma unroll
          for (int qq = 0; qq < 8; qq++) {
            const int mu = m0 + md + 8 * qq;
            const bool ok = mu < nao;
            cp_async8(a_base + a_dst_d + (uint32_t)(qq * 8 * kHtLd) * 8u,
                      BpP + (ok ? (uint32_t)(mu * (mu + 1) / 2 + l0 + kd) : 0u), ok);
          }
        } else if (l0 >= m0 + 63) {                  // transpose of the stored tile, all lam >= mu
#pragma unroll
          for (int qq = 0; qq < 8; qq++) {
            const int lam = l0 + kt + 2 * qq;
            const bool ok = okt && lam < nao;
            cp_async8(a_base + a_dst_t + (uint32_t)(qq * 2 * kHtLdT) * 8u,
                      BpP + (ok ? (uint32_t)(lam * (lam + 1) / 2 + m0 + mt) : 0u), ok);
          }
        } else {                                     // crossing the diagonal
          const int lam = l0 + kd;
#pragma unroll
          for (int qq = 0; qq < 8; qq++) {
            const int mu = m0 + md + 8 * qq;
            const bool ok = mu < nao && lam < nao;
            uint32_t off = 0;
            if (ok) off = (lam <= mu) ? (uint32_t)(mu * (mu + 1) / 2 + lam) : (uint32_t)(lam * (lam + 1) / 2 + mu);
            cp_async8(a_base + a_dst_d + (uint32_t)(qq * 8 * kHtLd) * 8u, BpP + off, ok);
          }
        }
        cp_async_mbar_arrive_noinc(fullb);
      }
    }
    return;
  }

  // ===================== consumer warpgroups =====================
  reg_inc<ht_ctas_per_sm(WN) == 2 ? 96 : kConsumerRegs>();
  const int r = l >> 2, j = l & 3;
  const int wm = w & 3, wn = w >> 2;
  double acc[2][WN][2];

  int g = 0;
  for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const HtTile ht = ht_tile<PAIR>(q, tile);
    const int mb = ht.mb, nt = ht.nt, rem = PAIR ? mb * q.ntn + nt : tile - ht.pl * tiles_per_p;
    const int m0 = mb * 64, n0 = nt * NT;
#pragma unroll
    for (int t = 0; t < 2; t++)
#pragma unroll
      for (int u = 0; u < WN; u++) acc[t][u][0] = acc[t][u][1] = 0.0;

    for (int c = 0; c < nchunks; c++, g++) {
      const int stage = g % kS;
      const int l0 = c * kHtBK;
      const bool tr = (l0 >= m0 + 63) && !(l0 + kHtBK - 1 <= m0);
      const int ksteps = min(4, nk4 - c * 4);
      mbar_wait(full0 + 8 * stage, (g / kS) & 1);
      const double* b_ptr = sB + stage * NT * kHtLd + (wn * 8 * WN + r) * kHtLd + j;
      if (!tr) {
        const double* a_ptr = sA + stage * kHtATile + (wm * 16 + r) * kHtLd + j;
#pragma unroll
        for (int kk = 0; kk < 4; kk++) {
          if (kk < ksteps) {
            const double a0 = a_ptr[4 * kk], a1 = a_ptr[8 * kHtLd + 4 * kk];
            double b[WN];
#pragma unroll
            for (int u = 0; u < WN; u++) b[u] = b_ptr[u * 8 * kHtLd + 4 * kk];
#pragma unroll
            for (int u = 0; u < WN; u++) {
              dmma884(acc[0][u][0], acc[0][u][1], a0, b[u]);
              dmma884(acc[1][u][0], acc[1][u][1], a1, b[u]);
            }
          }
        }
      } else {
        // gathered: one [16 lam][64 mu + 4] tile; re-tiled: four [16 lam][16 mu + 4] pieces, piece wm
        // holds this warp's 16 rows
        const int ldt = q.Bt ? kHtLd : kHtLdT;
        const double* a_ptr = sA + stage * kHtATile + (q.Bt ? wm * 16 * kHtLd + r : wm * 16 + r) + j * ldt;
#pragma unroll
        for (int kk = 0; kk < 4; kk++) {
          if (kk < ksteps) {
            const double a0 = a_ptr[4 * kk * ldt], a1 = a_ptr[8 + 4 * kk * ldt];
            double b[WN];
#pragma unroll
            for (int u = 0; u < WN; u++) b[u] = b_ptr[u * 8 * kHtLd + 4 * kk];
#pragma unroll
            for (int u = 0; u < WN; u++) {
              dmma884(acc[0][u][0], acc[0][u][1], a0, b[u]);
              dmma884(acc[1][u][0], acc[1][u][1], a1, b[u]);
            }
          }
        }
      }
      __syncwarp();
      if (l == 0) mbar_arrive(empty0 + 8 * stage);
    }
    // epilogue: lane owns X[mu][n], X[mu][n+1] with mu = mrow0 + 8t + r, n = n0 + 8 (wn WN + u) + 2j
    // rows of this warp: 16 wm.. of aux row pl; in a paired tile piece ht.pl + wm = rows 16 ip.. of aux row pl
    const int pl = (PAIR && ht.paired) ? (ht.pl + wm) / q.pair_last : ht.pl;
    const int ip = (PAIR && ht.paired) ? ht.pl + wm - pl * q.pair_last : wm;
    const int mrow0 = m0 + ip * 16;
    if (PAIR && pl >= q.nb) continue;             // a piece slot of the last packed tile past the last aux row
    if (EPI == 2) {
      double* Xp = q.X + (size_t)pl * q.xrows * q.ldx;
#pragma unroll
      for (int t = 0; t < 2; t++) {
        const int mu = mrow0 + 8 * t + r;
        if (mu >= nao) continue;
#pragma unroll
        for (int u = 0; u < WN; u++) {
          const int n = n0 + 8 * (wn * WN + u) + 2 * j;
          if (n < q.nocc_pad)
            *reinterpret_cast<double2*>(Xp + (size_t)mu * q.ldx + n) = make_double2(acc[t][u][0], acc[t][u][1]);
        }
      }
    } else {
      double* Xp = q.X + (size_t)pl * q.nch * q.mu_pad * kLdT;
#pragma unroll
      for (int t = 0; t < 2; t++) {
        const int mu = mrow0 + 8 * t + r;
        if (mu >= nao) continue;
#pragma unroll
        for (int u = 0; u < WN; u++) {
          const int n = n0 + 8 * (wn * WN + u) + 2 * j;
          if (n < q.nocc_pad)
            *reinterpret_cast<double2*>(Xp + ((size_t)(n >> 5) * q.mu_pad + mu) * kLdT + (n & 31)) =
                make_double2(acc[t][u][0], acc[t][u][1]);
        }
      }
    }
    if (EPI == 1) {
      // rho partial of this warp: sum over its 16 rows x 8 WN columns of X .* C', set by set (every
      // 8-column tile belongs to one set; a warp's tiles of one set are contiguous).  One slot of
      // nset doubles per (aux row, tile, warp); k_rho_reduce sums the slots in fixed order.
      const int nslots = tiles_per_p * 8;
      double* slot = q.rho_ht + ((size_t)(q.p_first + pl) * nslots + (size_t)rem * 8 + (ip + 4 * wn)) * q.nset;
      for (int s = l; s < q.nset; s += 32) slot[s] = 0.0;
      if ((PAIR && ht.paired) && ip == 0)                          // the slots of the pieces the last block does not have stay empty
        for (int i2 = q.pair_last; i2 < 4; i2++)
          for (int s = l; s < q.nset; s += 32) (slot + i2 * q.nset)[s] = 0.0;
      int myset = -1;
      if (l < WN) {
        const int col = n0 + 8 * (wn * WN + l);
        for (int s = 0; s < q.nset; s++)
          if (col >= q.col0[s] && col < q.col0[s + 1]) myset = s;
      }
      __syncwarp();
      // common case: every column tile of this warp belongs to the same set -> straight-line code,
      // four independent partial sums, one reduction
      const int set0 = __shfl_sync(0xffffffffu, myset, 0);
      const bool one_set = set0 >= 0 && __all_sync(0xffffffffu, l >= WN || myset == set0);
      if (one_set) {
        double p4[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int u0 = 0; u0 < WN; u0 += 4) {
          double cv[4][2][2];
#pragma unroll
          for (int uu = 0; uu < 4; uu++) {
            if (u0 + uu >= WN) continue;
            const int n = n0 + 8 * (wn * WN + u0 + uu) + 2 * j;
#pragma unroll
            for (int t = 0; t < 2; t++) {
              const int mu = min(mrow0 + 8 * t + r, nao - 1);     // rows past nao hold acc = 0
              const double* cp = q.Ct + ((size_t)(mu >> 4) * q.ct_rows + n) * kHtLd + (mu & 15);
              cv[uu][t][0] = __ldg(cp);
              cv[uu][t][1] = __ldg(cp + kHtLd);
            }
            // rho = sum X' C' sign(occ): flip the sign bit of C' for columns with a negative occupation
            const unsigned int sw = __ldg(q.sgnbits + (n >> 5)) >> (n & 31);
            if (sw & 3u) {
#pragma unroll
              for (int t = 0; t < 2; t++) {
                cv[uu][t][0] = flip_sign(cv[uu][t][0], (sw & 1u) << 31);
                cv[uu][t][1] = flip_sign(cv[uu][t][1], (sw & 2u) << 30);
              }
            }
          }
#pragma unroll
          for (int uu = 0; uu < 4; uu++) {
            if (u0 + uu >= WN) continue;
#pragma unroll
            for (int t = 0; t < 2; t++) {
              p4[2 * t] = fma(acc[t][u0 + uu][0], cv[uu][t][0], p4[2 * t]);
              p4[2 * t + 1] = fma(acc[t][u0 + uu][1], cv[uu][t][1], p4[2 * t + 1]);
            }
          }
        }
        double v = (p4[0] + p4[1]) + (p4[2] + p4[3]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (l == 0) slot[set0] = v;
        continue;
      }
      double cur = 0.0;
      int cur_s = -1;
      auto flush = [&]() {
        double v = cur;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (l == 0) slot[cur_s] = v;
      };
      // groups of four column tiles: all 16 C' loads of a group are issued before its FMAs, so the
      // L2 latency is paid once per group and not once per element
#pragma unroll
      for (int u0 = 0; u0 < WN; u0 += 4) {
        double cv[4][2][2];
        int su[4];
#pragma unroll
        for (int uu = 0; uu < 4; uu++) {
          if (u0 + uu >= WN) continue;
          su[uu] = __shfl_sync(0xffffffffu, myset, u0 + uu);
          const int n = n0 + 8 * (wn * WN + u0 + uu) + 2 * j;
#pragma unroll
          for (int t = 0; t < 2; t++) {
            const int mu = mrow0 + 8 * t + r;
            const bool ok = su[uu] >= 0 && mu < nao;
            const double* cp = q.Ct + ((size_t)(ok ? (mu >> 4) : 0) * q.ct_rows + (ok ? n : 0)) * kHtLd + (mu & 15);
            cv[uu][t][0] = ok ? __ldg(cp) : 0.0;
            cv[uu][t][1] = ok ? __ldg(cp + kHtLd) : 0.0;
          }
          if (su[uu] >= 0) {
            const unsigned int sw = __ldg(q.sgnbits + (n >> 5)) >> (n & 31);
#pragma unroll
            for (int t = 0; t < 2; t++) {
              cv[uu][t][0] = flip_sign(cv[uu][t][0], (sw & 1u) << 31);
              cv[uu][t][1] = flip_sign(cv[uu][t][1], (sw & 2u) << 30);
            }
          }
        }
#pragma unroll
        for (int uu = 0; uu < 4; uu++) {
          if (u0 + uu >= WN) continue;
          if (su[uu] != cur_s) {
            if (cur_s >= 0) flush();
            cur = 0.0;
            cur_s = su[uu];
          }
#pragma unroll
          for (int t = 0; t < 2; t++) {
            cur = fma(acc[t][u0 + uu][0], cv[uu][t][0], cur);
            cur = fma(acc[t][u0 + uu][1], cv[uu][t][1], cur);
          }
        }
      }
      if (cur_s >= 0) flush();
    }
  }
}

// One-time re-tiling of B for the half-transform (dfjk_create): image (mb, c) of aux row P holds
// Bsym_P[64 mb + i][16 c + k] for i < 64, k < 16 (zero past nao, zero padding columns 16..19).
__global__ void __launch_bounds__(256)
k_retile(const double* __restrict__ Bp, size_t npair, int nao, int ntm, double* __restrict__ Bt, size_t bt_pstride) {
  const int P = blockIdx.y;
  const double* BpP = Bp + (size_t)P * npair;
  double* BtP = Bt + (size_t)P * bt_pstride;
  const int nimg = 2 * ntm * (ntm + 1);
  for (int img = blockIdx.x; img < nimg; img += gridDim.x) {
    int mb = (int)(sqrt(0.5 * img + 0.25) - 0.5);               // img = 2 mb (mb + 1) + c, 0 <= c < 4 (mb + 1)
    while (2 * (mb + 1) * (mb + 2) <= img) mb++;
    while (2 * mb * (mb + 1) > img) mb--;
    const int c = img - 2 * mb * (mb + 1);
    double* dst = BtP + (size_t)img * (64 * kHtLd);
    for (int e = threadIdx.x; e < 64 * kHtLd; e += 256) {
      const int i = e / kHtLd, k = e - i * kHtLd;
      const int mu = 64 * mb + i, lam = 16 * c + k;
      double v = 0.0;
      if (k < kHtBK && mu < nao && lam < nao) v = BpP[lam <= mu ? tri(mu) + lam : tri(lam) + mu];
      dst[e] = v;
    }
  }
}

size_t retile_doubles_per_aux_row(int nao) {
  const int ntm = cdiv(nao, 64);
  return (size_t)2 * ntm * (ntm + 1) * 64 * kHtLd;
}

cudaError_t launch_retile(const double* Bp, size_t npair, int nao, int naux, double* Bt) {
  if (naux == 0) return cudaSuccess;
  const int ntm = cdiv(nao, 64);
  const int nimg = 2 * ntm * (ntm + 1);
  for (int p0 = 0; p0 < naux; p0 += 32768) {                   // gridDim.y limit
    const int nb = naux - p0 < 32768 ? naux - p0 : 32768;
    dim3 grid(nimg < 64 ? nimg : 64, nb);
    k_retile<<<grid, 256>>>(Bp + (size_t)p0 * npair, npair, nao, ntm, Bt + (size_t)p0 * retile_doubles_per_aux_row(nao),
                            retile_doubles_per_aux_row(nao));
  }
  return cudaGetLastError();
}

// rho[s][P] = sum over the per-warp slots of k_half_transform<., 1>, ascending (fixed order)
__global__ void k_rho_reduce(const double* __restrict__ rho_ht, int nslots, int nset, int naux,
                             double* __restrict__ rho) {
  const int P = blockIdx.x * blockDim.x + threadIdx.x, s = blockIdx.y;
  if (P >= naux) return;
  const double* p = rho_ht + (size_t)P * nslots * nset + s;
  double t = 0.0;
  for (int k = 0; k < nslots; k++) t += p[(size_t)k * nset];
  rho[(size_t)s * naux + P] = t;
}

// ------------------------------------------------------------------ SYRK
// CTA: one lower-triangle T x T tile (ta >= tb) of K_s, T = 16*WM in {64,80,96,112} chosen per nao
// by least modelled work, and one split of the block's aux rows.  The reduction runs over (aux
// row, 32-column chunk of X) pairs; a chunk that straddles two sets contributes only the k4 steps
// of this set.  Both operand tiles are contiguous T x 36 blocks of the tiled X, fetched by one
// elected producer thread with bulk async copies.  The T x T tile is cut into 2 x 2
// blocks of WM x WM MMA tiles, one block per SM sub-partition; the two warps of a sub-partition
// (w and w+4) both hold the whole block in registers and take alternate k4 steps (an in-CTA
// split-K), so they are perfectly symmetric: 2 WM fragment loads per WM^2 DMMAs each.
// Diagonal tiles (ta == tb) skip what the epilogue never reads: the strictly-upper block is not
// computed at all -- its sub-partition instead shares the k4 steps of the lower block (4-way) --
// and the two diagonal blocks compute their lower MMA tiles only: WM(WM+1)/2 DMMAs per k4 step on
// the critical sub-partition instead of WM^2.
// At the end the partner warps pass their accumulators through the (drained) pipeline stages and
// the owner warp adds them in a fixed order before the read-modify-write of the private partial.
__device__ __forceinline__ void consumer_bar_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }

struct Syrk2Consumer {
  const double* sA; const double* sB; uint32_t full0, empty0;
  int nchunks, ch0, ch1, c0, c1, tile_doubles;
  int row0, col0;          // block origin inside the CTA tile
  int kidx;                // this warp takes the k4 steps kk = kidx mod KMOD of every chunk
  const unsigned int* sgn; // sign bits of the occupations per 32-column chunk (nullptr: all positive)
};

template <int WM, bool LOWER, int KMOD>
__device__ __forceinline__ void syrk2_mainloop(const Syrk2Consumer& q, int l, double (&acc)[WM][WM][2]) {
  const int r = l >> 2, j = l & 3;
#pragma unroll
  for (int tt = 0; tt < WM; tt++)
#pragma unroll
    for (int u = 0; u < WM; u++) acc[tt][u][0] = acc[tt][u][1] = 0.0;
  int ch = q.ch0;
  for (int c = 0; c < q.nchunks; c++) {
    const int stage = c % kStages;
    // k4 steps of this chunk that belong to the set: columns [max(c0, 32 ch), min(c1, 32 ch + 32))
    const int k_lo = (max(q.c0, ch * 32) - ch * 32) >> 2, k_hi = (min(q.c1, ch * 32 + 32) - ch * 32 + 3) >> 2;
    // K = sum_i sign(occ_i) X'_i X'_i^T: columns with a negative occupation flip the sign bit of the
    // column-operand fragment (an integer op; the word is warp-uniform and zero in the common case)
    const unsigned int sw = q.sgn ? __ldg(q.sgn + ch) : 0u;
    if (++ch == q.ch1) ch = q.ch0;
    mbar_wait(q.full0 + 8 * stage, (c / kStages) & 1);
    const double* a_ptr = q.sA + stage * q.tile_doubles + (q.row0 + r) * kLdT + j;
    const double* b_ptr = q.sB + stage * q.tile_doubles + (q.col0 + r) * kLdT + j;
    auto step = [&](int kk) {
      double a[WM], b[WM];
#pragma unroll
      for (int tt = 0; tt < WM; tt++) a[tt] = a_ptr[tt * 8 * kLdT + 4 * kk];
#pragma unroll
      for (int u = 0; u < WM; u++) b[u] = b_ptr[u * 8 * kLdT + 4 * kk];
      if (sw) {
        const unsigned int m = ((sw >> (4 * kk + j)) & 1u) << 31;
#pragma unroll
        for (int u = 0; u < WM; u++) b[u] = flip_sign(b[u], m);
      }
#pragma unroll
      for (int tt = 0; tt < WM; tt++)
#pragma unroll
        for (int u = 0; u < WM; u++)
          if (!LOWER || u <= tt) dmma884(acc[tt][u][0], acc[tt][u][1], a[tt], b[u]);
    };
    if (k_lo == 0 && k_hi == 8) {
#pragma unroll
      for (int i = 0; i < 8 / KMOD; i++) step(q.kidx + i * KMOD);
    } else {
      // chunk shared with another set (or the ragged last chunk): same unrolled steps, each under a
      // warp-uniform predicate
#pragma unroll
      for (int i = 0; i < 8 / KMOD; i++) {
        const int kk = q.kidx + i * KMOD;
        if (kk >= k_lo && kk < k_hi) step(kk);
      }
    }
    __syncwarp();
    if (l == 0) mbar_arrive(q.empty0 + 8 * stage);
  }
}

// accumulators of a partner warp -> shared memory slot / owner adds a slot
template <int WM, bool LOWER>
__device__ __forceinline__ void syrk2_put(double* red, int slot, int l, const double (&acc)[WM][WM][2]) {
  double2* p = reinterpret_cast<double2*>(red) + (size_t)slot * WM * WM * 32 + l;
#pragma unroll
  for (int tt = 0; tt < WM; tt++)
#pragma unroll
    for (int u = 0; u < WM; u++)
      if (!LOWER || u <= tt) p[(tt * WM + u) * 32] = make_double2(acc[tt][u][0], acc[tt][u][1]);
}
template <int WM, bool LOWER>
__device__ __forceinline__ void syrk2_add(const double* red, int slot, int l, double (&acc)[WM][WM][2]) {
  const double2* p = reinterpret_cast<const double2*>(red) + (size_t)slot * WM * WM * 32 + l;
#pragma unroll
  for (int tt = 0; tt < WM; tt++)
#pragma unroll
    for (int u = 0; u < WM; u++)
      if (!LOWER || u <= tt) {
        const double2 v = p[(tt * WM + u) * 32];
        acc[tt][u][0] += v.x;
        acc[tt][u][1] += v.y;
      }
}
// read-modify-write of this CTA's private partial tile (entries above the diagonal of a diagonal
// MMA tile are written too; the epilogue reads mu >= nu only)
template <int WM, bool LOWER>
__device__ __forceinline__ void syrk2_store(double* Kp, int nao, int mu0, int nu0, int first, int l,
                                            const double (&acc)[WM][WM][2]) {
  const int r = l >> 2, j = l & 3;
#pragma unroll
  for (int tt = 0; tt < WM; tt++) {
    const int mu = mu0 + tt * 8 + r;
    if (mu >= nao) continue;
#pragma unroll
    for (int u = 0; u < WM; u++) {
      if (LOWER && u > tt) continue;
      const int nu = nu0 + u * 8 + 2 * j;
      double* p = Kp + (size_t)mu * nao + nu;
      if (nu < nao) p[0] = first ? acc[tt][u][0] : p[0] + acc[tt][u][0];
      if (nu + 1 < nao) p[1] = first ? acc[tt][u][1] : p[1] + acc[tt][u][1];
    }
  }
}

// grid: the n_off * ksplit off-diagonal CTAs first (blockIdx.x = g * n_off + t), then the
// ntiles_m * ksplit cheaper diagonal ones, which fill the tail of the last wave.
// the sets of one launch (blockIdx.y): columns [c0, c1) of X and the offset of K_s inside a partial slot; the
// widest set comes first so that the thin ones fill the tail of the launch
struct SyrkSets {
  int c0[kMaxSets], c1[kMaxSets];
  long long koff[kMaxSets];
};

template <int WM>
__global__ void __launch_bounds__(kThreads, 1)
k_syrk2(const double* __restrict__ X, const double* __restrict__ X2, const unsigned int* __restrict__ sgn, int nao,
        int nch, int mu_pad, const __grid_constant__ SyrkSets sets, int nrows_blk, int rows_per_split, int ntiles_m, int ksplit,
        double* __restrict__ Kpart, size_t split_stride, int first) {
  const int c0 = sets.c0[blockIdx.y], c1 = sets.c1[blockIdx.y];
  double* Kpart_s = Kpart + sets.koff[blockIdx.y];
  // X2 == nullptr: K += X X^T (SYRK).  Otherwise K += X X2^T for a product known to be symmetric
  // (density-matrix form, Eq. 16-17: X = B_P D, X2 = B_P): the column operand comes from X2, and
  // diagonal tiles fetch both operands.
  constexpr int T = 16 * WM;
  constexpr int kTileDoubles = T * kLdT;
  constexpr uint32_t kTileBytes = kTileDoubles * 8;
  extern __shared__ __align__(128) double smem[];
  double* sA = smem;
  double* sB = smem + kStages * kTileDoubles;
  __shared__ __align__(8) unsigned long long bars[2 * kStages];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kStages]);
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
  const int n_off = ntiles_m * (ntiles_m - 1) / 2;
  int ta, tb, g;
  const bool diag = (int)blockIdx.x >= n_off * ksplit;
  if (!diag) {
    const int t = blockIdx.x % n_off;
    g = blockIdx.x / n_off;
    ta = (int)((sqrt(8.0 * t + 1.0) + 1.0) * 0.5);          // t = ta(ta-1)/2 + tb, ta > tb
    while (ta * (ta + 1) / 2 <= t) ta++;
    while (ta * (ta - 1) / 2 > t) ta--;
    tb = t - ta * (ta - 1) / 2;
  } else {
    const int t = blockIdx.x - n_off * ksplit;
    ta = tb = t % ntiles_m;
    g = t / ntiles_m;
  }
  const bool one_operand = diag && X2 == nullptr;
  const int a0 = ta * T, b0 = tb * T;
  const int p_beg = g * rows_per_split;
  int p_end = p_beg + rows_per_split;
  if (p_end > nrows_blk) p_end = nrows_blk;
  const int np = p_end > p_beg ? p_end - p_beg : 0;
  const int ch0 = c0 >> 5, ch1 = (c1 + 31) >> 5;   // X chunks that hold columns of this set
  const int nchunks = np * (ch1 - ch0);

  if (tid == 0) {
    for (int s = 0; s < kStages; s++) {
      mbar_init(full0 + 8 * s, 1);         // the expect_tx arrival of the elected producer
      mbar_init(empty0 + 8 * s, 8);        // one arrival per consumer warp
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (w >= 8) {
    // ===================== producer warpgroup (one elected thread works) =====================
    reg_dec<kProducerRegs>();
    if (tid == 256) {
      const uint32_t sA_u32 = smem_u32(sA), sB_u32 = smem_u32(sB);
      const size_t chunk_stride = (size_t)mu_pad * kLdT, row_stride = (size_t)nch * chunk_stride;
      int P = p_beg, ch = ch0;
      for (int c = 0; c < nchunks; c++) {
        const int stage = c % kStages;
        const uint32_t fullb = full0 + 8 * stage;
        mbar_wait(empty0 + 8 * stage, ((c / kStages) & 1) ^ 1);
        const size_t off = (size_t)P * row_stride + (size_t)ch * chunk_stride;
        mbar_arrive_expect_tx(fullb, one_operand ? kTileBytes : 2 * kTileBytes);
        bulk_g2s(sA_u32 + (uint32_t)stage * kTileBytes, X + off + (size_t)a0 * kLdT, kTileBytes, fullb);
        if (!one_operand)
          bulk_g2s(sB_u32 + (uint32_t)stage * kTileBytes, (X2 ? X2 : X) + off + (size_t)b0 * kLdT, kTileBytes, fullb);
        if (++ch == ch1) { ch = ch0; P++; }
      }
    }
    return;
  }

  // ===================== consumer warpgroups =====================
  reg_inc<kConsumerRegs>();
  const int sp = w & 3, hh = w >> 2;                 // SM sub-partition, first/second warp of the pair
  double* Kp = Kpart_s + (size_t)g * split_stride;
  double* red = smem;                                // reused after the main loop
  Syrk2Consumer q{sA, one_operand ? sA : sB, full0, empty0, nchunks, ch0, ch1, c0, c1, kTileDoubles, 0, 0, 0, sgn};
  if (!diag && a0 + 8 * WM >= nao) {
    // half-height tile of the last tile row: the rows of the lower block row (bm = 1) lie past the basis, so the two
    // sub-partitions of a block column share the upper block 4-way: warp (sp, hh) takes the k4 steps
    // (sp & 1) + 2 hh mod 4 of block (0, bn), bn = sp >> 1; half the DMMAs of a full tile on every sub-partition
    const int bn = sp >> 1, part = (sp & 1) + 2 * hh;
    q.row0 = 0; q.col0 = bn * 8 * WM; q.kidx = part;
    double acc[WM][WM][2];
    syrk2_mainloop<WM, false, 4>(q, l, acc);
    consumer_bar_sync();
    if (part != 0) syrk2_put<WM, false>(red, 3 * bn + part - 1, l, acc);
    consumer_bar_sync();
    if (part == 0) {
      syrk2_add<WM, false>(red, 3 * bn, l, acc);
      syrk2_add<WM, false>(red, 3 * bn + 1, l, acc);
      syrk2_add<WM, false>(red, 3 * bn + 2, l, acc);
      syrk2_store<WM, false>(Kp, nao, a0, b0 + q.col0, first, l, acc);
    }
  } else if (!diag) {
    // block (bm, bn) = (sp & 1, sp >> 1); pair split-K 2
    q.row0 = (sp & 1) * 8 * WM; q.col0 = (sp >> 1) * 8 * WM; q.kidx = hh;
    double acc[WM][WM][2];
    syrk2_mainloop<WM, false, 2>(q, l, acc);
    consumer_bar_sync();
    if (hh == 1) syrk2_put<WM, false>(red, sp, l, acc);
    consumer_bar_sync();
    if (hh == 0) {
      syrk2_add<WM, false>(red, sp, l, acc);
      syrk2_store<WM, false>(Kp, nao, a0 + q.row0, b0 + q.col0, first, l, acc);
    }
  } else if (sp == 0 || sp == 3) {
    // diagonal blocks (0,0) and (1,1): lower MMA tiles only, pair split-K 2
    q.row0 = q.col0 = (sp == 3) * 8 * WM; q.kidx = hh;
    double acc[WM][WM][2];
    syrk2_mainloop<WM, true, 2>(q, l, acc);
    consumer_bar_sync();
    if (hh == 1) syrk2_put<WM, true>(red, sp, l, acc);
    consumer_bar_sync();
    if (hh == 0) {
      syrk2_add<WM, true>(red, sp, l, acc);
      syrk2_store<WM, true>(Kp, nao, a0 + q.row0, b0 + q.col0, first, l, acc);
    }
  } else {
    // block (1,0), shared 4-way by the warps of sub-partitions 1 and 2 (the strictly-upper block
    // (0,1) is not computed): warp (sp, hh) takes the k4 steps kk = (sp - 1) + 2 hh mod 4
    q.row0 = 8 * WM; q.col0 = 0; q.kidx = (sp - 1) + 2 * hh;
    double acc[WM][WM][2];
    syrk2_mainloop<WM, false, 4>(q, l, acc);
    const bool owner = (sp == 1 && hh == 0);
    const int slot = (sp == 1) ? 1 : (hh == 0 ? 2 : 4);      // partners: w=5 -> 1, w=2 -> 2, w=6 -> 4
    consumer_bar_sync();
    if (!owner) syrk2_put<WM, false>(red, slot, l, acc);
    consumer_bar_sync();
    if (owner) {
      syrk2_add<WM, false>(red, 1, l, acc);
      syrk2_add<WM, false>(red, 2, l, acc);
      syrk2_add<WM, false>(red, 4, l, acc);
      syrk2_store<WM, false>(Kp, nao, a0 + q.row0, b0 + q.col0, first, l, acc);
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
static size_t ht_smem_bytes(int wn) { return (size_t)ht_stages(wn) * (kHtATile + 16 * wn * kHtLd) * sizeof(double); }
static size_t syrk_smem_bytes(int wm) { return (size_t)kStages * 2 * (16 * wm * kLdT) * sizeof(double); }

template <int WN, int EPI, bool PAIR>
static cudaError_t launch_ht_p(int device, int grid, cudaStream_t st, const HtParams& a) {
  static std::atomic<unsigned long long> attr_done{0};   // per instantiation, one bit per device
  cudaError_t e = ensure_dyn_smem(k_half_transform<WN, EPI, PAIR>, ht_smem_bytes(WN), device, attr_done);
  if (e != cudaSuccess) return e;
  k_half_transform<WN, EPI, PAIR><<<grid, kThreads, ht_smem_bytes(WN), st>>>(a);
  return cudaSuccess;
}

// the packed-piece variant exists for the k-tiled epilogues (JK path, density-matrix form); row-major X (AO2MO) has none
template <int WN, int EPI>
static cudaError_t launch_ht(int device, int grid, cudaStream_t st, const HtParams& a) {
  if (EPI != 2 && a.pair_last) return launch_ht_p<WN, EPI, EPI != 2>(device, grid, st, a);
  return launch_ht_p<WN, EPI, false>(device, grid, st, a);
}

template <int EPI>
static cudaError_t dispatch_ht_wn(int device, int wn, int grid, cudaStream_t st, const HtParams& a) {
  switch (wn) {
#define DFJK_HT_CASE(N) \
  case N: return launch_ht<N, EPI>(device, grid, st, a);
    DFJK_HT_CASE(1) DFJK_HT_CASE(2) DFJK_HT_CASE(3) DFJK_HT_CASE(4) DFJK_HT_CASE(5) DFJK_HT_CASE(6)
    DFJK_HT_CASE(7) DFJK_HT_CASE(8) DFJK_HT_CASE(9) DFJK_HT_CASE(10) DFJK_HT_CASE(11) DFJK_HT_CASE(12)
    DFJK_HT_CASE(13) DFJK_HT_CASE(14) DFJK_HT_CASE(15) DFJK_HT_CASE(16) DFJK_HT_CASE(17) DFJK_HT_CASE(18)
    DFJK_HT_CASE(19) DFJK_HT_CASE(20) DFJK_HT_CASE(21) DFJK_HT_CASE(22)
#undef DFJK_HT_CASE
    default: return cudaErrorInvalidValue;
  }
}

// pieces (16 rows) in the last 64-row block when it is part-empty and the re-tiled copy exists: packed tiles (HtParams::pair_last)
static int ht_pair_last(const dfjk_ctx* h) { return h->Bt != nullptr && (h->nao & 63) >= 1 && (h->nao & 63) <= 48 ? ((h->nao & 63) + 15) >> 4 : 0; }

// epi: 0 = k-tiled X, 1 = k-tiled X + rho partials, 2 = row-major X
static cudaError_t dispatch_ht(int device, int wn, int epi, int grid, cudaStream_t st, const HtParams& a) {
  switch (epi) {
    case 0: return dispatch_ht_wn<0>(device, wn, grid, st, a);
    case 1: return dispatch_ht_wn<1>(device, wn, grid, st, a);
    case 2: return dispatch_ht_wn<2>(device, wn, grid, st, a);
    default: return cudaErrorInvalidValue;
  }
}

struct SyrkArgs {
  const double* X; int nao, nch, mu_pad, nsets; SyrkSets sets; int nrows_blk, rows_per_split, ntiles_m; double* Kpart;
  size_t split_stride; int first;
  const double* X2 = nullptr;   // k_syrk2 only: column operand of the two-operand form
  const unsigned int* sgn = nullptr;   // sign bits of the occupations (C-form), nullptr for the two-operand form
};

template <int WM>
static cudaError_t launch_syrk2(int device, int ksplit, cudaStream_t st, const SyrkArgs& a) {
  static std::atomic<unsigned long long> attr_done{0};
  cudaError_t e = ensure_dyn_smem(k_syrk2<WM>, syrk_smem_bytes(WM), device, attr_done);
  if (e != cudaSuccess) return e;
  const dim3 grid(a.ntiles_m * (a.ntiles_m + 1) / 2 * ksplit, a.nsets);
  k_syrk2<WM><<<grid, kThreads, syrk_smem_bytes(WM), st>>>(a.X, a.X2, a.sgn, a.nao, a.nch, a.mu_pad, a.sets, a.nrows_blk,
                                                         a.rows_per_split, a.ntiles_m, ksplit, a.Kpart,
                                                         a.split_stride, a.first);
  return cudaSuccess;
}

static cudaError_t dispatch_syrk2(int device, int wm, int ksplit, cudaStream_t st, const SyrkArgs& a) {
  switch (wm) {
    case 4: return launch_syrk2<4>(device, ksplit, st, a);
    case 5: return launch_syrk2<5>(device, ksplit, st, a);
    case 6: return launch_syrk2<6>(device, ksplit, st, a);
    case 7: return launch_syrk2<7>(device, ksplit, st, a);
    default: return cudaErrorInvalidValue;
  }
}

// Eq. 18 for AO2MO: X[pl][mu][n] = sum_lam B_{p_first+pl}[mu][lam] C'[lam][n], row-major with row
// stride ldx (the same kernel as the JK half-transform, epilogue 2).  Returns 0 on success.
int launch_half_transform_rowmajor(dfjk_ctx* h, const SetInfo& si, int p_first, int nb, double* X, int ldx,
                                   cudaStream_t st) {
  const int n8 = si.nocc_pad / 8;
  const int ntn = cdiv(n8, 2 * kHtMaxWN), wn = cdiv(n8, 2 * ntn);
  const int ntm_ht = cdiv(h->nao, 64);
  HtParams a;
  a.Bt = h->Bt; a.bt_pstride = h->bt_pstride; a.pair_last = ht_pair_last(h); a.Bp = h->B; a.npair = h->npair; a.nao = h->nao; a.Ct = h->Ct; a.ct_rows = h->ct_rows; a.nocc_pad = si.nocc_pad;
  a.X = X; a.nch = 0; a.mu_pad = 0; a.p_first = p_first; a.nb = nb; a.ntm = ntm_ht; a.ntn = ntn;
  a.rho_ht = nullptr; a.nset = 0; a.ldx = ldx; a.xrows = h->nao; a.sgnbits = nullptr; a.pair_last = 0;
  a.col0[0] = 0;
  const long long ht_tiles = (long long)nb * ntm_ht * ntn;
  const long long ht_slots = (long long)h->ht_grid * ht_ctas_per_sm(wn);   // persistent: one or two CTAs per SM
  const int ht_grid = (int)(ht_tiles < ht_slots ? ht_tiles : ht_slots);
  return dispatch_ht(h->device, wn, 2, ht_grid, st, a) == cudaSuccess ? 0 : -1;
}

// Modelled SYRK time of one aux block in units of one off-diagonal CTA's aux row: greedy list
// schedule of the CTAs in launch order (off-diagonal first, then the cheaper diagonal ones) on
// `sms` SMs, one CTA per SM.
static double syrk_makespan(int n_off, int n_diag, double diag_cost, int ksplit, int rps, int sms) {
  const long long total = (long long)(n_off + n_diag) * ksplit;
  const double work = ((double)n_off + diag_cost * n_diag) * ksplit * rps;
  if (total > 8192 || total <= sms) return total <= sms ? (double)rps * (n_off ? 1.0 : diag_cost) : work / sms + rps;
  std::priority_queue<double, std::vector<double>, std::greater<double>> free_at;
  for (int i = 0; i < sms; i++) free_at.push(0.0);
  double end = 0.0;
  for (long long i = 0; i < total; i++) {
    const double c = (i < (long long)n_off * ksplit ? 1.0 : diag_cost) * rps;
    const double t = free_at.top() + c;
    free_at.pop();
    free_at.push(t);
    if (t > end) end = t;
  }
  return end;
}

// SYRK tile T = 16 * WM, WM in {4, 5, 6, 7}: the least modelled work over the lower triangle (ties -> the larger
// tile); a diagonal CTA costs (WM + 1) / (2 WM) of an off-diagonal one, a half-height one 1/2
static int pick_syrk_tile(int nao) {
  int wm = 7;
  double best = 1e300;
  for (int wmc = 7; wmc >= 4; wmc--) {
    const int T = 16 * wmc, nt = cdiv(nao, T);
    // the off-diagonal tiles of the last tile row cost half when at most T / 2 of its rows exist
    const bool half_last = nao - (nt - 1) * T <= T / 2;
    const double n_off = 0.5 * nt * (nt - 1) - (half_last ? 0.5 * (nt - 1) : 0.0);
    const double area = (n_off + (wmc + 1) / (2.0 * wmc) * nt) * (double)T * T;
    if (area < best * 0.995) { best = area; wm = wmc; }
  }
  return wm;
}

// Split-K factor of the SYRK for blocks of nblk aux rows: the split with the shortest modelled
// makespan (one CTA per SM), 0.2 % per split for the extra partial tiles; remembered in the handle
// because the model costs a few thousand heap operations.
static int pick_ksplit(dfjk_ctx* h, int nblk, int ntiles, int ntm, double diag_cost) {
  int ksplit = h->ksplit_forced;
  if (ksplit <= 0) {
    if (h->ks_cache_val > 0 && h->ks_cache_nblk == nblk && h->ks_cache_ntiles == ntiles) return h->ks_cache_val;
    double best = 1e300;
    ksplit = 1;
    for (int k = 1; k <= h->ksplit && k <= nblk; k++) {
      const int rps = cdiv(nblk, k);
      if (cdiv(nblk, rps) != k) continue;                       // splits that actually get rows
      const double t = syrk_makespan(ntiles - ntm, ntm, diag_cost, k, rps, h->num_sms) * (1.0 + 0.002 * k);
      if (t < best) { best = t; ksplit = k; }
    }
    h->ks_cache_nblk = nblk; h->ks_cache_ntiles = ntiles; h->ks_cache_val = ksplit;
  }
  if (ksplit > h->ksplit) ksplit = h->ksplit;
  if (ksplit > nblk) ksplit = nblk;
  return ksplit < 1 ? 1 : ksplit;
}

// Rows per aux block under a cap: the fewest blocks that fit, made equal (no short last block: 3 x 1122 + 634 rows at
// `large` become 4 x 1000), then up to 15 rows more per block if that saves a round of half-transform tiles over the
// persistent grid (1002, 1002, 1002, 994 rows: 127 + 127 + 127 + 126 rounds of 148 tiles, the minimum, not 4 x 127)
static long long pick_block_rows(const dfjk_ctx* h, long long cap, int naux, int ntm_ht, int ntn, int wn) {
  const long long nblocks = cdiv_ll(naux, cap), slots = (long long)h->ht_grid * ht_ctas_per_sm(wn);
  const int v = ht_pair_last(h);
  auto tiles = [&](long long nb) { return v ? (nb * (ntm_ht - 1) + ((nb * v + 3) >> 2)) * ntn : nb * ntm_ht * ntn; };
  const long long bal = cdiv_ll(naux, nblocks);
  long long best_nb = bal, best_rounds = -1;
  for (long long nb = bal; nb <= cap && nb < bal + 16; nb++) {
    const long long last = naux - (nblocks - 1) * nb;
    if (last < 1) break;
    const long long rounds = (nblocks - 1) * cdiv_ll(tiles(nb), slots) + cdiv_ll(tiles(last), slots);
    if (best_rounds < 0 || rounds < best_rounds) { best_rounds = rounds; best_nb = nb; }
  }
  return best_nb;
}

// Aux-block scheduler: cap the X workspace, pick the split-K factor, enqueue
// half-transform and SYRK block after block on one stream.  No allocation, no host sync.
// With want_rho the half-transform also produces rho (step a2 fused): the
// caller then runs J pass 2 only.
int launch_k_path(dfjk_ctx* h, const SetInfo& si, double* K_out, bool want_rho, cudaStream_t st) {
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
  const int nch = cdiv(ldx, kBK);
  const size_t row_doubles = (size_t)nch * h->mu_pad * kLdT;     // tiled X, one aux row
  // opt-in FP64 emulation of the SYRK on the int8 tensor cores: the block also holds the sliced X
  const bool emu = h->k_emu_slices > 0;
  int emu_nchs = 0;
  for (int s = 0; s < si.nset; s++) {
    const int c0 = si.col0[s], c1 = c0 + si.nocc[s];
    if (c1 > c0 && ((c1 + 31) >> 5) - (c0 >> 5) > emu_nchs) emu_nchs = ((c1 + 31) >> 5) - (c0 >> 5);
  }
  // the int32 accumulators of one scale group take pgroup * columns products of at most 64 * 64, S of them
  // per accumulator: the group must stay below 2^31
  if (emu && (double)h->k_emu_pgroup * 32.0 * emu_nchs * 4096.0 * h->k_emu_slices >= 2147483648.0) return -2;
  const size_t emu_row_bytes = emu ? emu_bytes_per_aux_row(nao, emu_nchs, h->k_emu_slices, h->k_emu_pgroup) : 0;
  long long nblk = (long long)((h->X_doubles * sizeof(double) - (emu ? 4096 : 0)) / (row_doubles * sizeof(double) + emu_row_bytes));
  if (h->nblk_forced > 0 && nblk > h->nblk_forced) nblk = h->nblk_forced;
  if (nblk > naux) nblk = naux;
  if (nblk > 32768) nblk = 32768;
  if (nblk < 1) { if (emu) return -2; nblk = 1; }
  const int n8 = ldx / 8;
  const int ntn = cdiv(n8, 2 * kHtMaxWN), wn = cdiv(n8, 2 * ntn);  // N tile = 16*wn columns
  const int ntm_ht = cdiv(nao, 64);
  if (!emu && h->nblk_forced <= 0) nblk = pick_block_rows(h, nblk, naux, ntm_ht, ntn, wn);
  const int wm_s = pick_syrk_tile(nao);
  const double diag_cost = (wm_s + 1) / (2.0 * wm_s);
  const int ntm = cdiv(nao, 16 * wm_s), ntiles = ntm * (ntm + 1) / 2;
  const int ksplit = emu ? emu_pick_ksplit(nao, cdiv((int)nblk, h->k_emu_pgroup), h->ksplit, h->num_sms)
                         : pick_ksplit(h, (int)nblk, ntiles, ntm, diag_cost);
  const size_t split_stride = (size_t)h->max_nset * n2;
  // emulated SYRK: int8 slices and scales behind the fp64 block
  signed char* emu_xq = nullptr;
  double* emu_scale = nullptr;
  if (emu) {
    uintptr_t a = (uintptr_t)(h->X + (size_t)nblk * row_doubles);
    a = (a + 255) & ~(uintptr_t)255;
    emu_xq = (signed char*)a;
    a += (size_t)nblk * emu_nchs * h->k_emu_slices * (size_t)emu_mu_q(nao) * 32;
    a = (a + 255) & ~(uintptr_t)255;
    emu_scale = (double*)a;
  }

  const bool emu_ht = h->ht_emu_slices > 0;
  const bool thin = !emu && !emu_ht && si.nset == 1 && ldx == 8 && symm_thin_ok(h, si.nocc[0]);
  if (emu_ht) {
    prof_mark(h, DFJK_PHASE_PREP, st);
    launches += launch_emu_slice_ct(h, ldx, st);
  }

  int nblocks = 0;
  for (int p0 = 0; p0 < naux; p0 += (int)nblk, nblocks++) {
    const int nb = (int)(naux - p0 < nblk ? naux - p0 : nblk);
    prof_mark(h, DFJK_PHASE_HALF_TRANSFORM, st);
    HtParams a;
    a.Bt = h->Bt; a.bt_pstride = h->bt_pstride; a.pair_last = ht_pair_last(h); a.Bp = h->B; a.npair = h->npair; a.nao = nao; a.Ct = h->Ct; a.ct_rows = h->ct_rows; a.nocc_pad = ldx;
    a.X = h->X; a.nch = nch; a.mu_pad = h->mu_pad; a.p_first = p0; a.nb = nb; a.ntm = ntm_ht; a.ntn = ntn;
    a.rho_ht = h->rho_ht; a.nset = si.nset; a.ldx = 0; a.xrows = 0; a.sgnbits = h->sgnbits;
    for (int s = 0; s <= si.nset; s++) a.col0[s] = si.col0[s];
    const long long ht_tiles = (long long)nb * ntm_ht * ntn;
    const long long ht_slots = (long long)h->ht_grid * ht_ctas_per_sm(wn);   // persistent: one or two CTAs per SM
  const int ht_grid = (int)(ht_tiles < ht_slots ? ht_tiles : ht_slots);
    if (thin) {
      // one set of at most 8 columns: one pass over the packed triangle (symm.cu), rho written directly
      if (launch_symm_thin_jk(h, si.nocc[0], p0, nb, h->X, want_rho ? h->rho : nullptr, st) != 0) return -1;
    } else if (emu_ht) {
      if (launch_emu_ht(h, ldx, p0, nb, h->X, nch, st) < 0) return -1;
    } else if (dispatch_ht(h->device, wn, want_rho ? 1 : 0, ht_grid, st, a) != cudaSuccess) {
      return -1;
    }
    launches++;
    const int rps = cdiv(nb, ksplit);
    prof_mark(h, DFJK_PHASE_SYRK, st);
    if (emu) {
      for (int s = 0; s < si.nset; s++) {
        if (si.col0[s + 1] == si.col0[s]) continue;
        const int k = launch_emu_syrk_set(h, h->X, nch, si.col0[s], si.col0[s] + si.nocc[s], nb, emu_xq, emu_scale,
                                          h->Kpart + n2 * s, split_stride, ksplit, p0 == 0 ? 1 : 0, st);
        if (k < 0) return -1;
        launches += k;
      }
    } else {
      // all sets in ONE launch (grid.y): the widest first, the thin ones (rank-8 fragment sets) fill its tail.
      // Columns past nocc[s] (padding to the 8-column MMA tile) are zero: stop at the k4 step
      SyrkArgs sa{h->X, nao, nch, h->mu_pad, 0, {}, nb, rps, ntm, h->Kpart, split_stride, p0 == 0 ? 1 : 0};
      int order[kMaxSets];
      for (int s = 0; s < si.nset; s++)
        if (si.col0[s + 1] != si.col0[s]) order[sa.nsets++] = s;
      std::stable_sort(order, order + sa.nsets, [&](int a, int b) { return si.nocc[a] > si.nocc[b]; });
      for (int q = 0; q < sa.nsets; q++) {
        const int s = order[q];
        sa.sets.c0[q] = si.col0[s];
        sa.sets.c1[q] = si.col0[s] + round_up(si.nocc[s], 4);
        sa.sets.koff[q] = (long long)(n2 * s);
      }
      sa.sgn = h->sgnbits;
      if (dispatch_syrk2(h->device, wm_s, ksplit, st, sa) != cudaSuccess) return -1;
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
  if (want_rho && !thin) {
    prof_mark(h, DFJK_PHASE_J1, st);
    dim3 gr(cdiv(naux, 128), si.nset);
    k_rho_reduce<<<gr, 128, 0, st>>>(h->rho_ht, ntm_ht * ntn * 8, si.nset, naux, h->rho);
    launches++;
  }
  h->plan_nblk = (int)nblk;
  h->plan_ksplit = ksplit;
  h->plan_nblocks = nblocks;
  return launches;
}

// ------------------------------------------------------------------ density-matrix form (Eq. 16-17 as printed)
// K = sum_P (B_P D) B_P for a general symmetric D (it need not be positive semidefinite, so no
// C sqrt(occ) factor exists): Eq. 16 is the half-transform with C' = D (nao columns), Eq. 17 the
// two-operand form of k_syrk2 against the unpacked slice.
// The unpacked slice is written in the same k-tiled layout as X ("unpacked to the square-matrix
// form"): X2[P][sigma/32][nu][sigma%32] = B_P[nu][sigma], zero past nao.
__global__ void __launch_bounds__(256)
k_unpack_tiled(const double* __restrict__ Bp, size_t npair, int nao, int p_first, int nch, int mu_pad,
               double* __restrict__ X2) {
  const int pl = blockIdx.y, ch = blockIdx.x;
  const double* BpP = Bp + (size_t)(p_first + pl) * npair;
  double* dst = X2 + ((size_t)pl * nch + ch) * mu_pad * kLdT;
  for (int e = threadIdx.x; e < nao * 32; e += 256) {
    const int nu = e >> 5, k = e & 31, sg = ch * 32 + k;
    double v = 0.0;
    if (sg < nao) v = BpP[sg <= nu ? tri(nu) + sg : tri(sg) + nu];
    dst[(size_t)nu * kLdT + k] = v;
  }
}

// Dw[pair] = (2 - delta) (D[mu][nu] + D[nu][mu]) / 2 from a full square density
__global__ void k_prep_dw_dm(const double* __restrict__ D, int nao, size_t npair, double* __restrict__ Dw) {
  const int s = blockIdx.y;
  const double* Ds = D + (size_t)s * nao * nao;
  for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < (size_t)nao * nao; e += (size_t)gridDim.x * blockDim.x) {
    const int mu = (int)(e / nao), nu = (int)(e % nao);
    if (nu <= mu) Dw[(size_t)s * npair + tri(mu) + nu] = (mu == nu) ? Ds[e] : (Ds[e] + Ds[(size_t)nu * nao + mu]);
  }
}

int launch_prep_dw_dm(dfjk_ctx* h, int nset, const double* D, cudaStream_t st) {
  prof_mark(h, DFJK_PHASE_PREP, st);
  dim3 grid(592, nset);
  k_prep_dw_dm<<<grid, 256, 0, st>>>(D, h->nao, h->npair, h->Dw);
  return 1;
}

int launch_k_path_dm(dfjk_ctx* h, int nset, const double* D, double* K_out, cudaStream_t st) {
  int launches = 0;
  const int nao = h->nao, naux = h->naux;
  const size_t n2 = (size_t)nao * nao;
  if (naux == 0) {
    prof_mark(h, DFJK_PHASE_K_EPILOGUE, st);
    k_zero<<<148, 256, 0, st>>>(K_out, n2 * nset);
    return 1;
  }
  SetInfo si;
  si.nset = 1; si.col0[0] = 0; si.nocc[0] = nao; si.coff[0] = 0; si.ooff[0] = 0;
  si.col0[1] = si.nocc_pad = round_up(nao, 8);
  if (si.nocc_pad > h->nocc_pad_cap) return -2;
  const int ldx = si.nocc_pad, nch = cdiv(ldx, kBK);
  const size_t row_doubles = (size_t)nch * h->mu_pad * kLdT;
  long long nblk = (long long)(h->X_doubles / (2 * row_doubles));     // X = B_P D and the unpacked slice
  if (h->nblk_forced > 0 && nblk > h->nblk_forced) nblk = h->nblk_forced;
  if (nblk > naux) nblk = naux;
  if (nblk > 32768) nblk = 32768;
  if (nblk < 1) return -2;
  const int n8 = ldx / 8;
  const int ntn = cdiv(n8, 2 * kHtMaxWN), wn = cdiv(n8, 2 * ntn);
  const int ntm_ht = cdiv(nao, 64);
  if (h->nblk_forced <= 0) nblk = pick_block_rows(h, nblk, naux, ntm_ht, ntn, wn);
  double* X1 = h->X;
  double* X2 = h->X + (size_t)nblk * row_doubles;
  const int wm_s = pick_syrk_tile(nao);
  const double diag_cost = (wm_s + 1) / (2.0 * wm_s);
  const int ntm = cdiv(nao, 16 * wm_s), ntiles = ntm * (ntm + 1) / 2;
  const int ksplit = pick_ksplit(h, (int)nblk, ntiles, ntm, diag_cost);
  const size_t split_stride = (size_t)h->max_nset * n2;
  const int nb32 = cdiv(nao, 32);
  for (int s = 0; s < nset; s++) {
    SetInfo sj = si;
    launches += launch_prep_ct(h, sj, D + n2 * s, nullptr, st);         // C' = D_s
    for (int p0 = 0; p0 < naux; p0 += (int)nblk) {
      const int nb = (int)(naux - p0 < nblk ? naux - p0 : nblk);
      prof_mark(h, DFJK_PHASE_HALF_TRANSFORM, st);
      HtParams a;
      a.Bt = h->Bt; a.bt_pstride = h->bt_pstride; a.pair_last = ht_pair_last(h); a.Bp = h->B; a.npair = h->npair; a.nao = nao; a.Ct = h->Ct; a.ct_rows = h->ct_rows; a.nocc_pad = ldx;
      a.X = X1; a.nch = nch; a.mu_pad = h->mu_pad; a.p_first = p0; a.nb = nb; a.ntm = ntm_ht; a.ntn = ntn;
      a.rho_ht = nullptr; a.nset = 0; a.ldx = 0; a.xrows = 0; a.col0[0] = 0; a.sgnbits = nullptr;
      const long long ht_tiles = (long long)nb * ntm_ht * ntn;
      const long long ht_slots = (long long)h->ht_grid * ht_ctas_per_sm(wn);
      if (dispatch_ht(h->device, wn, 0, (int)(ht_tiles < ht_slots ? ht_tiles : ht_slots), st, a) != cudaSuccess) return -1;
      dim3 gu(nch, nb);
      k_unpack_tiled<<<gu, 256, 0, st>>>(h->B, h->npair, nao, p0, nch, h->mu_pad, X2);
      launches += 2;
      prof_mark(h, DFJK_PHASE_SYRK, st);
      SyrkArgs sa{X1, nao, nch, h->mu_pad, 1, {}, nb, cdiv(nb, ksplit), ntm, h->Kpart, split_stride, p0 == 0 ? 1 : 0, X2};
      sa.sets.c0[0] = 0; sa.sets.c1[0] = round_up(nao, 4); sa.sets.koff[0] = (long long)(n2 * s);
      if (dispatch_syrk2(h->device, wm_s, ksplit, st, sa) != cudaSuccess) return -1;
      launches++;
    }
    prof_mark(h, DFJK_PHASE_K_EPILOGUE, st);
    dim3 ge(nb32, nb32, 1), be(32, 8);
    k_k_epilogue<<<ge, be, 0, st>>>(h->Kpart + n2 * s, ksplit, split_stride, nao, K_out + n2 * s);
    launches++;
  }
  h->plan_nblk = (int)nblk;
  h->plan_ksplit = ksplit;
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
