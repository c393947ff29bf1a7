// One-pass symmetric thin half-transform on the packed triangle:
//   Z[P][mu][a] = sum_lam b^P[mu][lam] M[lam][a],   a < 8      (Eq. 16 / Eq. 18)
// for a thin right-hand side (AO2MO's active columns, Eq. 18-19 of the "active first" route).  With 8
// columns the operation is HBM-bound (16 flop per stored element): the packed tensor must be streamed
// ONCE, as stored, and every stored element b^P[mu][lam], lam < mu, must serve both
// Z[mu] += b M[lam] and Z[lam] += b M[mu].
//
// A CTA owns one aux row P at a time (persistent over P).  The packed row is walked in super-groups
// of 8 G matrix rows x chunks of LC columns; one stage of the mbarrier ring holds such a piece, each
// matrix row of it fetched by ONE bulk async copy (TMA engine, UBLKCP) issued by a lane of one of the
// four producer warps.  Packed rows start at 8-byte granularity: a row whose first element sits at an
// odd index is over-fetched by one element in front (and/or one behind), so that source, destination
// and size stay 16-byte multiples; the consumers add that parity bit to their shared-memory offset.
// The 8 rows of a row group land in shared memory in the order (0,3,4,7,1,2,5,6): tri(mu) is even
// for mu % 4 in {0,3} and odd otherwise, so each half of that order has ONE parity, and with a slot
// stride of 4 mod 16 doubles both fragment patterns below are bank-conflict free.
//
// Consumer warp w owns the 8-column blocks Jb = w mod NW of the matrix.  For a stored 8 x 8 block
// (row group I, column block Jb < I) it issues four DMMA.8x8x4:
//   direct      Zd[I]  += T   (8 x 8)  M[8 Jb ..]      (A fragment: lane (r, j) reads T[r][4h + j])
//   transposed  Zt[Jb] += T^T (8 x 8)  M[8 I ..]       (A fragment: lane (r, j) reads T[rows(g)[j]][r])
// Zt (all the warp's blocks of a panel of 1280 columns: 20 accumulator tiles with 8 warps) lives in registers
// for the whole aux row (a larger basis takes one launch per panel, SymmParams::cb0); the B fragments of the direct products (rows of M of the warp's own column
// blocks) sit in shared memory as ready fragment pairs (or in registers, MREG); the B fragments of
// the transposed products (rows of M of the current row group) are loaded one super-group ahead.
// The direct accumulators Zd are partial over the warp's column blocks: after every super-group the
// warps pass them through shared memory and the owner of row group I (warp I mod NW) adds them, in
// fixed order, to its Zt tile -- no atomics, bitwise deterministic.  The diagonal block (I, I) is
// handled by its owner with masks (direct: lam <= mu; transposed: lam < mu).
// Algorithmic bytes: the packed row once (npair * 8) + Z (nao * 8 * 8) per aux row; 4 DMMA per 64
// stored elements, i.e. the FP64 tensor pipe would be 75 % busy at the full HBM rate.
#include "common.cuh"
#include "ctx.h"
#include "pipeline.cuh"

namespace dfjk {

constexpr int kSyMaxNao = 1280;                 // 20 register-resident accumulator tiles per warp

// G row groups (8 rows) per super-group, LC columns per stage, STAGES ring slots
template <int NW, int G, int LC, int STAGES, bool MREG>
struct SyCfg {
  static constexpr int kThreads = 32 * NW + 128;  // NW consumer warps + 4 producer warps
  static constexpr int kNSLOT = kSyMaxNao / (8 * NW);   // column blocks per warp
  static constexpr int kConsRegs = NW == 8 ? 232 : 104; // setmaxnreg budgets (the producers keep 40): NW 16 -> 96 * 640 registers at launch >= 104 * 512 + 40 * 128
  static constexpr int kRows = 8 * G;             // matrix rows per stage
  static constexpr int kS = LC + 4;               // slot stride in doubles (4 mod 16)
  static constexpr int kStageDoubles = kRows * kS;
  static constexpr int kNCH = kSyMaxNao / LC;     // chunks per matrix row
  static constexpr int kQ = LC / (8 * NW);        // column blocks per warp and chunk
  static constexpr int kZdDoubles = 2 * NW * G * 64;  // double-buffered partial direct tiles of the NW warps
  // MREG: the B fragments of a warp's own column blocks stay in registers (80 of them); otherwise they sit in
  // shared memory as ready fragment pairs, [column block][lane][h], one conflict-free LDS.128 per block
  static constexpr int kMpDoubles = MREG ? 0 : (kSyMaxNao / 8) * 64;
  static constexpr size_t kSmemBytes = (size_t)(STAGES * kStageDoubles + kZdDoubles + kMpDoubles) * sizeof(double);
  static_assert(LC % (8 * G) == 0 && LC % (8 * NW) == 0 && kSyMaxNao % LC == 0, "chunk shape");
  static_assert(NW == 8 || NW == 16, "consumer warps");
  static_assert(!MREG || NW == 8, "register-resident B fragments need the 232-register budget");
  static_assert((8 * G) % 4 == 0, "rows are split over four producer warps");
};

// fragment row f of a row group holds matrix row perm(f): (0,3,4,7 | 1,2,5,6)
__device__ __forceinline__ int sy_perm(int f) { return (int)((0x65217430u >> (4 * f)) & 7u); }
__device__ __forceinline__ int sy_invperm(int a) { return (int)((0x37621540u >> (4 * a)) & 7u); }

struct SymmParams {
  const double* Bp; size_t npair; size_t b_elems;   // packed tensor (16-byte aligned), elements it holds
  int nao;
  // right-hand side, element (lam, a), a < ncols <= 8, at M[(lam >> m_sh) * m_hi + (lam & m_msk) * m_lo + a * m_a]:
  // row-major M[lam * ldm + a] (AO2MO), or the k-tiled C'^T of k_prep_ct (JK call on one thin set)
  const double* M; int ncols; int m_sh, m_msk; long long m_hi, m_lo, m_a;
  double* X; long long x_pstride, x_rstride;        // out: X[pl * x_pstride + mu * x_rstride + a], a < 8 (strides even)
  int p_first, nb;                                  // aux rows [p_first, p_first + nb)
  double* rho; const unsigned int* sgn;             // optional: rho[p_first + pl] = sum_{mu, a} sign_a Z[mu][a] M[mu][a] (Eq. 14, R16)
  // column panel of this launch: the column blocks [cb0, cb0 + 160) (1280 columns: what a warp's register-resident
  // accumulators cover).  A basis beyond 1280 takes one launch per panel, in ascending order on one stream; panel 0
  // writes every row of Z (rows past its columns: the direct sums alone), later panels add to it
  int cb0;
};

__device__ __forceinline__ double sy_m(const SymmParams& q, int lam, int a) {
  return __ldg(q.M + (size_t)(lam >> q.m_sh) * q.m_hi + (size_t)(lam & q.m_msk) * q.m_lo + (size_t)a * q.m_a);
}

// PANELS: the basis needs more than one column panel (cb0 may be nonzero, outputs may be added to); RHO: rho is
// wanted.  Both are compile-time so that the common single-panel AO2MO instance keeps its hot loop small (the
// unrolled chunk loop is instruction-cache sensitive: 2800 vs 4100 instructions made 4.3 vs 4.8 ms)
template <int NW, int G, int LC, int STAGES, bool MREG, bool PANELS, bool RHO>
__global__ void __launch_bounds__(32 * NW + 128, 1)
k_symm_thin(const __grid_constant__ SymmParams q) {
  using Cfg = SyCfg<NW, G, LC, STAGES, MREG>;
  constexpr int kSyThreads = Cfg::kThreads, kSyNSLOT = Cfg::kNSLOT;
  constexpr int kSyG = G, kSyRows = Cfg::kRows, kSyLC = LC, kSyS = Cfg::kS, kSyStageDoubles = Cfg::kStageDoubles;
  constexpr int kSyStages = STAGES, kSyNCH = Cfg::kNCH, kQ = Cfg::kQ;
  extern __shared__ __align__(128) double smem[];
  double* ring = smem;                                  // kSyStages x kSyStageDoubles
  double* zd = smem + kSyStages * kSyStageDoubles;      // [2][8][kSyG][64]
  double* Mp = zd + Cfg::kZdDoubles;                    // !MREG: [column block][lane][h] = M[8 Jb + 4h + j][r]
  __shared__ __align__(8) unsigned long long bars[2 * kSyStages];
  __shared__ double rho_red[NW];
  const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[kSyStages]);
  const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
  const int nao = q.nao;
  const int nsg = (nao + kSyRows - 1) / kSyRows;
  const int ngroups = (nao + 7) >> 3;
  const int cb0 = PANELS ? q.cb0 : 0, col_base = 8 * cb0;   // first column block / column of this panel
  const int sg0 = col_base / kSyRows;                  // rows above the panel's first column hold none of its columns
  const bool first_panel = !PANELS || cb0 == 0;
  constexpr int kPanelBlocks = kSyMaxNao / 8;

  for (int e = tid; e < kSyStages * kSyStageDoubles; e += kSyThreads) ring[e] = 0.0;   // stale slots must hold finite numbers
  if (!MREG)
    for (int e = tid; e < Cfg::kMpDoubles; e += kSyThreads) {
      const int h = e & 1, ln = (e >> 1) & 31, lam = col_base + 8 * (e >> 6) + 4 * h + (ln & 3), a = ln >> 2;
      Mp[e] = (a < q.ncols && lam < nao) ? sy_m(q, lam, a) : 0.0;
    }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  if (tid == 0) {
    for (int s = 0; s < kSyStages; s++) {
      mbar_init(full0 + 8 * s, 4);         // one expect_tx arrival per producer warp
      mbar_init(empty0 + 8 * s, NW);       // one arrival per consumer warp
    }
    mbar_fence_init();
  }
  __syncthreads();

  if (w >= NW) {
    // ===================== producer warpgroup: 8G / 4 matrix rows per warp, one per lane =====================
    reg_dec<kProducerRegs>();
    constexpr int kRowsPerWarp = kSyRows / 4;
    const int rr = (w - NW) * kRowsPerWarp + l;             // row inside the super-group (lanes past the share idle)
    const bool lane_on = l < kRowsPerWarp;
    const int gi = rr >> 3, a = rr & 7;
    const int slot = gi * 8 + sy_invperm(a);
    const uint32_t ring_u32 = smem_u32(ring);
    int it = 0;
    for (int pl = blockIdx.x; pl < q.nb; pl += gridDim.x) {
      const size_t rowbase = (size_t)(q.p_first + pl) * q.npair;
      for (int sg = sg0; sg < nsg; sg++) {
        const int mu = sg * kSyRows + rr;
        const int nch = (min(sg * kSyRows + kSyRows, col_base + kSyMaxNao) - col_base + kSyLC - 1) / kSyLC;
        const size_t trimu = tri(mu);
        for (int cc = 0; cc < nch; cc++, it++) {
          const int stage = it % kSyStages;
          const uint32_t fullb = full0 + 8 * stage;
          mbar_wait(empty0 + 8 * stage, ((it / kSyStages) & 1) ^ 1);
          const uint32_t dst = ring_u32 + (uint32_t)(stage * kSyStageDoubles + slot * kSyS) * 8u;
          uint32_t bytes = 0;
          size_t as2 = 0;
          if (lane_on && mu < nao) {
            const int c0 = col_base + cc * kSyLC;          // c0 <= first row of the super-group <= mu: never empty
            const size_t as = rowbase + trimu + c0, ae = rowbase + trimu + min(c0 + kSyLC, mu + 1);
            as2 = as & ~(size_t)1;
            const size_t ae2 = (ae + 1) & ~(size_t)1;
            if (ae2 <= q.b_elems) {
              bytes = (uint32_t)(ae2 - as2) * 8u;
            } else {
              // the last element of an odd-sized tensor: no over-fetch behind it, plain loads instead
              double* d = ring + stage * kSyStageDoubles + slot * kSyS + (int)(as - as2);
              for (size_t i = as; i < ae; i++) d[i - as] = q.Bp[i];
            }
          }
          const uint32_t total = __reduce_add_sync(0xffffffffu, bytes);
          __syncwarp();                                    // plain stores above are ordered before the arrival
          if (l == 0) mbar_arrive_expect_tx(fullb, total);
          __syncwarp();                                    // the barrier is armed before any byte lands
          if (bytes) bulk_g2s(dst, q.Bp + as2, bytes, fullb);
        }
      }
    }
    return;
  }

  // ===================== consumer warpgroups =====================
  reg_inc<Cfg::kConsRegs>();
  const int r = l >> 2, j = l & 3;
  const bool col_ok = r < q.ncols;                      // B-fragment column a = r
  // B fragments of this warp's own column blocks (direct products): M[8 Jb + 4h + j][r]
  double Mf[MREG ? kSyNSLOT : 1][2];
  if (MREG) {
#pragma unroll
    for (int sl = 0; sl < (MREG ? kSyNSLOT : 1); sl++)
#pragma unroll
      for (int h = 0; h < 2; h++) {
        const int lam = col_base + 8 * (NW * sl + w) + 4 * h + j;
        Mf[sl][h] = (col_ok && lam < nao) ? sy_m(q, lam, r) : 0.0;
      }
  }
  const double* Mp_lane = Mp + (w * 32 + l) * 2;         // + 64 NW sl: this warp's column block NW sl + w
  auto get_mf = [&](int sl) -> double2 {
    if (MREG) return make_double2(Mf[MREG ? sl : 0][0], Mf[MREG ? sl : 0][1]);
    return *reinterpret_cast<const double2*>(Mp_lane + 64 * NW * sl);
  };
  const int pr = sy_perm(r);                            // matrix row (within its group) of fragment row r
  int it = 0, sgc = 0;
  for (int pl = blockIdx.x; pl < q.nb; pl += gridDim.x) {
    const int bpar = (int)(((size_t)(q.p_first + pl) * q.npair) & 1);
    // shared-memory offsets inside a row group (doubles), column offset of the warp's block added
    const int offD = r * kSyS + (bpar ^ (r >> 2)) + j + 8 * w;          // direct: T[frag row r][4h + j]
    const int offT0 = j * kSyS + bpar + r + 8 * w;                      // transposed, rows (0,3,4,7)[j]
    const int offT1 = (4 + j) * kSyS + (bpar ^ 1) + r + 8 * w;          // transposed, rows (1,2,5,6)[j]
    double Zt[kSyNSLOT][2];
#pragma unroll
    for (int sl = 0; sl < kSyNSLOT; sl++) Zt[sl][0] = Zt[sl][1] = 0.0;

    // B fragments of the transposed products, M[mu0 + 8 gi + rows(g)[j]][r]: fetched one super-group ahead
    // (they come from L2; a super-group lasts a few thousand cycles)
    auto load_tB = [&](int sgx, double (&dst)[kSyG][2]) {
#pragma unroll
      for (int gi = 0; gi < kSyG; gi++)
#pragma unroll
        for (int g = 0; g < 2; g++) {
          const int mu = sgx * kSyRows + 8 * gi + sy_perm(4 * g + j);
          dst[gi][g] = (col_ok && mu < nao) ? sy_m(q, mu, r) : 0.0;
        }
    };
    double tB[kSyG][2], tBn[kSyG][2];
    load_tB(sg0, tBn);
    for (int sg = sg0; sg < nsg; sg++, sgc++) {
      const int mu0 = sg * kSyRows;
      const int nch = (min(mu0 + kSyRows, col_base + kSyMaxNao) - col_base + kSyLC - 1) / kSyLC;
#pragma unroll
      for (int gi = 0; gi < kSyG; gi++) { tB[gi][0] = tBn[gi][0]; tB[gi][1] = tBn[gi][1]; }
      load_tB(sg + 1, tBn);                              // rows past nao give zeros
      const bool sg_full = kSyG * sg + kSyG <= ngroups;  // every row group of the super-group exists
      double Zd[kSyG][2];
#pragma unroll
      for (int gi = 0; gi < kSyG; gi++) Zd[gi][0] = Zd[gi][1] = 0.0;

      const double* stage_ptr = ring;
#pragma unroll
      for (int cc = 0; cc < kSyNCH; cc++) {
        if (cc < nch) {
          const int stage = it % kSyStages;
          mbar_wait(full0 + 8 * stage, (it / kSyStages) & 1);
          stage_ptr = ring + stage * kSyStageDoubles;
          if (sg_full && cb0 + (kSyLC / 8) * (cc + 1) <= kSyG * sg) {
            // every block of the chunk is a full stored block: straight-line code, two row groups at a time so
            // that consecutive DMMAs on one accumulator are four instructions apart
#pragma unroll
            for (int qq = 0; qq < kQ; qq++) {
              const int sl = kQ * cc + qq;
              const double2 mf = get_mf(sl);
#pragma unroll
              for (int gp = 0; gp < kSyG; gp += 2) {
                const double* g0 = stage_ptr + gp * 8 * kSyS + 8 * NW * qq;
                const double* g1 = g0 + 8 * kSyS;
                const double ad00 = g0[offD], ad01 = g0[offD + 4], at00 = g0[offT0], at01 = g0[offT1];
                const double ad10 = g1[offD], ad11 = g1[offD + 4], at10 = g1[offT0], at11 = g1[offT1];
                dmma884(Zd[gp][0], Zd[gp][1], ad00, mf.x);
                dmma884(Zd[gp + 1][0], Zd[gp + 1][1], ad10, mf.x);
                dmma884(Zt[sl][0], Zt[sl][1], at00, tB[gp][0]);
                dmma884(Zd[gp][0], Zd[gp][1], ad01, mf.y);
                dmma884(Zd[gp + 1][0], Zd[gp + 1][1], ad11, mf.y);
                dmma884(Zt[sl][0], Zt[sl][1], at01, tB[gp][1]);
                dmma884(Zt[sl][0], Zt[sl][1], at10, tB[gp + 1][0]);
                dmma884(Zt[sl][0], Zt[sl][1], at11, tB[gp + 1][1]);
              }
            }
          } else {
#pragma unroll
            for (int gi = 0; gi < kSyG; gi++) {
              const int I = kSyG * sg + gi;
#pragma unroll
              for (int qq = 0; qq < kQ; qq++) {
                const int sl = kQ * cc + qq, Jb = cb0 + NW * sl + w;
                if (Jb < I && I < ngroups) {               // a full stored block (warp-uniform)
                  const double* gb = stage_ptr + gi * 8 * kSyS + 8 * NW * qq;
                  const double ad0 = gb[offD], ad1 = gb[offD + 4];
                  const double at0 = gb[offT0], at1 = gb[offT1];
                  const double2 mf = get_mf(sl);
                  dmma884(Zd[gi][0], Zd[gi][1], ad0, mf.x);
                  dmma884(Zt[sl][0], Zt[sl][1], at0, tB[gi][0]);
                  dmma884(Zd[gi][0], Zd[gi][1], ad1, mf.y);
                  dmma884(Zt[sl][0], Zt[sl][1], at1, tB[gi][1]);
                }
              }
            }
          }
          if (cc < nch - 1) {                            // the last chunk also holds the diagonal blocks
            __syncwarp();
            if (l == 0) mbar_arrive(empty0 + 8 * stage);
          }
          it++;
        }
      }
      // diagonal blocks (I, I) of the super-group: all four lie in its last chunk, each handled by its owner
      {
        const int cl = nch - 1;
#pragma unroll
        for (int gi = 0; gi < kSyG; gi++) {
          const int I = kSyG * sg + gi;
          if ((I & (NW - 1)) == w && I < ngroups && I < cb0 + kPanelBlocks) {   // I >= cb0: rows start at the panel
            const int x0 = 8 * I - col_base - kSyLC * cl;
            const double* gb = stage_ptr + gi * 8 * kSyS + x0;
#pragma unroll
            for (int h = 0; h < 2; h++) {
              // direct, stored part of the row only: lam <= mu
              const int lam = 8 * I + 4 * h + j;
              double a = gb[r * kSyS + (bpar ^ (r >> 2)) + 4 * h + j];
              if (4 * h + j > pr) a = 0.0;
              const double b = (col_ok && lam < nao) ? sy_m(q, lam, r) : 0.0;
              dmma884(Zd[gi][0], Zd[gi][1], a, b);
            }
#pragma unroll
            for (int g = 0; g < 2; g++) {
              // transposed with the output rows in fragment order: Z[8I + pr] += T[row][pr] M[8I + row], pr < row
              const int row = sy_perm(4 * g + j);
              double a = gb[(4 * g + j) * kSyS + (bpar ^ g) + pr];
              if (pr >= row) a = 0.0;
              dmma884(Zd[gi][0], Zd[gi][1], a, tB[gi][g]);
            }
          }
        }
        __syncwarp();
        if (l == 0) mbar_arrive(empty0 + 8 * ((it - 1) % kSyStages));
      }
      // partial direct tiles -> shared memory; the owner of each row group adds the 8 partials in fixed order
      double* zb = zd + (sgc & 1) * (NW * kSyG * 64);
#pragma unroll
      for (int gi = 0; gi < kSyG; gi++)
        *reinterpret_cast<double2*>(zb + (w * kSyG + gi) * 64 + r * 8 + 2 * j) = make_double2(Zd[gi][0], Zd[gi][1]);
      asm volatile("bar.sync 1, %0;" ::"n"(32 * NW) : "memory");
#pragma unroll
      for (int gi = 0; gi < kSyG; gi++) {
        const int I = kSyG * sg + gi;
        if ((I & (NW - 1)) == w && I < ngroups) {
          // natural row r of the block sits in fragment row invperm(r)
          const double* src = zb + gi * 64 + sy_invperm(r) * 8 + 2 * j;
          double s0 = 0.0, s1 = 0.0;
#pragma unroll
          for (int ww = 0; ww < NW; ww++) {
            const double2 v = *reinterpret_cast<const double2*>(src + ww * kSyG * 64);
            s0 += v.x;
            s1 += v.y;
          }
          if (I < cb0 + kPanelBlocks) {
            const int slI = (I - cb0) / NW;
#pragma unroll
            for (int sl = 0; sl < kSyNSLOT; sl++)
              if (sl == slI) { Zt[sl][0] += s0; Zt[sl][1] += s1; }
          } else if (PANELS && 8 * I + r < nao) {
            // a row group past this panel's columns: its Z tile lives in a later panel's registers; the direct sum goes
            // to memory (the first panel writes, later panels add)
            double2* zp = reinterpret_cast<double2*>(q.X + (size_t)pl * q.x_pstride + (size_t)(8 * I + r) * q.x_rstride + 2 * j);
            if (first_panel) *zp = make_double2(s0, s1);
            else { const double2 o = *zp; *zp = make_double2(o.x + s0, o.y + s1); }
          }
        }
      }
    }
    // Z of this aux row: block Jb = cb0 + NW sl + w, rows 8 Jb + r, columns 2j, 2j + 1 (later panels add to what
    // the first one stored for their rows)
    double* Xp = q.X + (size_t)pl * q.x_pstride;
#pragma unroll
    for (int sl = 0; sl < kSyNSLOT; sl++) {
      const int mu = 8 * (cb0 + NW * sl + w) + r;
      if (mu < nao) {
        double2* zp = reinterpret_cast<double2*>(Xp + (size_t)mu * q.x_rstride + 2 * j);
        if (!first_panel) { const double2 o = *zp; Zt[sl][0] += o.x; Zt[sl][1] += o.y; }
        *zp = make_double2(Zt[sl][0], Zt[sl][1]);
      }
    }
    if (RHO && q.rho) {
      // rho_P = sum_{mu, a} sign_a Z[mu][a] M[mu][a] over the rows of this panel: lanes -> warp (xor tree), warps -> CTA
      // in warp order, panels in launch order
      const unsigned int sw = __ldg(q.sgn) >> (2 * j);
      const double s0 = (sw & 1u) ? -1.0 : 1.0, s1 = (sw & 2u) ? -1.0 : 1.0;
      const bool c0_ok = 2 * j < q.ncols, c1_ok = 2 * j + 1 < q.ncols;
      double t = 0.0;
#pragma unroll
      for (int sl = 0; sl < kSyNSLOT; sl++) {
        const int mu = 8 * (cb0 + NW * sl + w) + r;
        if (mu < nao) {
          if (c0_ok) t = fma(Zt[sl][0] * s0, sy_m(q, mu, 2 * j), t);
          if (c1_ok) t = fma(Zt[sl][1] * s1, sy_m(q, mu, 2 * j + 1), t);
        }
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
      if (l == 0) rho_red[w] = t;
      asm volatile("bar.sync 1, %0;" ::"n"(32 * NW) : "memory");
      if (w == 0 && l == 0) {
        double v = 0.0;
#pragma unroll
        for (int ww = 0; ww < NW; ww++) v += rho_red[ww];
        q.rho[q.p_first + pl] = first_panel ? v : q.rho[q.p_first + pl] + v;
      }
    }
  }
}

// usable when the packed tensor is 16-byte aligned and the right-hand side has at most 8 columns
template <int NW, int G, int LC, int STAGES, bool MREG, bool PANELS, bool RHO>
static int launch_symm_cfg(dfjk_ctx* h, const SymmParams& p, int grid, cudaStream_t st) {
  using Cfg = SyCfg<NW, G, LC, STAGES, MREG>;
  static_assert(Cfg::kSmemBytes + 1024 <= 227 * 1024, "shared memory");
  static std::atomic<unsigned long long> attr_done{0};
  if (ensure_dyn_smem(k_symm_thin<NW, G, LC, STAGES, MREG, PANELS, RHO>, Cfg::kSmemBytes, h->device, attr_done) != cudaSuccess) return -1;
  k_symm_thin<NW, G, LC, STAGES, MREG, PANELS, RHO><<<grid, Cfg::kThreads, Cfg::kSmemBytes, st>>>(p);
  return 0;
}

bool symm_thin_ok(const dfjk_ctx* h, int ncols) {
  return !h->no_symm_thin && h->b_aligned16 && ncols >= 1 && ncols <= 8 && h->naux > 0;
}

static int launch_symm(dfjk_ctx* h, SymmParams p, int nb, cudaStream_t st) {
  const int grid = nb < h->num_sms ? nb : h->num_sms;
  // measured at nao = 1200, naux = 4000 (B200): 16 rows x 256 columns per stage, 3 stages, B fragments in shared
  // memory 4.3 ms; 32 x 128 x 3: 4.4; register-resident B fragments (32 x 128 x 5): 4.9-5.4; 16 consumer warps: 4.8
  const bool panels = h->nao > kSyMaxNao, rho = p.rho != nullptr;
  for (p.cb0 = 0; 8 * p.cb0 < h->nao; p.cb0 += kSyMaxNao / 8) {     // one launch per panel of 1280 columns
    int rc;
    if (panels) rc = rho ? launch_symm_cfg<8, 2, 256, 3, false, true, true>(h, p, grid, st)
                         : launch_symm_cfg<8, 2, 256, 3, false, true, false>(h, p, grid, st);
    else rc = rho ? launch_symm_cfg<8, 2, 256, 3, false, false, true>(h, p, grid, st)
                  : launch_symm_cfg<8, 2, 256, 3, false, false, false>(h, p, grid, st);
    if (rc != 0) return -1;
  }
  return 0;
}

// AO2MO: Z[pl][mu][a] (row-major, row stride ldx >= 8, even) for the aux rows [p_first, p_first + nb), M row-major
int launch_symm_thin(dfjk_ctx* h, const double* M, int ldm, int ncols, int p_first, int nb, double* X, int ldx,
                     cudaStream_t st) {
  SymmParams p{h->B, h->npair, (size_t)h->naux * h->npair, h->nao, M, ncols, 0, 0, ldm, 0, 1,
               X, (long long)h->nao * ldx, ldx, p_first, nb, nullptr, nullptr, 0};
  return launch_symm(h, p, nb, st);
}

// JK call on one set of at most 8 columns: X k-tiled for k_syrk2 (one 32-column chunk), C' from the k-tiled Ct of
// k_prep_ct, rho[P] (Eq. 14 through the half-transformed block, R16) when rho != nullptr
int launch_symm_thin_jk(dfjk_ctx* h, int ncols, int p_first, int nb, double* X, double* rho, cudaStream_t st) {
  SymmParams p{h->B, h->npair, (size_t)h->naux * h->npair, h->nao, h->Ct, ncols, 4, 15, (long long)h->ct_rows * kHtLd, 1, kHtLd,
               X, (long long)h->mu_pad * kLdT, kLdT, p_first, nb, rho, h->sgnbits, 0};
  return launch_symm(h, p, nb, st);
}

}  // namespace dfjk
