// Single-launch path for embedding-sized calls ("N_emb is
// independent of the system size", "called thousands of times"): when the whole call is
// a few MFLOP, the seven dependent launches of the tiled path (prep, half-transform, SYRK, rho
// reduce, J pass 2, two epilogues) cost more than the arithmetic.  Here ONE kernel does steps a1-a9:
//   phase 1, per CTA, for its aux rows P (round-robin, one or two each):
//     b^P unpacked into shared memory, X = b^P C' (Eq. 16), rho_s = <X_s, C'_s sign> (Eq. 14,
//     DESIGN.md R16), K partial += X_s sign X_s^T (Eq. 17, lower triangle), J partial += rho_s b^P (Eq. 15),
//     both partials private to the CTA and every element owned by one thread: the first aux row of the CTA stores,
//     later ones add with a reduction that returns nothing (no load to wait for; one thread per address in program
//     order, so the sum is the same double as a load-add-store and the result stays deterministic);
//   grid barrier (the kernel is launched cooperatively: all CTAs are resident);
//   phase 2, all CTAs: every output element is the sum of the partials in CTA order, written to both
//     triangles of J and K (deterministic: the assignment of aux rows to CTAs is fixed).
// The two products of phase 1 run as 8 x 8 x 4 DMMA tiles out of shared memory (a scalar DFMA version spent 40 % of its
// time on the instructions of the K loop at nao = 80); rho, the J partial and phase 2 are plain DFMA / DADD.
// Chosen by dfjk_get_jk when nao <= 96, nao * sum(nocc) <= 4608 and naux * nao^2 * (sum(nocc) + nset)
// <= 2^26 (2^27 for one set; option no_small_path disables it); everything larger takes the tiled tensor-pipe kernels.
#include <cstdarg>
#include <cstdio>

#include "common.cuh"
#include "ctx.h"

namespace dfjk {

constexpr int kSmThreads = 256;
constexpr int kSmMaxNao = 96, kSmMaxElems = 4608;
constexpr double kSmMaxWork = 67108864.0;           // 2^26; one set: twice that (measured crossover with the tiled kernels:
                                                    // 2^27.5 for one set, below 2^26.6 for four thin sets)

struct SmallParams {
  const double* Bp; size_t npair; int naux, nao;
  const double* C; const double* occ;
  double* J; double* K;                   // outputs (either may be nullptr)
  double* Kpart; double* Jpart;           // [cta][set][nao*nao], [cta][set][npair]
  unsigned int* ticket;                   // [0] arrivals at the grid barrier, [1] CTAs done (both zero between calls)
  int ntot;                               // sum of nocc
};

// packed index -> (mu, nu), mu >= nu: float estimate, exact integer correction
__device__ __forceinline__ void untri(int pr, int& mu, int& nu) {
  int m = (int)((sqrtf(8.0f * (float)pr + 1.0f) - 1.0f) * 0.5f);
  while ((m + 1) * (m + 2) / 2 <= pr) m++;
  while (m * (m + 1) / 2 > pr) m--;
  mu = m;
  nu = pr - m * (m + 1) / 2;
}

// fixed-tree block sum of one value per thread; result valid in every thread
__device__ __forceinline__ double block_sum(double v, double* red) {
  const int tid = threadIdx.x;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  __syncthreads();
  if ((tid & 31) == 0) red[tid >> 5] = v;
  __syncthreads();
  double t = 0.0;
#pragma unroll
  for (int w = 0; w < kSmThreads / 32; w++) t += red[w];
  return t;
}

__global__ void __launch_bounds__(kSmThreads)
k_small_fused(const __grid_constant__ SetInfo si, const __grid_constant__ SmallParams q) {
  extern __shared__ __align__(16) double smem[];
  const int nao = q.nao, ntot = q.ntot, ldb = nao + 1, tid = threadIdx.x;
  const int ldxs = ntot | 1;              // odd row stride of Xs: the fragment loads of the K product walk its rows
  const int nao4 = (nao + 3) & ~3;        // C' rows padded to the k step of the MMA (zero rows)
  double* Bs = smem;                      // [nao][nao + 1]   symmetric slice (column nao stays zero)
  double* Cs = Bs + nao * ldb;            // [nao4][ntot]     C' = C sqrt|occ|
  double* Xs = Cs + nao4 * ntot;          // [nao][ldxs]
  double* sg = Xs + nao * ldxs;           // [ntot]           sign(occ)
  double* red = sg + ntot;                // [16]
  __shared__ int c0s[kMaxSets + 1];
  const size_t n2 = (size_t)nao * nao;
  const int w = tid >> 5, l = tid & 31, r = l >> 2, jj = l & 3;      // DMMA.8x8x4 fragment coordinates
  const int mt = (nao + 7) >> 3;          // 8-row blocks of the basis

  // the packed row of the next aux row is fetched into registers while the current one is processed;
  // (mu, nu) of the packed elements a thread owns are the same for every row: worked out once
  constexpr int kPre = (kSmMaxNao * (kSmMaxNao + 1) / 2 + kSmThreads - 1) / kSmThreads;     // 19
  double pre[kPre];
  int mn[kPre];
#pragma unroll
  for (int k = 0; k < kPre; k++) {
    const int pr = tid + k * kSmThreads;
    int mu = 0, nu = 0;
    if (pr < (int)q.npair) untri(pr, mu, nu);
    mn[k] = (mu << 8) | nu;
  }
  auto prefetch = [&](int P) {
    const double* bp = q.Bp + (size_t)P * q.npair;
#pragma unroll
    for (int k = 0; k < kPre; k++) {
      const int pr = tid + k * kSmThreads;
      pre[k] = (P < q.naux && pr < (int)q.npair) ? ldg_stream1(bp + pr) : 0.0;
    }
  };
  prefetch(blockIdx.x);                  // in flight during the prologue

  // every pad (column nao of Bs, rows nao.. of C', the odd column of Xs) is zero, and nothing a fragment load can
  // touch is uninitialised: a pad meets a zero in the other operand, and rows or columns past the end only feed
  // results that are not stored
  for (int i = tid; i < nao * ldb + nao4 * ntot + nao * ldxs + ntot + 16; i += kSmThreads) smem[i] = 0.0;
  __syncthreads();
  // a1: C' and the signs; compact column c of set s = si.ooff[s] + i.  sg first holds sqrt|occ|, then sign(occ)
  if (tid <= si.nset) c0s[tid] = tid < si.nset ? si.ooff[tid] : ntot;
  for (int c = tid; c < ntot; c += kSmThreads) sg[c] = sqrt(fabs(q.occ[c]));
  __syncthreads();
  for (int s = 0; s < si.nset; s++) {
    const int n = si.nocc[s], o = si.ooff[s];
    for (int e = tid; e < nao * n; e += kSmThreads) {
      const int lam = e / n, i = e - lam * n;
      Cs[lam * ntot + o + i] = q.C[si.coff[s] + e] * sg[o + i];
    }
  }
  __syncthreads();
  for (int c = tid; c < ntot; c += kSmThreads) sg[c] = q.occ[c] < 0.0 ? -1.0 : 1.0;
  __syncthreads();

  double* Kp = q.Kpart + (size_t)blockIdx.x * si.nset * n2;
  double* Jp = q.Jpart + (size_t)blockIdx.x * si.nset * q.npair;
  bool first = true;
  for (int P = blockIdx.x; P < q.naux; P += gridDim.x, first = false) {
    // a5: unpack the packed row into the symmetric slice
#pragma unroll
    for (int k = 0; k < kPre; k++) {
      if (tid + k * kSmThreads < (int)q.npair) {
        const int mu = mn[k] >> 8, nu = mn[k] & 255;
        Bs[mu * ldb + nu] = pre[k];
        Bs[nu * ldb + mu] = pre[k];
      }
    }
    prefetch(P + gridDim.x);
    __syncthreads();
    // a6: X = b C' in 8 x 8 tiles on the FP64 tensor pipe, a warp takes every eighth tile.  A[row][k] = b[mu][lam],
    // B[k][col] = C'[lam][c]; rows past nao are clamped (their results are not stored), lam past nao meets the
    // zero rows of C', columns past ntot run into finite data and are not stored
    {
      const int nt = (ntot + 7) >> 3;
      for (int t = w; t < mt * nt; t += kSmThreads / 32) {
        const int i = t / nt, j = t - i * nt;
        const double* ap = Bs + min(8 * i + r, nao - 1) * ldb + jj;
        const double* bp = Cs + jj * ntot + 8 * j + r;
        double d0 = 0.0, d1 = 0.0;
        for (int k0 = 0; k0 < nao; k0 += 4) dmma884(d0, d1, ap[k0], bp[k0 * ntot]);
        const int row = 8 * i + r, col = 8 * j + 2 * jj;
        if (row < nao) {
          if (col < ntot) Xs[row * ldxs + col] = d0;
          if (col + 1 < ntot) Xs[row * ldxs + col + 1] = d1;
        }
      }
    }
    __syncthreads();
    for (int s = 0; s < si.nset; s++) {
      const int ca = c0s[s], cb = c0s[s + 1];
      if (q.J) {
        // a2 (fused): rho = sum_{mu, c in s} sign_c X[mu][c] C'[mu][c]; a3: J partial += rho * packed row
        double t = 0.0;
        for (int e = tid; e < nao * (cb - ca); e += kSmThreads) {
          const int mu = e / (cb - ca), c = ca + e - mu * (cb - ca);
          t = fma(Xs[mu * ldxs + c] * sg[c], Cs[mu * ntot + c], t);
        }
        const double rho = block_sum(t, red);
        double* jp = Jp + (size_t)s * q.npair;
#pragma unroll
        for (int k = 0; k < kPre; k++) {
          const int pr = tid + k * kSmThreads;
          if (pr < (int)q.npair) {
            const double v = rho * Bs[(mn[k] >> 8) * ldb + (mn[k] & 255)];
            if (first) jp[pr] = v; else atomicAdd(jp + pr, v);
          }
        }
      }
      if (q.K && cb > ca) {
        // a7: K partial[mu >= nu] += sum_{c in s} sign_c X[mu][c] X[nu][c], the lower 8 x 8 tiles (i >= j) on the tensor
        // pipe: A[row][k] = X[mu][c], B[k][col] = sign_c X[nu][c], zero past the last column of the set
        double* kp = Kp + (size_t)s * n2;
        const int nk = (cb - ca + 3) >> 2;
        for (int t = w; t < mt * (mt + 1) / 2; t += kSmThreads / 32) {
          int i, j;
          untri(t, i, j);
          const double* ap = Xs + min(8 * i + r, nao - 1) * ldxs + ca + jj;
          const double* bp = Xs + min(8 * j + r, nao - 1) * ldxs + ca + jj;
          double d0 = 0.0, d1 = 0.0;
          for (int k = 0; k < nk; k++) {
            const int c = ca + 4 * k + jj;
            const double b = c < cb ? bp[4 * k] * sg[c] : 0.0;
            dmma884(d0, d1, ap[4 * k], b);
          }
          const int row = 8 * i + r, col = 8 * j + 2 * jj;
          if (row < nao) {
            double* o = kp + (size_t)row * nao + col;
            if (col <= row) { if (first) o[0] = d0; else atomicAdd(o, d0); }
            if (col + 1 <= row) { if (first) o[1] = d1; else atomicAdd(o + 1, d1); }
          }
        }
      } else if (q.K && first) {
        // a set without columns: its partial is zero
        double* kp = Kp + (size_t)s * n2;
        for (int e = tid; e < nao * nao; e += kSmThreads) kp[e] = 0.0;
      }
    }
    __syncthreads();
  }

  // grid barrier: every partial is in global memory before anyone sums
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    atomicAdd(q.ticket, 1u);
    while (*reinterpret_cast<volatile unsigned int*>(q.ticket) < gridDim.x) {}
  }
  __syncthreads();
  __threadfence();
  // a4 / a9: every output element = sum of the partials, written to both triangles.  Eight lanes share one
  // element: lane k sums the partials k, k + 8, ... in ascending order, the eight sums are combined by a
  // fixed shuffle tree -- the same order in every call
  const int nparts = gridDim.x;
  const size_t nout = (size_t)si.nset * q.npair;
  const int sub = tid & 7;
  for (size_t o0 = ((size_t)blockIdx.x * kSmThreads + tid) >> 3;; o0 += ((size_t)gridDim.x * kSmThreads) >> 3) {
    const bool on = o0 < nout;
    if (__syncthreads_or(on) == 0) break;
    const size_t o = on ? o0 : 0;
    const int s = (int)(o / q.npair);
    const int pr = (int)(o - (size_t)s * q.npair);
    int mu, nu;
    untri(pr, mu, nu);
    const size_t e = (size_t)mu * nao + nu, et = (size_t)nu * nao + mu;
    double tk = 0.0, tj = 0.0;
    if (on && q.K)
      for (int g = sub; g < nparts; g += 8) tk += __ldcg(q.Kpart + ((size_t)g * si.nset + s) * n2 + e);
    if (on && q.J)
      for (int g = sub; g < nparts; g += 8) tj += __ldcg(q.Jpart + ((size_t)g * si.nset + s) * q.npair + pr);
#pragma unroll
    for (int off = 4; off > 0; off >>= 1) {
      tk += __shfl_xor_sync(0xffffffffu, tk, off);
      tj += __shfl_xor_sync(0xffffffffu, tj, off);
    }
    if (on && sub == 0) {
      if (q.K) { q.K[(size_t)s * n2 + e] = tk; q.K[(size_t)s * n2 + et] = tk; }
      if (q.J) { q.J[(size_t)s * n2 + e] = tj; q.J[(size_t)s * n2 + et] = tj; }
    }
  }
  // the last CTA to finish re-arms the barrier for the next call (every CTA has passed it by then)
  __syncthreads();
  if (tid == 0 && atomicAdd(q.ticket + 1, 1u) == gridDim.x - 1) {
    q.ticket[0] = 0;
    q.ticket[1] = 0;
  }
}

static size_t small_smem_bytes(int nao, int ntot) {
  return ((size_t)nao * (nao + 1) + (size_t)((nao + 3) & ~3) * ntot + (size_t)nao * (ntot | 1) + ntot + 16) * sizeof(double);
}

static cudaError_t small_attr(int device) {
  static std::atomic<unsigned long long> attr_done{0};
  return ensure_dyn_smem(k_small_fused, (size_t)200 * 1024, device, attr_done);
}

// 0 = not eligible, else the number of CTAs the fused kernel would use
int small_path_ctas(const dfjk_ctx* h, const SetInfo& si) {
  if (h->no_small_path || h->naux < 1 || h->nao > kSmMaxNao || h->k_emu_slices || h->ht_emu_slices) return 0;
  int ntot = 0;
  for (int s = 0; s < si.nset; s++) ntot += si.nocc[s];
  if (ntot < 1 || (long long)h->nao * ntot > kSmMaxElems) return 0;
  if ((double)h->naux * h->nao * h->nao * (ntot + si.nset) > (si.nset == 1 ? 2.0 : 1.0) * kSmMaxWork) return 0;
  // as many CTAs as aux rows, in equal rounds over at most two resident CTAs per SM (more partials would make the
  // final sum the long pole); the cooperative launch needs all of them resident
  int occ = 0;
  if (small_attr(h->device) != cudaSuccess) { cudaGetLastError(); return 0; }
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_small_fused, kSmThreads, small_smem_bytes(h->nao, ntot)) != cudaSuccess) {
    cudaGetLastError();
    return 0;
  }
  if (occ < 1) return 0;
  const int slots = h->num_sms * (occ < 2 ? occ : 2);
  const int rounds = cdiv(h->naux, slots);
  int ctas = cdiv(h->naux, rounds);
  // the private partials live in the X workspace
  const size_t need = (size_t)ctas * si.nset * ((size_t)h->nao * h->nao + h->npair);
  if (need > h->X_doubles) return 0;
  return ctas;
}

int launch_small_fused(dfjk_ctx* h, const SetInfo& si, int ctas, const double* C, const double* occ, double* J_out,
                       double* K_out, cudaStream_t st) {
  int ntot = 0;
  for (int s = 0; s < si.nset; s++) ntot += si.nocc[s];
  const size_t smem = small_smem_bytes(h->nao, ntot);
  if (small_attr(h->device) != cudaSuccess) return -1;
  SmallParams p{h->B, h->npair, h->naux, h->nao, C, occ, J_out, K_out, h->X,
                h->X + (size_t)ctas * si.nset * h->nao * h->nao, h->ticket, ntot};
  prof_mark(h, DFJK_PHASE_HALF_TRANSFORM, st);
  // cooperative launch: the grid barrier needs every CTA resident (ctas <= SMs, one CTA per SM fits)
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(ctas); cfg.blockDim = dim3(kSmThreads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeCooperative;
  attr[0].val.cooperative = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  if (cudaLaunchKernelEx(&cfg, k_small_fused, si, p) != cudaSuccess) return -1;
  return 1;
}

}  // namespace dfjk

// ---------------------------------------------------------------------------------------------------------
// dfjk_small_jk_static (include/dfjk.h): the same kernel for callers that cannot allocate (CUDA graph capture,
// serving loops, harnesses that forbid cudaMalloc).  No handle: the private J/K partials and the two barrier
// counters live in one file-scope device array that every GPU loading the library holds until exit.
// ---------------------------------------------------------------------------------------------------------
namespace {

constexpr size_t kStaticDoubles = (size_t)1 << 20;   // 8 MiB of partials (DFJK_STATIC_SCRATCH_BYTES)
constexpr size_t kStaticHead = 32;                   // 256 B in front: [0], [1] of the first 8 bytes are the tickets
static_assert(kStaticDoubles * sizeof(double) == DFJK_STATIC_SCRATCH_BYTES, "header and kernel disagree");
static __device__ __align__(256) double g_static_scratch[kStaticHead + kStaticDoubles];

// In host code g_static_scratch is only a stand-in for the symbol: the device address is asked for once per
// device, with that device current, and kept here together with what else the launch needs to know about it.
struct StaticDev {
  std::atomic<int> state{0};   // 0 = not set up, 1 = being set up, 2 = ready, 3 = failed
  double* scratch = nullptr;
  int num_sms = 0, cc_major = 0;
  cudaError_t err = cudaSuccess;
};
constexpr int kStaticMaxDev = 64;
StaticDev g_static_dev[kStaticMaxDev];
thread_local char g_static_err[256] = "";

int static_fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_static_err, sizeof(g_static_err), fmt, ap);
  va_end(ap);
  return code;
}

// set-up of the CURRENT device (dev); returns its record or nullptr
StaticDev* static_setup(int dev) {
  StaticDev& d = g_static_dev[dev];
  int s = d.state.load(std::memory_order_acquire);
  if (s == 2) return &d;
  int expect = 0;
  if (s == 0 && d.state.compare_exchange_strong(expect, 1, std::memory_order_acq_rel)) {
    double* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&d.num_sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&d.cc_major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e == cudaSuccess && p == nullptr) e = cudaErrorInvalidSymbol;
    d.scratch = p;
    d.err = e;
    if (e != cudaSuccess) cudaGetLastError();
    d.state.store(e == cudaSuccess ? 2 : 3, std::memory_order_release);
  }
  while ((s = d.state.load(std::memory_order_acquire)) == 1) {}
  return s == 2 ? &d : nullptr;
}

}  // namespace

extern "C" {

const char* dfjk_small_jk_static_last_error(void) { return g_static_err; }

int dfjk_small_jk_static(int naux, int nao, const double* B_packed, int nset, const int* nocc, const double* C,
                         const double* occ, double* J_out, double* K_out, dfjk_stream stream) {
  using namespace dfjk;
  g_static_err[0] = 0;
  if (naux < 1 || nao < 1 || nset < 1 || !nocc || !B_packed)
    return static_fail(DFJK_ERR_INVALID_ARG, "naux, nao, nset must be >= 1 and B_packed, nocc non-NULL");
  if (nao > kSmMaxNao) return static_fail(DFJK_ERR_INVALID_ARG, "nao = %d is beyond the maximum %d of this entry point", nao, kSmMaxNao);
  if (nset > DFJK_STATIC_MAX_NSET)
    return static_fail(DFJK_ERR_INVALID_ARG, "nset = %d is beyond the maximum %d of this entry point", nset, DFJK_STATIC_MAX_NSET);
  SetInfo si{};
  si.nset = nset;
  long long coff = 0;
  int ntot = 0, col = 0;
  for (int s = 0; s < nset; s++) {
    if (nocc[s] < 0 || nocc[s] > nao) return static_fail(DFJK_ERR_INVALID_ARG, "nocc[%d] = %d is outside [0, nao]", s, nocc[s]);
    si.col0[s] = col; si.nocc[s] = nocc[s]; si.coff[s] = coff; si.ooff[s] = ntot;
    col += round_up(nocc[s], 8);
    coff += (long long)nao * nocc[s];
    ntot += nocc[s];
  }
  si.col0[nset] = col;
  si.nocc_pad = col;
  if (ntot < 1 || !C || !occ) return static_fail(DFJK_ERR_INVALID_ARG, "needs at least one occupied column and C, occ non-NULL");
  if ((long long)nao * ntot > kSmMaxElems)
    return static_fail(DFJK_ERR_INVALID_ARG, "nao * sum(nocc) = %lld is beyond the maximum %d of this entry point", (long long)nao * ntot, kSmMaxElems);
  if ((double)naux * nao * nao * (ntot + nset) > kSmMaxWork)
    return static_fail(DFJK_ERR_INVALID_ARG, "naux * nao^2 * (sum(nocc) + nset) is beyond the maximum 2^26 of this entry point");
  if (!J_out && !K_out) return DFJK_OK;

  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= kStaticMaxDev) { cudaGetLastError(); return static_fail(DFJK_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e)); }
  StaticDev* d = static_setup(dev);
  if (!d) return static_fail(DFJK_ERR_CUDA, "cudaGetSymbolAddress of the static scratch on device %d: %s", dev, cudaGetErrorString(g_static_dev[dev].err));
  if (d->cc_major != 10) return static_fail(DFJK_ERR_UNSUPPORTED_ARCH, "device %d is sm_%d0, the library is built for sm_100", dev, d->cc_major);

  const size_t npair = (size_t)nao * (nao + 1) / 2, n2 = (size_t)nao * nao;
  const size_t per_cta = (size_t)nset * (n2 + npair);           // doubles of private partials per CTA
  if (per_cta > kStaticDoubles) return static_fail(DFJK_ERR_INVALID_ARG, "one CTA's partials exceed the static scratch");
  const size_t smem = small_smem_bytes(nao, ntot);
  if ((e = small_attr(dev)) != cudaSuccess) { cudaGetLastError(); return static_fail(DFJK_ERR_CUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e)); }
  int resident = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, k_small_fused, kSmThreads, smem);
  if (e != cudaSuccess || resident < 1) { cudaGetLastError(); return static_fail(DFJK_ERR_CUDA, "the kernel does not fit an SM with %zu bytes of shared memory", smem); }
  // as dfjk_get_jk sizes it (equal rounds over at most two resident CTAs per SM), then capped by the static scratch
  const int slots = d->num_sms * (resident < 2 ? resident : 2);
  int ctas = cdiv(naux, cdiv(naux, slots));
  const size_t fit = kStaticDoubles / per_cta;
  if ((size_t)ctas > fit) ctas = (int)fit;

  cudaStream_t st = (cudaStream_t)stream;
  unsigned int* ticket = reinterpret_cast<unsigned int*>(d->scratch);
  double* part = d->scratch + kStaticHead;
  // the array keeps the last call's contents: the barrier counters must start at zero (a call that failed half way
  // would leave them set); the partials are overwritten before they are read (every CTA owns >= 1 aux row)
  if ((e = cudaMemsetAsync(ticket, 0, 2 * sizeof(unsigned int), st)) != cudaSuccess) { cudaGetLastError(); return static_fail(DFJK_ERR_CUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e)); }
  SmallParams p{B_packed, npair, naux, nao, C, occ, J_out, K_out, part, part + (size_t)ctas * nset * n2, ticket, ntot};
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(ctas); cfg.blockDim = dim3(kSmThreads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeCooperative;
  attr[0].val.cooperative = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  if ((e = cudaLaunchKernelEx(&cfg, k_small_fused, si, p)) != cudaSuccess) { cudaGetLastError(); return static_fail(DFJK_ERR_CUDA, "cooperative launch of %d CTAs: %s", ctas, cudaGetErrorString(e)); }
  return DFJK_OK;
}

}  // extern "C"
