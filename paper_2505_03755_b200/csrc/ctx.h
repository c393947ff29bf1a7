// Internal context and kernel-launch prototypes of the DF-JK library (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#include <atomic>

#include "../../include/dfjk.h"

namespace dfjk {

constexpr int kMaxSets = 32;       // hard upper bound for options.max_nset
constexpr int kBK = 32;            // k-chunk (doubles) of the SYRK tile pipeline
constexpr int kLdT = kBK + 4;      // 36: row stride of a [rows][32] tile (4 mod 16: conflict-free fragments)
constexpr int kHtBK = 16;          // k-chunk of the half-transform
constexpr int kHtLd = kHtBK + 4;   // 20: row stride of [rows][16] tiles (4 mod 16)
constexpr int kHtMaxWN = 22;       // half-transform N tile = 16*WN columns, WN <= 22 (352 columns in one pass)
constexpr int kJ1Rows = 64;        // aux rows per J-pass-1 work item (8 DMMA row groups per warp)
constexpr int kJ1SubChunk = 2048;  // pairs per warp per J-pass-1 work item
constexpr int kJ1Warps = 8;
constexpr int kJ1Chunk = kJ1SubChunk * kJ1Warps;  // pairs per CTA work item
constexpr int kJ2Threads = 256;

// Column bookkeeping of one get_jk call: set s owns padded columns [col0[s], col0[s+1]) of C'/X,
// of which the first nocc[s] are real and the rest zero.
struct SetInfo {
  int nset;
  int nocc_pad;             // col0[nset]
  int col0[kMaxSets + 1];
  int nocc[kMaxSets];
  long long coff[kMaxSets];  // offset of block s inside the caller's C
  int ooff[kMaxSets];        // offset of set s inside the caller's occ
};

}  // namespace dfjk

struct dfjk_ctx {
  int naux, nao;
  size_t npair;
  int nck;                   // 16-wide k chunks of the half-transform = ceil(nao/16)
  int ct_rows;               // rows (padded columns of C') per chunk in the tiled C' buffer
  int mu_pad;                // nao rounded up to 128 (row extent of the tiled X)
  int device;
  const double* B;           // packed tensor (borrowed or owned)
  int b_aligned16;           // B is 16-byte aligned (8-byte aligned tensors take the scalar-load J paths)
  double* B_owned;
  double* Bt;                // optional re-tiled copy of B for the half-transform (HtParams)
  size_t bt_pstride;
  // options / plan
  int max_nset, max_nocc_total, nocc_pad_cap;
  int nblk, ksplit;          // capacities: aux rows of X at nocc_pad_cap columns; split-K partial slots
  int nblk_forced, ksplit_forced;
  int plan_nblk, plan_ksplit, plan_nblocks;  // what the last get_jk actually used
  int ks_cache_nblk, ks_cache_ntiles, ks_cache_val;   // last answer of the split-K model
  int n_mtiles;              // 128-row tiles along nao
  int j1_chunks, j2_splits;
  int j1_mma_min_sets;       // J pass 1: sets per group from which the DMMA kernel replaces the DFMA one
  int j2_mma_min_sets;       // J pass 2: likewise
  int num_sms;
  int ht_grid;               // persistent half-transform: CTAs (= SMs)
  int ao2mo_route;           // option: 0 = cheaper route, 1 = Eq. 18-21 as printed, 2 = active first
  int plan_ao2mo_route;      // what the last dfjk_ao2mo used
  int two_pass_j;            // option: never fuse J pass 1 into the half-transform
  int k_emu_slices;          // option: 0 = native fp64 SYRK (DMMA); 3..6 = FP64 emulated on the int8 tensor cores with that many 7-bit slices
  int k_emu_pgroup;          // aux rows that share one power-of-two scale per AO row in the emulated SYRK
  int ht_emu_slices;         // option: 0 = native fp64 half-transform; 3..6 = emulated on the int8 tensor cores
  int no_symm_thin;          // option: never use the one-pass symmetric thin half-transform (symm.cu)
  int no_small_path;         // option: never use the single-launch path for embedding-sized calls (small.cu)
  unsigned int* ticket;      // arrival counter of the single-launch path (zero between calls)
  signed char* Bq;           // emulated half-transform: int8 slice images of the unpacked B (built at create)
  double* bscale;            // [naux][mu_q] power-of-two scale of every row of every slice B_P
  signed char* Ctq;          // int8 slice images of C'^T (per call)
  double* cscale;            // [i_q] scale of every column of C'
  // scratch (all allocated at create)
  double* Ct;                // [nck][ct_rows][20]  C' transposed and k-tiled, sqrt(occ) folded, zero padded
  unsigned int* sgnbits;     // [nocc_pad_cap / 32 + 1]   bit c%32 of word c/32 = 1 iff padded column c has occ < 0
  double* Dw;                // [max_nset][npair]         packed density, off-diagonal weight 2
  double* rho_part;          // [j1_chunks][8][naux_pad]
  double* rho;               // [max_nset][naux]
  double* rho_ht;            // [naux][ht slots][nset] per-warp rho partials of the fused half-transform
  size_t rho_ht_doubles;
  double* Jp_part;           // [j2_splits][max_nset][npair]
  double* X;                 // [plan_nblk][nch][mu_pad][36] half-transformed block, k-tiled
  size_t X_doubles;          // capacity of X
  double* Kpart;             // [ksplit][max_nset][nao][nao]
  // staging for dfjk_get_jk_host
  double *C_stage, *occ_stage, *J_stage, *K_stage;
  size_t workspace_bytes;
  int last_launches;
  // optional per-phase CUDA-event profile of the last call (dfjk_set_profiling)
  int profiling, ev_cap, ev_n;
  cudaEvent_t* ev;
  int* ev_phase;
  char last_error[256];
};

namespace dfjk {

// Phase marker of the event profile: the phase lasts until the next marker on the stream.  The
// event pool grows on demand (host-side only; profiling is never on during a graph capture).
bool prof_grow(dfjk_ctx* h);
inline void prof_mark(dfjk_ctx* h, int phase, cudaStream_t st) {
  if (!h->profiling) return;
  if (h->ev_n >= h->ev_cap && !prof_grow(h)) return;
  cudaEventRecord(h->ev[h->ev_n], st);
  h->ev_phase[h->ev_n++] = phase;
}

// Opt-in to more than 48 KB of dynamic shared memory.  The attribute is per function AND per
// device, so every launcher keeps one bit per device (a second handle on another GPU of the same
// process sets it again); setting it twice is harmless, which makes the race between threads benign.
template <typename F>
inline cudaError_t ensure_dyn_smem(F* func, size_t bytes, int device, std::atomic<unsigned long long>& done) {
  const unsigned long long bit = device >= 0 && device < 64 ? 1ull << device : 0ull;
  if (bit && (done.load(std::memory_order_acquire) & bit)) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e == cudaSuccess && bit) done.fetch_or(bit, std::memory_order_release);
  return e;
}

// Each launcher enqueues on `st` and returns the number of kernels it launched.
int launch_prep_ct(dfjk_ctx* h, const SetInfo& si, const double* C, const double* occ, cudaStream_t st);
int launch_prep_dw(dfjk_ctx* h, const SetInfo& si, cudaStream_t st);
int launch_j_passes(dfjk_ctx* h, const SetInfo& si, double* J_out, bool rho_ready, cudaStream_t st);
int launch_k_path(dfjk_ctx* h, const SetInfo& si, double* K_out, bool want_rho, cudaStream_t st);
int launch_half_transform_rowmajor(dfjk_ctx* h, const SetInfo& si, int p_first, int nb, double* X, int ldx,
                                   cudaStream_t st);
// AO2MO (Eq. 18-21); returns the number of launches, -1 on a launch failure, -2 if the workspace
// cannot hold one aux row
int launch_ao2mo(dfjk_ctx* h, int nmo, int a0, int nact, const double* M, double* bpa_out, double* ppaa_out,
                 double* papa_out, cudaStream_t st);
// density-matrix form: packed weighted density from D, and K by Eq. 16-17 as printed
int launch_prep_dw_dm(dfjk_ctx* h, int nset, const double* D, cudaStream_t st);
int launch_k_path_dm(dfjk_ctx* h, int nset, const double* D, double* K_out, cudaStream_t st);
// FP64-emulated SYRK on the int8 tensor cores (emu.cu)
int emu_mu_q(int nao);
size_t emu_bytes_per_aux_row(int nao, int nchs_max, int S, int pgroup);
int emu_pick_ksplit(int nao, int ngroups, int max_split, int sms);
int launch_emu_syrk_set(dfjk_ctx* h, const double* X, int nch, int c0, int c1, int nb, signed char* Xq, double* scale,
                        double* Kpart_s, size_t split_stride, int ksplit, int first, cudaStream_t st);
size_t emu_bq_bytes(int naux, int nao, int S);
size_t emu_ctq_bytes(int nao, int nocc_pad_cap, int S);
int emu_i_q(int nocc_pad);
cudaError_t launch_emu_slice_b(dfjk_ctx* h);
int launch_emu_slice_ct(dfjk_ctx* h, int nocc_pad, cudaStream_t st);
int launch_emu_ht(dfjk_ctx* h, int nocc_pad, int p_first, int nb, double* X, int nch, cudaStream_t st);
// single-launch path for embedding-sized calls (small.cu): CTAs it would use (0 = not eligible); launch
int small_path_ctas(const dfjk_ctx* h, const SetInfo& si);
int launch_small_fused(dfjk_ctx* h, const SetInfo& si, int ctas, const double* C, const double* occ, double* J_out,
                       double* K_out, cudaStream_t st);
// one-pass symmetric thin half-transform on the packed triangle (symm.cu): <= 8 columns, row-major Z
bool symm_thin_ok(const dfjk_ctx* h, int ncols);
int launch_symm_thin(dfjk_ctx* h, const double* M, int ldm, int ncols, int p_first, int nb, double* X, int ldx,
                     cudaStream_t st);
int launch_symm_thin_jk(dfjk_ctx* h, int ncols, int p_first, int nb, double* X, double* rho, cudaStream_t st);
size_t retile_doubles_per_aux_row(int nao);
cudaError_t launch_retile(const double* Bp, size_t npair, int nao, int naux, double* Bt);
int run_dmma_selftest();

}  // namespace dfjk
