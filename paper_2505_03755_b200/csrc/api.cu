// C ABI of the DF-JK library (include/dfjk.h): handle, validation, planning, enqueue.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "common.cuh"
#include "ctx.h"

using namespace dfjk;

namespace {

void set_err(dfjk_ctx* h, const char* where, cudaError_t e) {
  if (h) snprintf(h->last_error, sizeof(h->last_error), "%s: %s", where, cudaGetErrorString(e));
}

template <typename T>
bool dev_alloc(dfjk_ctx* h, T** p, size_t count) {
  *p = nullptr;
  if (count == 0) count = 1;
  cudaError_t e = cudaMalloc((void**)p, count * sizeof(T));
  if (e != cudaSuccess) {
    set_err(h, "cudaMalloc", e);
    cudaGetLastError();
    return false;
  }
  h->workspace_bytes += count * sizeof(T);
  return true;
}

void free_all(dfjk_ctx* h) {
  cudaFree(h->B_owned); cudaFree(h->Bt); cudaFree(h->Ct); cudaFree(h->sgnbits); cudaFree(h->Dw); cudaFree(h->rho_part); cudaFree(h->rho); cudaFree(h->rho_ht);
  cudaFree(h->Jp_part); cudaFree(h->X); cudaFree(h->Kpart);
  cudaFree(h->ticket); cudaFree(h->Bq); cudaFree(h->bscale); cudaFree(h->Ctq); cudaFree(h->cscale);
  cudaFree(h->C_stage); cudaFree(h->occ_stage); cudaFree(h->J_stage); cudaFree(h->K_stage);
  for (int i = 0; i < h->ev_cap; i++) cudaEventDestroy(h->ev[i]);
  delete[] h->ev;
  delete[] h->ev_phase;
}

// validate nocc and lay out the padded columns of C'/X
int build_setinfo(const dfjk_ctx* h, int nset, const int* nocc, SetInfo* si) {
  if (nset < 1 || nset > h->max_nset || !nocc) return DFJK_ERR_INVALID_ARG;
  si->nset = nset;
  long long coff = 0;
  int ooff = 0, col = 0;
  for (int s = 0; s < nset; s++) {
    if (nocc[s] < 0 || nocc[s] > h->nao) return DFJK_ERR_INVALID_ARG;
    si->col0[s] = col;
    si->nocc[s] = nocc[s];
    si->coff[s] = coff;
    si->ooff[s] = ooff;
    col += round_up(nocc[s], 8);
    coff += (long long)h->nao * nocc[s];
    ooff += nocc[s];
  }
  si->col0[nset] = col;
  si->nocc_pad = col;
  if (ooff > h->max_nocc_total || col > h->nocc_pad_cap) return DFJK_ERR_INVALID_ARG;
  return DFJK_OK;
}

// Every entry point that touches the device runs on the handle's device: the scratch, the
// function attributes and the caller's stream all belong to it.
bool on_handle_device(dfjk_ctx* h) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return false; }
  if (dev != h->device) {
    snprintf(h->last_error, sizeof(h->last_error), "current device %d is not the handle's device %d", dev, h->device);
    return false;
  }
  return true;
}

}  // namespace

namespace dfjk {
// doubles the event pool of the phase profile; false if no more events can be had
bool prof_grow(dfjk_ctx* h) {
  const int cap = h->ev_cap > 0 ? 2 * h->ev_cap : 1024;
  cudaEvent_t* ev = new (std::nothrow) cudaEvent_t[cap];
  int* ph = new (std::nothrow) int[cap];
  if (!ev || !ph) { delete[] ev; delete[] ph; return false; }
  for (int i = 0; i < h->ev_cap; i++) { ev[i] = h->ev[i]; ph[i] = h->ev_phase[i]; }
  int n = h->ev_cap;
  for (; n < cap; n++)
    if (cudaEventCreate(&ev[n]) != cudaSuccess) { cudaGetLastError(); break; }
  delete[] h->ev;
  delete[] h->ev_phase;
  h->ev = ev; h->ev_phase = ph;
  const bool grew = n > h->ev_cap;
  h->ev_cap = n;
  return grew;
}
}  // namespace dfjk

extern "C" {

const char* dfjk_strerror(int code) {
  switch (code) {
    case DFJK_OK: return "ok";
    case DFJK_ERR_INVALID_ARG: return "invalid argument";
    case DFJK_ERR_ALLOC: return "allocation failed";
    case DFJK_ERR_CUDA: return "CUDA error";
    case DFJK_ERR_UNSUPPORTED_ARCH: return "unsupported device architecture (needs sm_100)";
    default: return "unknown error code";
  }
}

int dfjk_create(int naux, int nao, const double* B_packed, const dfjk_options* opt, dfjk_handle* out) {
  if (!out) return DFJK_ERR_INVALID_ARG;
  *out = nullptr;
  if (naux < 0 || nao < 1 || nao > 32768) return DFJK_ERR_INVALID_ARG;
  if (naux > 0 && !B_packed) return DFJK_ERR_INVALID_ARG;
  if (((uintptr_t)B_packed & 7u) != 0) return DFJK_ERR_INVALID_ARG;
  dfjk_options o;
  memset(&o, 0, sizeof(o));
  if (opt) o = *opt;
  if (o.nblk < 0 || o.max_nocc_total < 0 || o.max_nset < 0 || o.max_nset > kMaxSets || o.ksplit < 0 ||
      o.ao2mo_route < 0 || o.ao2mo_route > 2)
    return DFJK_ERR_INVALID_ARG;
  if (o.k_emulation_slices != 0 && (o.k_emulation_slices < 3 || o.k_emulation_slices > 6)) return DFJK_ERR_INVALID_ARG;
  if (o.k_emulation_group < 0 || o.k_emulation_group > 64) return DFJK_ERR_INVALID_ARG;
  if (o.ht_emulation_slices != 0 && (o.ht_emulation_slices < 3 || o.ht_emulation_slices > 6)) return DFJK_ERR_INVALID_ARG;

  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
    cudaGetLastError();
    return DFJK_ERR_CUDA;
  }
  if (prop.major != 10) return DFJK_ERR_UNSUPPORTED_ARCH;

  dfjk_ctx* h = new (std::nothrow) dfjk_ctx;
  if (!h) return DFJK_ERR_ALLOC;
  memset(h, 0, sizeof(*h));
  h->naux = naux; h->nao = nao; h->device = dev;
  h->num_sms = prop.multiProcessorCount;
  h->ht_grid = h->num_sms;
  h->two_pass_j = o.two_pass_j;
  h->k_emu_slices = o.k_emulation_slices;
  h->k_emu_pgroup = o.k_emulation_group ? o.k_emulation_group : 16;
  h->ht_emu_slices = o.ht_emulation_slices;
  h->no_symm_thin = o.no_symm_thin;
  h->no_small_path = o.no_small_path;
  h->ao2mo_route = o.ao2mo_route;
  h->npair = (size_t)nao * (nao + 1) / 2;
  h->nck = cdiv(nao, kHtBK);
  h->mu_pad = round_up(nao, 8) + 128;   // any SYRK tile of <= 128 rows stays inside the tiled X
  h->max_nset = o.max_nset ? o.max_nset : 8;
  h->max_nocc_total = o.max_nocc_total ? o.max_nocc_total : nao;
  h->nocc_pad_cap = round_up(h->max_nocc_total + 7 * h->max_nset, 8);
  h->ct_rows = h->nocc_pad_cap + 16 * kHtMaxWN;   // any N tile of the half-transform stays in bounds
  h->n_mtiles = cdiv(nao, 128);
  h->nblk_forced = o.nblk;
  h->ksplit_forced = o.ksplit;
  // split-K partial slots of the SYRK (each is max_nset x nao x nao doubles)
  // 16 slots, more for small bases (up to 64 while the slots stay under 1 GB): the finer the split
  // can be, the closer the SYRK's CTA count gets to a whole number of waves
  {
    const double slot_bytes = (double)h->max_nset * nao * nao * sizeof(double);
    int cap = (int)(1.0e9 / slot_bytes);
    if (cap < 16) cap = 16;
    if (cap > 64) cap = 64;
    h->ksplit = o.ksplit ? o.ksplit : cap;
  }
  // X capacity (k-tiled layout [nch][mu_pad][36] per aux row): the cap, but at least one aux row
  // at full column capacity
  {
    // default: 4 GiB, but no more than a tenth of the memory that is free right now (the "dynamic
    // N_blk based on available memory" the paper leaves to future work)
    size_t cap = o.workspace_cap_bytes;
    if (cap == 0) {
      cap = (size_t)4 << 30;
      size_t free_b = 0, total_b = 0;
      if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && free_b / 10 < cap) cap = free_b / 10;
      else cudaGetLastError();
    }
    size_t one_row = (size_t)cdiv(h->nocc_pad_cap, kBK) * h->mu_pad * kLdT;
    if (h->k_emu_slices > 0)    // the emulated SYRK keeps the int8 slices of the block beside the fp64 block
      one_row += emu_bytes_per_aux_row(nao, cdiv(h->nocc_pad_cap, kBK) + 1, h->k_emu_slices, h->k_emu_pgroup) / sizeof(double) + 1024;
    size_t dbl = cap / sizeof(double);
    if (o.nblk > 0) dbl = (size_t)o.nblk * one_row;
    if (dbl < 2 * one_row) dbl = 2 * one_row;     // the density-matrix form keeps two operands per aux row
    const size_t all_rows = (size_t)(naux > 0 ? naux : 1) * one_row;
    if (dbl > all_rows && all_rows >= 2 * one_row) dbl = all_rows;
    h->X_doubles = dbl;
    h->nblk = (int)(dbl / one_row);
  }
  h->j1_chunks = (int)((h->npair + kJ1Chunk - 1) / kJ1Chunk);
  h->j2_mma_min_sets = 1;   // measured at large: k_j2 (DFMA) 3.18 / 3.39 / 4.58 ms at 1 / 4 / 8 sets, k_j2_mma 3.13 / 3.20 / 3.35
  h->j1_mma_min_sets = 3;   // measured at large: DFMA kernel 3.27 / 3.41 / 3.81 ms at 1 / 2 / 4 sets, DMMA kernel 3.43 / 3.47 / 3.51 (3.65 at 8)
  {
    const long long xcols = (long long)((h->npair + 2 * kJ2Threads - 1) / (2 * kJ2Threads));
    long long g = (148LL * 32 + xcols - 1) / xcols;
    if (g < 1) g = 1;
    if (g > 16) g = 16;
    if (g > (naux + 7) / 8) g = (naux + 7) / 8 > 0 ? (naux + 7) / 8 : 1;
    h->j2_splits = (int)g;
  }
  const int naux_pad = round_up(naux > 0 ? naux : 1, kJ1Rows);
  const size_t n2 = (size_t)nao * nao;
  bool ok = true;
  ok = ok && dev_alloc(h, &h->Ct, (size_t)h->nck * h->ct_rows * kHtLd);
  ok = ok && dev_alloc(h, &h->sgnbits, (size_t)h->ct_rows / 32 + 2);
  if (ok && cudaMemset(h->sgnbits, 0, ((size_t)h->ct_rows / 32 + 2) * sizeof(unsigned int)) != cudaSuccess) { cudaGetLastError(); ok = false; }
  ok = ok && dev_alloc(h, &h->ticket, (size_t)2);
  if (ok && cudaMemset(h->ticket, 0, 2 * sizeof(unsigned int)) != cudaSuccess) { cudaGetLastError(); ok = false; }
  ok = ok && dev_alloc(h, &h->Dw, (size_t)h->max_nset * h->npair);
  ok = ok && dev_alloc(h, &h->rho_part, (size_t)h->j1_chunks * 8 * naux_pad);
  ok = ok && dev_alloc(h, &h->rho, (size_t)h->max_nset * (naux > 0 ? naux : 1));
  // fused rho: 8 per-warp slots per (aux row, 64-row block, N tile) of the half-transform
  h->rho_ht_doubles = o.two_pass_j ? 0 : (size_t)(naux > 0 ? naux : 1) * cdiv(nao, 64) * cdiv(h->nocc_pad_cap, 16 * kHtMaxWN) * 8 * h->max_nset;
  ok = ok && dev_alloc(h, &h->rho_ht, h->rho_ht_doubles);
  ok = ok && dev_alloc(h, &h->Jp_part, (size_t)h->j2_splits * h->max_nset * h->npair);
  ok = ok && dev_alloc(h, &h->X, h->X_doubles);
  ok = ok && dev_alloc(h, &h->Kpart, (size_t)h->ksplit * h->max_nset * n2);
  ok = ok && dev_alloc(h, &h->C_stage, (size_t)nao * h->max_nocc_total);
  ok = ok && dev_alloc(h, &h->occ_stage, (size_t)h->max_nocc_total);
  ok = ok && dev_alloc(h, &h->J_stage, (size_t)h->max_nset * n2);
  ok = ok && dev_alloc(h, &h->K_stage, (size_t)h->max_nset * n2);
  if (ok && o.copy_B && naux > 0) {
    size_t ws = h->workspace_bytes;
    ok = dev_alloc(h, &h->B_owned, (size_t)naux * h->npair);
    h->workspace_bytes = ws;
    if (ok) {
      cudaError_t e = cudaMemcpy(h->B_owned, B_packed, (size_t)naux * h->npair * sizeof(double), cudaMemcpyDeviceToDevice);
      if (e != cudaSuccess) { free_all(h); delete h; cudaGetLastError(); return DFJK_ERR_CUDA; }
    }
  }
  if (!ok) { free_all(h); delete h; return DFJK_ERR_ALLOC; }
  h->B = h->B_owned ? h->B_owned : B_packed;
  h->b_aligned16 = ((uintptr_t)h->B & 15u) == 0;
  // emulated half-transform: int8 slice images of the unpacked tensor (S x 1.07 naux nao^2 bytes), built once;
  // it replaces the re-tiled fp64 copy
  if (h->ht_emu_slices > 0) {
    size_t ws = h->workspace_bytes;
    bool ok2 = dev_alloc(h, &h->Bq, emu_bq_bytes(naux > 0 ? naux : 1, nao, h->ht_emu_slices));
    h->workspace_bytes = ws;
    ok2 = ok2 && dev_alloc(h, &h->bscale, (size_t)(naux > 0 ? naux : 1) * emu_mu_q(nao));
    ok2 = ok2 && dev_alloc(h, &h->Ctq, emu_ctq_bytes(nao, h->nocc_pad_cap, h->ht_emu_slices));
    ok2 = ok2 && dev_alloc(h, &h->cscale, (size_t)emu_i_q(h->nocc_pad_cap));
    if (!ok2) { free_all(h); delete h; return DFJK_ERR_ALLOC; }
    if (naux > 0) {
      cudaError_t e = launch_emu_slice_b(h);
      if (e == cudaSuccess) e = cudaDeviceSynchronize();
      if (e != cudaSuccess) { free_all(h); delete h; cudaGetLastError(); return DFJK_ERR_CUDA; }
    }
  }
  // re-tiled copy for the half-transform (1.35x the packed bytes): used if it can be had
  if (!o.no_retile && naux > 0 && h->ht_emu_slices == 0) {
    h->bt_pstride = retile_doubles_per_aux_row(nao);
    cudaError_t e = cudaMalloc((void**)&h->Bt, (size_t)naux * h->bt_pstride * sizeof(double));
    if (e == cudaSuccess) {
      e = launch_retile(h->B, h->npair, nao, naux, h->Bt);
      if (e == cudaSuccess) e = cudaDeviceSynchronize();
      if (e != cudaSuccess) { set_err(h, "re-tiling B", e); free_all(h); delete h; cudaGetLastError(); return DFJK_ERR_CUDA; }
    } else {
      cudaGetLastError();
      h->Bt = nullptr;                       // not enough memory: gather from the packed triangle instead
    }
  }
  *out = h;
  return DFJK_OK;
}

int dfjk_get_jk(dfjk_handle h, int nset, const int* nocc, const double* C, const double* occ, double* J_out,
                double* K_out, dfjk_stream stream) {
  if (!h) return DFJK_ERR_INVALID_ARG;
  SetInfo si;
  int rc = build_setinfo(h, nset, nocc, &si);
  if (rc != DFJK_OK) return rc;
  int ntot = 0;
  for (int s = 0; s < nset; s++) ntot += nocc[s];
  if (ntot > 0 && (!C || !occ)) return DFJK_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  h->last_launches = 0;
  h->last_error[0] = 0;
  h->ev_n = 0;
  if (!on_handle_device(h)) return DFJK_ERR_INVALID_ARG;
  if (!J_out && !K_out) return DFJK_OK;
  int n = 0, k;
  // embedding-sized call: one launch does steps a1-a9 (small.cu)
  if (const int ctas = small_path_ctas(h, si)) {
    if (launch_small_fused(h, si, ctas, C, occ, J_out, K_out, st) >= 0) {
      prof_mark(h, -1, st);
      h->last_launches = 1;
      h->plan_nblk = h->naux; h->plan_ksplit = ctas; h->plan_nblocks = 1;
      cudaError_t e = cudaGetLastError();
      if (e != cudaSuccess) { set_err(h, "kernel launch", e); return DFJK_ERR_CUDA; }
      return DFJK_OK;
    }
    cudaGetLastError();          // the cooperative launch was refused (e.g. not every CTA can be resident): the tiled kernels serve the call
    h->ev_n = 0;
  }
  n += launch_prep_ct(h, si, C, occ, st);
  // both outputs: rho falls out of the half-transform, so J needs one stream over B instead of two
  const bool fuse = J_out && K_out && !h->two_pass_j && h->naux > 0 && si.nocc_pad > 0 && h->ht_emu_slices == 0;
  if (J_out && !fuse) {
    n += launch_prep_dw(h, si, st);
    k = launch_j_passes(h, si, J_out, false, st);
    if (k < 0) { set_err(h, "j pass launch", cudaGetLastError()); return DFJK_ERR_CUDA; }
    n += k;
  }
  if (K_out) {
    k = launch_k_path(h, si, K_out, fuse, st);
    if (k == -2) {
      snprintf(h->last_error, sizeof(h->last_error), "workspace cap too small for one aux row of the emulated K path (or k_emulation_group x columns of a set >= 87381: int32 accumulators)");
      return DFJK_ERR_INVALID_ARG;
    }
    if (k < 0) { set_err(h, "k path launch", cudaGetLastError()); return DFJK_ERR_CUDA; }
    n += k;
  }
  if (fuse) {
    k = launch_j_passes(h, si, J_out, true, st);
    if (k < 0) { set_err(h, "j pass launch", cudaGetLastError()); return DFJK_ERR_CUDA; }
    n += k;
  }
  prof_mark(h, -1, st);
  h->last_launches = n;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err(h, "kernel launch", e); return DFJK_ERR_CUDA; }
  return DFJK_OK;
}

int dfjk_get_jk_host(dfjk_handle h, int nset, const int* nocc, const double* C, const double* occ, double* J_out,
                     double* K_out, dfjk_stream stream) {
  if (!h) return DFJK_ERR_INVALID_ARG;
  SetInfo si;
  int rc = build_setinfo(h, nset, nocc, &si);
  if (rc != DFJK_OK) return rc;
  size_t ntot = 0;
  for (int s = 0; s < nset; s++) ntot += (size_t)nocc[s];
  if (ntot > 0 && (!C || !occ)) return DFJK_ERR_INVALID_ARG;
  if (!on_handle_device(h)) return DFJK_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaSuccess;
  if (ntot > 0) {
    e = cudaMemcpyAsync(h->C_stage, C, ntot * h->nao * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h->occ_stage, occ, ntot * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) { set_err(h, "H2D copy", e); cudaGetLastError(); return DFJK_ERR_CUDA; }
  }
  rc = dfjk_get_jk(h, nset, nocc, h->C_stage, h->occ_stage, J_out ? h->J_stage : nullptr,
                   K_out ? h->K_stage : nullptr, stream);
  if (rc != DFJK_OK) return rc;
  const size_t bytes = (size_t)nset * h->nao * h->nao * sizeof(double);
  if (J_out) e = cudaMemcpyAsync(J_out, h->J_stage, bytes, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess && K_out) e = cudaMemcpyAsync(K_out, h->K_stage, bytes, cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) { set_err(h, "D2H copy / sync", e); cudaGetLastError(); return DFJK_ERR_CUDA; }
  return DFJK_OK;
}

int dfjk_get_jk_dm(dfjk_handle h, int nset, const double* D, double* J_out, double* K_out, dfjk_stream stream) {
  if (!h) return DFJK_ERR_INVALID_ARG;
  if (nset < 1 || nset > h->max_nset || !D) return DFJK_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  h->last_launches = 0;
  h->last_error[0] = 0;
  h->ev_n = 0;
  if (!on_handle_device(h)) return DFJK_ERR_INVALID_ARG;
  if (!J_out && !K_out) return DFJK_OK;
  int n = 0;
  if (J_out) {
    SetInfo si;
    memset(&si, 0, sizeof(si));
    si.nset = nset;
    n += launch_prep_dw_dm(h, nset, D, st);
    const int kj = launch_j_passes(h, si, J_out, false, st);
    if (kj < 0) { set_err(h, "j pass launch", cudaGetLastError()); return DFJK_ERR_CUDA; }
    n += kj;
  }
  if (K_out) {
    const int k = launch_k_path_dm(h, nset, D, K_out, st);
    if (k == -2) {
      snprintf(h->last_error, sizeof(h->last_error), "workspace or column capacity too small for the density-matrix form");
      return DFJK_ERR_INVALID_ARG;
    }
    if (k < 0) { set_err(h, "k path launch", cudaGetLastError()); return DFJK_ERR_CUDA; }
    n += k;
  }
  prof_mark(h, -1, st);
  h->last_launches = n;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err(h, "kernel launch", e); return DFJK_ERR_CUDA; }
  return DFJK_OK;
}

int dfjk_ao2mo(dfjk_handle h, int nmo, int a0, int nact, const double* M, double* bpa_out, double* ppaa_out,
               double* papa_out, dfjk_stream stream) {
  if (!h) return DFJK_ERR_INVALID_ARG;
  if (nmo < 0 || nmo > h->max_nocc_total || round_up(nmo, 8) > h->nocc_pad_cap) return DFJK_ERR_INVALID_ARG;
  if (nact < 0 || a0 < 0 || a0 + nact > nmo) return DFJK_ERR_INVALID_ARG;
  if (nmo > 0 && !M) return DFJK_ERR_INVALID_ARG;
  if (nmo > 0 && nact > 0 && h->naux > 0 && !bpa_out) return DFJK_ERR_INVALID_ARG;
  if ((long long)nmo * nmo > 2147483647LL || (long long)nmo * nact > 2147483647LL) return DFJK_ERR_INVALID_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  h->last_launches = 0;
  h->last_error[0] = 0;
  h->ev_n = 0;
  if (!on_handle_device(h)) return DFJK_ERR_INVALID_ARG;
  const int n = launch_ao2mo(h, nmo, a0, nact, M, bpa_out, ppaa_out, papa_out, st);
  if (n == -2) { snprintf(h->last_error, sizeof(h->last_error), "workspace cap too small for one aux row of AO2MO"); return DFJK_ERR_INVALID_ARG; }
  if (n < 0) { set_err(h, "ao2mo launch", cudaGetLastError()); return DFJK_ERR_CUDA; }
  h->last_launches = n;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { set_err(h, "kernel launch", e); return DFJK_ERR_CUDA; }
  return DFJK_OK;
}

int dfjk_destroy(dfjk_handle h) {
  if (!h) return DFJK_OK;
  free_all(h);
  delete h;
  return DFJK_OK;
}

const char* dfjk_last_error(dfjk_handle h) { return h ? h->last_error : ""; }

size_t dfjk_workspace_bytes(dfjk_handle h) { return h ? h->workspace_bytes : 0; }

int dfjk_get_plan(dfjk_handle h, int* nblk, int* ksplit, int* nocc_pad_capacity, int* retiled) {
  if (!h) return DFJK_ERR_INVALID_ARG;
  if (nblk) *nblk = h->plan_nblk ? h->plan_nblk : h->nblk;
  if (ksplit) *ksplit = h->plan_ksplit ? h->plan_ksplit : h->ksplit;
  if (nocc_pad_capacity) *nocc_pad_capacity = h->nocc_pad_cap;
  if (retiled) *retiled = h->Bt ? 1 : 0;
  return DFJK_OK;
}

int dfjk_last_launch_count(dfjk_handle h) { return h ? h->last_launches : 0; }

int dfjk_last_ao2mo_route(dfjk_handle h) { return h ? h->plan_ao2mo_route : 0; }

int dfjk_set_profiling(dfjk_handle h, int on) {
  if (!h) return DFJK_ERR_INVALID_ARG;
  if (on && !h->ev && !prof_grow(h)) return DFJK_ERR_ALLOC;
  h->profiling = on ? 1 : 0;
  h->ev_n = 0;
  return DFJK_OK;
}

int dfjk_get_profile(dfjk_handle h, double* ms, int* groups) {
  if (!h || !ms || !groups) return DFJK_ERR_INVALID_ARG;
  for (int p = 0; p < DFJK_NUM_PHASES; p++) { ms[p] = 0.0; groups[p] = 0; }
  if (h->ev_n < 2) return DFJK_OK;
  cudaError_t e = cudaEventSynchronize(h->ev[h->ev_n - 1]);
  if (e != cudaSuccess) { set_err(h, "event sync", e); cudaGetLastError(); return DFJK_ERR_CUDA; }
  for (int i = 0; i + 1 < h->ev_n; i++) {
    const int p = h->ev_phase[i];
    if (p < 0 || p >= DFJK_NUM_PHASES) continue;
    float t = 0.f;
    if (cudaEventElapsedTime(&t, h->ev[i], h->ev[i + 1]) != cudaSuccess) { cudaGetLastError(); continue; }
    ms[p] += t;
    groups[p] += 1;
  }
  return DFJK_OK;
}

int dfjk_selftest_dmma(void) {
  const int bad = run_dmma_selftest();
  if (bad < 0) return DFJK_ERR_CUDA;
  return bad == 0 ? DFJK_OK : DFJK_ERR_UNSUPPORTED_ARCH;
}

}  // extern "C"
