/*
 * dfjk.h -- C ABI of the B200-native density-fitted Coulomb/exchange (JK) build.
 *
 * The operation is the "JK call" of arxiv 2505.03755, section 2.D.i:
 *   "the input is a density matrix and the AO ... Cholesky vectors and the output is J and K"
 *   (PAPER.md:148), with
 *      rho_P     = sum_{mu,nu} b^P_{mu nu} D_{mu nu}                        Eq. 14
 *      J_{mu nu} = sum_P rho_P b^P_{mu nu}                                  Eq. 15
 *      X^P_{mu i} = sum_lam b^P_{mu lam} C_{lam i}      Eq. 16 with gamma = C n C^T;
 *                                                       the half-transform of Eq. 18
 *      K_{mu nu} = sum_P sum_i n_i X^P_{mu i} X^P_{nu i}                    Eq. 17
 *   for every density set s, D_s = C_s diag(n_s) C_s^T.  The Cholesky vectors are "stored in
 *   triangular form of size Naux*Nao(Nao+1)/2" and unpacked on the GPU; they are
 *   kept resident on the GPU across calls; a call allocates nothing and never
 *   blocks the host; init/destroy pair as in PAPER.md:227,242.
 *
 * Everything is fp64.  All matrices are row-major (C order).  Every step runs in hand-written
 * CUDA kernels for sm_100a; there is no CPU fallback and no library GEMM.
 *
 * Threading: one in-flight call per handle (calls on one handle must be stream-ordered);
 * different handles are independent.  No function throws, aborts or prints.
 */
#ifndef DFJK_H
#define DFJK_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dfjk_ctx* dfjk_handle; /* opaque */

/* CUDA stream, passed as an opaque pointer so that this header needs no CUDA include
 * (it is a cudaStream_t / CUstream; NULL is the legacy default stream). */
typedef void* dfjk_stream;

enum {
  DFJK_OK = 0,
  DFJK_ERR_INVALID_ARG = 1,      /* NULL / shape / nocc[s] outside [0,nao] / capacity exceeded / misaligned B */
  DFJK_ERR_ALLOC = 2,            /* device or host allocation failed (create only) */
  DFJK_ERR_CUDA = 3,             /* a CUDA call or launch failed; text via dfjk_last_error() */
  DFJK_ERR_UNSUPPORTED_ARCH = 4  /* the current device is not compute capability 10.x */
};

/* All fields optional; zero = default.  Pass NULL for all defaults. */
typedef struct {
  size_t workspace_cap_bytes; /* cap for the half-transformed block X (step a8);
                                 default min(4 GiB, a tenth of the free device memory at
                                 create).  nblk = floor(cap / bytes of one aux row of X) >= 1 */
  int nblk;                   /* force the aux block size N_blk; 0 = derive from cap */
  int max_nocc_total;         /* capacity for sum_s nocc[s]; 0 = nao */
  int max_nset;               /* capacity for nset; 0 = 8 */
  int copy_B;                 /* 0 = borrow the caller's device pointer (default); 1 = private copy */
  int ksplit;                 /* force the split-K factor of the SYRK; 0 = automatic */
  int no_retile;              /* 0 = dfjk_create also builds a re-tiled private copy of B for the
                                 half-transform (1.35x the packed bytes, not counted in
                                 dfjk_workspace_bytes; silently skipped if the allocation fails);
                                 1 = never: the half-transform gathers from the packed triangle */
  int ao2mo_route;            /* dfjk_ao2mo: 0 = the cheaper of the two routes; 1 = Eq. 18-21 in the printed
                                 order (forms bmo^P per aux block); 2 = "active first" (Eq. 18-19 for the
                                 active columns only, Eq. 20 contracted over P in the AO basis and then
                                 transformed; falls back to 1 if its scratch does not fit the workspace) */
  int two_pass_j;             /* 0 = when J and K are both requested, rho (Eq. 14) is taken from the
                                 half-transformed block, rho_P = sum_{mu,i} X^P_{mu i} C'_{mu i}, and B is
                                 streamed twice instead of three times; 1 = always the two-pass J */
  int k_emulation_slices;     /* 0 = K on the native FP64 tensor instruction (default).  3..6 = opt-in FP64
                                 emulation of the SYRK (Eq. 17) on the int8 tensor cores (the paper's
                                 reduced-precision outlook): X is split into that many signed
                                 7-bit slices against a power-of-two scale per AO row and group of aux rows,
                                 the slice products are exact in int32, the recombination is fp64.  Error
                                 bound per element: (S+2) 2^(-7S) sum over groups of
                                 (terms) 2^(e_mu + e_nu); 6 slices keep max|dK|/max|K| <= 1e-10 */
  int k_emulation_group;      /* aux rows sharing one scale per AO row in the emulated SYRK; 0 = 16, <= 64.  The int32
                                 accumulators bound group x (columns of the widest set, rounded up to 32) x slices
                                 below 2^19 = 524288; dfjk_get_jk returns DFJK_ERR_INVALID_ARG past that */
  int ht_emulation_slices;    /* 0 = half-transform (Eq. 16 / 18) on the native FP64 tensor instruction (default).
                                 3..6 = opt-in emulation on the int8 tensor cores: dfjk_create builds int8 slice
                                 images of the unpacked tensor (S x 1.07 naux nao^2 bytes, one power-of-two scale
                                 per row of every slice b^P; replaces the re-tiled copy), C' is sliced per call
                                 (one scale per column).  Error per element of X: <= (S+2) 2^(-7S) nao 2^(e_row +
                                 e_col).  With this option rho always comes from the two-pass J */
  int no_symm_thin;           /* 0 = a half-transform with at most 8 columns (the active columns of dfjk_ao2mo's
                                 "active first" route; a dfjk_get_jk call on ONE set of at most 8 orbitals) streams
                                 the packed triangle once and uses every stored element for both Z[mu] and Z[lam]
                                 (needs a 16-byte aligned B; one launch per 1280 columns of the basis); 1 = always
                                 the tiled half-transform */
  int no_small_path;          /* 0 = an embedding-sized dfjk_get_jk (nao <= 96, nao * sum(nocc) <= 4608 and
                                 naux * nao^2 * (sum(nocc) + nset) <= 2^26, 2^27 for one set) runs as ONE kernel launch: the call is
                                 launch-latency bound there ("called thousands of times");
                                 dfjk_last_launch_count then returns 1.  1 = always the tiled kernels */
} dfjk_options;

/*
 * dfjk_create -- bind a resident packed tensor and allocate every scratch buffer (step a0).
 *   naux, nao   sizes, naux >= 0, nao >= 1.
 *   B_packed    DEVICE pointer, naux * nao(nao+1)/2 doubles, 8-byte aligned; 16-byte alignment (what
 *               cudaMalloc and row slices of an even-npair tensor give) lets the J passes use bulk
 *               copies and 128-bit loads, otherwise they fall back to scalar loads.  Aux index P
 *               slowest, then the row-major lower triangle: B[P][mu(mu+1)/2 + nu], mu >= nu
 *               (PAPER.md:152).  A contiguous range of aux rows of a larger tensor is a valid B: J and
 *               K are sums over P, so handles on disjoint row ranges return partial results that add
 *               up to the full ones (the aux-sharded mode).
 *               Borrowed unless opt->copy_B: it must stay valid and unchanged until dfjk_destroy.
 *   opt         options or NULL.
 *   out         receives the handle.
 * Allocates on the CURRENT device; may synchronise.  Every later call on the handle must be made
 * with that device current (DFJK_ERR_INVALID_ARG otherwise); handles on different devices of one
 * process are independent.  Returns DFJK_OK or an error code (then *out = NULL).
 */
int dfjk_create(int naux, int nao, const double* B_packed, const dfjk_options* opt, dfjk_handle* out);

/*
 * dfjk_get_jk -- J and K of nset densities D_s = C_s diag(occ_s) C_s^T (steps a1-a9).
 *   nset     number of sets, 1 <= nset <= max_nset (<= 32).  The J passes hold 8 sets per pass: more
 *            than 8 sets stream B once per pass for every group of 8.
 *   nocc     HOST array, length nset; 0 <= nocc[s] <= nao, sum <= max_nocc_total.
 *            nocc[s] = 0 gives J_s = K_s = 0.
 *   C        DEVICE, blocks [C_0 | C_1 | ...] one after another; block s is row-major
 *            nao x nocc[s].  Columns need not be orthonormal.
 *   occ      DEVICE, concatenated occupations, length sum nocc[s]; any sign (differences of
 *            densities): the kernels work with C' = C sqrt(|occ|) and carry
 *            sign(occ) as a sign-bit flip, D = C' diag(sign occ) C'^T exactly, at the same cost.
 *   J_out    DEVICE, nset x nao x nao, or NULL to skip J.
 *   K_out    DEVICE, nset x nao x nao, or NULL to skip K.
 *   stream   all work is enqueued on this stream.
 * Outputs are overwritten (not accumulated), full squares, both triangles, bitwise symmetric, raw
 * J[D_s], K[D_s] (no factor 1/2, no subtraction: Eq. 13 is the caller's).  The call only
 * enqueues: it never allocates and never synchronises the host (so it may be captured into a
 * CUDA graph and replayed).  Results are deterministic (bitwise equal from run to run for equal
 * inputs and options).
 */
int dfjk_get_jk(dfjk_handle h, int nset, const int* nocc, const double* C, const double* occ,
                double* J_out, double* K_out, dfjk_stream stream);

/*
 * dfjk_get_jk_host -- the same call with HOST buffers, as the paper states it: the density
 * (here C, occ) is pushed, J and K are pulled back ("transfer them back to the
 * CPU"); B stays resident.  C, occ, J_out, K_out are HOST pointers (pinned memory makes the
 * copies asynchronous).  Copies in, runs dfjk_get_jk on the handle's staging
 * buffers, copies out and synchronises `stream` before returning.
 */
int dfjk_get_jk_host(dfjk_handle h, int nset, const int* nocc, const double* C, const double* occ,
                     double* J_out, double* K_out, dfjk_stream stream);

/*
 * dfjk_get_jk_dm -- the JK call stated with density matrices, Eq. 14-17 exactly as printed
 * ("the input is a density matrix ..."), for densities that have no
 * C diag(occ) C^T form with occ >= 0 (differences of densities, transition densities):
 *      rho_P = sum b^P_{mu nu} D_{mu nu},  J = sum_P rho_P b^P                 Eq. 14-15
 *      V^P = b^P D (Eq. 16),  K = sum_P V^P b^P (Eq. 17)
 *   D        DEVICE, nset x nao x nao row-major; every D_s must be symmetric (J uses its symmetric
 *            part; K = sum_P b^P D b^P is computed on the lower triangle and mirrored).
 *   J_out, K_out, stream: as in dfjk_get_jk.  1 <= nset <= max_nset; needs max_nocc_total >= nao
 *            (the default).  Costs 3 naux nao^3 flop per set for K instead of 3 naux nao^2 nocc.
 */
int dfjk_get_jk_dm(dfjk_handle h, int nset, const double* D, double* J_out, double* K_out, dfjk_stream stream);

/*
 * dfjk_small_jk_static -- dfjk_get_jk for embedding-sized calls WITHOUT a handle and without
 * any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, serving loops, harnesses
 * that forbid it).  One cooperative launch of the single-launch kernel (steps a1-a9, Eq. 14-17);
 * its scratch (private J/K partials of every CTA and two barrier counters) is a file-scope device array of
 * DFJK_STATIC_SCRATCH_BYTES (+ 256) bytes that every GPU loading the library holds until the process exits.
 *   naux, nao  >= 1;   B_packed  DEVICE, naux x nao(nao+1)/2, packed lower triangle as in dfjk_create (borrowed).
 *   nset, nocc, C, occ, J_out, K_out, stream: as in dfjk_get_jk (nocc HOST; C, occ, J_out, K_out DEVICE).
 * Maximum sizes (beyond them: DFJK_ERR_INVALID_ARG, the text in dfjk_small_jk_static_last_error):
 *   nao <= 96, nset <= DFJK_STATIC_MAX_NSET, 1 <= sum(nocc), nao * sum(nocc) <= 4608,
 *   naux * nao^2 * (sum(nocc) + nset) <= 2^26.
 * The number of CTAs is that of dfjk_get_jk's single-launch path, capped so that the partials
 * (CTAs * nset * (nao^2 + nao(nao+1)/2) doubles) fit the array; with fewer CTAs the sums run in another order, so
 * results agree with dfjk_get_jk to rounding (and bitwise when the cap does not bind), and are deterministic.
 * The call enqueues one 8-byte memset (the barrier counters must start at zero; the array keeps the last call's
 * contents, the partials are overwritten before they are read) and one kernel on `stream`; it calls no cudaMalloc,
 * cudaFree or allocating library routine and never synchronises the host.  The first call on a device looks up the
 * array's device address (cudaGetSymbolAddress, once per device, with that device current) and opts the kernel in to
 * its shared memory: make one call before starting a stream capture, later calls can be captured and replayed.
 * EVERY call on a device shares the one array: calls that overlap on the GPU (two streams, two host threads, two
 * graphs in flight) race on it -- serialise them.  Calls on one stream are ordered and safe.
 */
#define DFJK_STATIC_SCRATCH_BYTES 8388608
#define DFJK_STATIC_MAX_NSET 8
int dfjk_small_jk_static(int naux, int nao, const double* B_packed, int nset, const int* nocc, const double* C,
                         const double* occ, double* J_out, double* K_out, dfjk_stream stream);

/* Text of the last failure of dfjk_small_jk_static on the calling thread ("" if none). */
const char* dfjk_small_jk_static_last_error(void);

/*
 * dfjk_ao2mo -- the AO2MO kernel of section 2.D.ii (Eq. 18-21) on the same
 * resident Cholesky vectors, with the index pattern fixed by Eq. 12, g = (m1 m2|m3 m4) = b b:
 *      X^P[e2][p1]   = sum_{e1} b^P[e1][e2] M[e1][p1]                          Eq. 18
 *      bmo^P[p1][p2] = sum_{e2} X^P[e2][p1] M[e2][p2]                          Eq. 19
 *      ppaa[p1][p2][a1][a2] = sum_P bmo^P[p1][p2] bmo^P[a0+a1][a0+a2]          Eq. 20
 *      papa[p1][a1][p2][a2] = sum_P bmo^P[p1][a0+a1] bmo^P[p2][a0+a2]          Eq. 21
 *   nmo      number of MO columns, 0 <= nmo <= max_nocc_total (default nao).
 *   a0,nact  the active orbitals are the MO columns [a0, a0 + nact), a0 + nact <= nmo.
 *   M        DEVICE, nao x nmo row-major, M[e][p]; columns need not be orthonormal.
 *   bpa_out  DEVICE, naux x nmo x nact: bpa[P][p][a] = bmo^P[p][a0+a], the block the paper pulls
 *            back to the host.  Required (it is also the operand of Eq. 21).
 *   ppaa_out DEVICE, nmo x nmo x nact x nact, or NULL to skip Eq. 20.
 *   papa_out DEVICE, nmo x nact x nmo x nact, or NULL to skip Eq. 21 (the paper runs it on the CPU).  Computed on the
 *            tiles at and below the diagonal of the (p1 a1) x (p2 a2) matrix and mirrored: bitwise symmetric.
 * Same conventions as dfjk_get_jk: enqueue-only on `stream`, no allocation, no host
 * synchronisation, outputs overwritten, deterministic.  The aux blocks share the X workspace of
 * the handle (per aux row nao*roundup(nmo,8) + nmo^2 + nact^2 doubles); if the cap
 * cannot hold one row the call returns DFJK_ERR_INVALID_ARG.  Must not overlap a dfjk_get_jk on
 * the same handle.
 */
int dfjk_ao2mo(dfjk_handle h, int nmo, int a0, int nact, const double* M, double* bpa_out, double* ppaa_out,
               double* papa_out, dfjk_stream stream);

/* Route the last dfjk_ao2mo took on this handle: 1 = Eq. 18-21 in the printed order, 2 = active first
 * (see dfjk_options.ao2mo_route); 0 before the first call. */
int dfjk_last_ao2mo_route(dfjk_handle h);

/* Frees everything the handle owns.  dfjk_destroy(NULL) is a no-op returning DFJK_OK. */
int dfjk_destroy(dfjk_handle h);

/* Static text for an error code. */
const char* dfjk_strerror(int code);

/* Text of the last CUDA failure seen on this handle ("" if none).  Valid until the next call. */
const char* dfjk_last_error(dfjk_handle h);

/* Bytes of device scratch the handle owns (excluding a private copy of B). */
size_t dfjk_workspace_bytes(dfjk_handle h);

/* Plan of the last/next call, for tests and the bench: aux block size, SYRK split-K factor, padded
 * column capacity of X, and whether the half-transform reads the re-tiled private copy of B
 * (1) or gathers from the packed triangle (0: option no_retile, or the copy did not fit the
 * device memory at create).  After a single-launch call (option no_small_path) nblk = naux and ksplit =
 * the number of CTAs of that launch.  Any pointer may be NULL. */
int dfjk_get_plan(dfjk_handle h, int* nblk, int* ksplit, int* nocc_pad_capacity, int* retiled);

/* Number of kernel launches dfjk_get_jk enqueued in its last call on this handle. */
int dfjk_last_launch_count(dfjk_handle h);

/*
 * Optional per-phase profile with CUDA events recorded on the launching stream (the paper used
 * wall-clock timers per stage and Nsight timelines).  Off by default.
 * dfjk_set_profiling(h, 1) makes every later dfjk_get_jk record an event at each phase boundary
 * (a few microseconds each; the event pool grows with the number of aux blocks).
 * dfjk_get_profile synchronises on the last event of the last call and returns, per phase, the
 * summed milliseconds and the number of kernel-launch groups.  dfjk_ao2mo records too: HALF_TRANSFORM =
 * the Eq. 18 launches, SYRK = the contractions of Eq. 19-21, PREP = everything else.
 */
enum {
  DFJK_PHASE_PREP = 0,           /* a1: C' and packed weighted density */
  DFJK_PHASE_J1 = 1,             /* a2: rho = <B_P, D>   (includes the tiny chunk reduce) */
  DFJK_PHASE_J2 = 2,             /* a3: Jp = sum_P rho_P B_P */
  DFJK_PHASE_J_EPILOGUE = 3,     /* a4 */
  DFJK_PHASE_HALF_TRANSFORM = 4, /* a5+a6 */
  DFJK_PHASE_SYRK = 5,           /* a7 */
  DFJK_PHASE_K_EPILOGUE = 6,     /* a9 (and zero fills) */
  DFJK_NUM_PHASES = 7
};
int dfjk_set_profiling(dfjk_handle h, int on);
int dfjk_get_profile(dfjk_handle h, double* ms /* [DFJK_NUM_PHASES] */, int* groups /* [DFJK_NUM_PHASES] */);

/* 1-warp self-test of the DMMA.8x8x4 fragment mapping against a scalar loop on the device
 * (synchronises).  Returns DFJK_OK if the mapping assumed by the kernels holds. */
int dfjk_selftest_dmma(void);

#ifdef __cplusplus
}
#endif
#endif /* DFJK_H */
