/*
 * ao2mo_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the AO2MO kernel of arxiv 2505.03755, section 2.D.ii
 * (Eq. 18-21; repeated as SI Eq. 1-4), written from the
 * definitions so a reader can check it against the paper by eye.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline leg may build, load or call this file.  It
 * shares no code, header, table or helper with the CUDA path (paper_2505_03755_b200/csrc).
 *
 * Conventions (rows R1, R2, R9, R15):
 *   - Bp is the packed Cholesky tensor b^P_{e1 e2} over the basis the MO coefficients are given in
 *     (AO or embedding basis, "e" in Eq. 18): aux index P slowest, then the row-major lower
 *     triangle idx(e1,e2) = e1(e1+1)/2 + e2 for e1 >= e2; b^P is symmetric.
 *   - M is nao x nmo row-major, M[e][p] = M_e^p "the matrix of MO coefficients that transforms
 *     from AO basis to MO basis".  Columns need not be orthonormal.
 *   - The active orbitals a are the MO columns [a0, a0 + nact).
 *   - Eq. 12's convention g^{m1 m3}_{m2 m4} = b_{m1 m2} b_{m3 m4} = (m1 m2|m3 m4) fixes the index
 *     pattern of Eq. 20-21 (the printed Eq. 19-21 are garbled and repeated):
 *        Eq. 18  bh^P[e2][p1]  = sum_{e1} b^P[e1][e2] M[e1][p1]
 *        Eq. 19  bmo^P[p1][p2] = sum_{e2} bh^P[e2][p1] M[e2][p2]
 *        Eq. 20  ppaa[p1][p2][a1][a2] = sum_P bmo^P[p1][p2] bmo^P[a0+a1][a0+a2]   = (p1 p2|a1 a2)
 *        Eq. 21  papa[p1][a1][p2][a2] = sum_P bmo^P[p1][a0+a1] bmo^P[p2][a0+a2]   = (p1 a1|p2 a2)
 *     and bpa[P][p][a] = bmo^P[p][a0+a] is the block the paper pulls back to the host
 *     ("b^P_{pa}").
 *
 * No symmetry shortcut, no blocking over P, no tiling; P ascending.  OpenMP splits OUTPUT rows
 * only, so every output element is summed in the same order whatever the thread count.
 *
 * Pins (tests/test_ao2mo_oracle_pins.py, -m "not gpu"): the direct 4-index transformation of the
 * Eq. 12 tensor (brute force below, itself checked against numpy.einsum), M = I (ppaa, papa are
 * slices of the AO 4-index tensor), permutational symmetries, the overlap of the two outputs on
 * all-active indices, an independent numpy.einsum evaluation, and the contraction with an active
 * density against the pinned JK oracle:  sum_{a1 a2} ppaa[..] D[a1][a2] = M^T J[D_ao] M,
 * sum_{a1 a2} papa[..] D[a1][a2] = M^T K[D_ao] M with D_ao = M_act D M_act^T.
 */
#include <stddef.h>
#include <stdlib.h>
#include <string.h>

#define DFJK_ORACLE_OK 0
#define DFJK_ORACLE_ERR_ARG 1
#define DFJK_ORACLE_ERR_ALLOC 2

static void unpack(int nao, const double* BpP, double* Bsq) {
  for (int e1 = 0; e1 < nao; e1++)
    for (int e2 = 0; e2 <= e1; e2++) {
      double v = BpP[(size_t)e1 * (e1 + 1) / 2 + e2];
      Bsq[(size_t)e1 * nao + e2] = v;
      Bsq[(size_t)e2 * nao + e1] = v;
    }
}

/*
 * Eq. 18-21, aux slice after aux slice.
 *   bmo_out  naux x nmo x nmo   or NULL      (Eq. 19, every slice)
 *   bpa_out  naux x nmo x nact  or NULL
 *   ppaa     nmo x nmo x nact x nact or NULL (Eq. 20)
 *   papa     nmo x nact x nmo x nact or NULL (Eq. 21)
 */
int dfjk_oracle_ao2mo(int naux, int nao, int nmo, int a0, int nact, const double* M, const double* Bp,
                      double* bmo_out, double* bpa_out, double* ppaa, double* papa) {
  if (naux < 0 || nao < 1 || nmo < 0 || nact < 0 || a0 < 0 || a0 + nact > nmo) return DFJK_ORACLE_ERR_ARG;
  const size_t npair = (size_t)nao * (nao + 1) / 2;
  const size_t n2 = (size_t)nmo * nmo, na2 = (size_t)nact * nact;
  if (ppaa) memset(ppaa, 0, n2 * na2 * sizeof(double));
  if (papa) memset(papa, 0, n2 * na2 * sizeof(double));
  double* Bsq = (double*)malloc((size_t)nao * nao * sizeof(double));
  double* bh = (double*)malloc(((size_t)nao * nmo + 1) * sizeof(double));
  double* bmo = (double*)malloc((n2 + 1) * sizeof(double));
  if (!Bsq || !bh || !bmo) {
    free(Bsq); free(bh); free(bmo);
    return DFJK_ORACLE_ERR_ALLOC;
  }
  for (int P = 0; P < naux; P++) {
    unpack(nao, Bp + (size_t)P * npair, Bsq);
    /* Eq. 18 */
#pragma omp parallel for schedule(static)
    for (int e2 = 0; e2 < nao; e2++)
      for (int p1 = 0; p1 < nmo; p1++) {
        double s = 0.0;
        for (int e1 = 0; e1 < nao; e1++) s += Bsq[(size_t)e1 * nao + e2] * M[(size_t)e1 * nmo + p1];
        bh[(size_t)e2 * nmo + p1] = s;
      }
    /* Eq. 19 */
#pragma omp parallel for schedule(static)
    for (int p1 = 0; p1 < nmo; p1++)
      for (int p2 = 0; p2 < nmo; p2++) {
        double s = 0.0;
        for (int e2 = 0; e2 < nao; e2++) s += bh[(size_t)e2 * nmo + p1] * M[(size_t)e2 * nmo + p2];
        bmo[(size_t)p1 * nmo + p2] = s;
      }
    if (bmo_out) memcpy(bmo_out + (size_t)P * n2, bmo, n2 * sizeof(double));
    if (bpa_out)
      for (int p = 0; p < nmo; p++)
        for (int a = 0; a < nact; a++)
          bpa_out[((size_t)P * nmo + p) * nact + a] = bmo[(size_t)p * nmo + a0 + a];
    /* Eq. 20 */
    if (ppaa) {
#pragma omp parallel for schedule(static)
      for (int p1 = 0; p1 < nmo; p1++)
        for (int p2 = 0; p2 < nmo; p2++)
          for (int a1 = 0; a1 < nact; a1++)
            for (int a2 = 0; a2 < nact; a2++)
              ppaa[(((size_t)p1 * nmo + p2) * nact + a1) * nact + a2] +=
                  bmo[(size_t)p1 * nmo + p2] * bmo[(size_t)(a0 + a1) * nmo + a0 + a2];
    }
    /* Eq. 21 */
    if (papa) {
#pragma omp parallel for schedule(static)
      for (int p1 = 0; p1 < nmo; p1++)
        for (int a1 = 0; a1 < nact; a1++)
          for (int p2 = 0; p2 < nmo; p2++)
            for (int a2 = 0; a2 < nact; a2++)
              papa[(((size_t)p1 * nact + a1) * nmo + p2) * nact + a2] +=
                  bmo[(size_t)p1 * nmo + a0 + a1] * bmo[(size_t)p2 * nmo + a0 + a2];
    }
  }
  free(Bsq); free(bh); free(bmo);
  return DFJK_ORACLE_OK;
}

/*
 * Brute force for tiny shapes: the AO 4-index tensor of Eq. 12,
 *   g[e1][e2][e3][e4] = sum_P b^P[e1][e2] b^P[e3][e4] = (e1 e2|e3 e4),
 * transformed index by index with M in one eight-fold loop nest:
 *   ppaa[p1][p2][a1][a2] = sum_{e1 e2 e3 e4} M[e1][p1] M[e2][p2] M[e3][a0+a1] M[e4][a0+a2] g[e1][e2][e3][e4]
 *   papa[p1][a1][p2][a2] = sum_{e1 e2 e3 e4} M[e1][p1] M[e2][a0+a1] M[e3][p2] M[e4][a0+a2] g[e1][e2][e3][e4]
 * Cost O(nao^4 (naux + nmo^2 nact^2)).
 */
int dfjk_oracle_ao2mo_bruteforce(int naux, int nao, int nmo, int a0, int nact, const double* M,
                                 const double* Bp, double* ppaa, double* papa) {
  if (naux < 0 || nao < 1 || nao > 16 || nmo < 0 || nact < 0 || a0 < 0 || a0 + nact > nmo)
    return DFJK_ORACLE_ERR_ARG;
  const size_t npair = (size_t)nao * (nao + 1) / 2;
  const size_t n = (size_t)nao, n4 = n * n * n * n;
  double* g = (double*)calloc(n4, sizeof(double));
  double* Bsq = (double*)malloc(n * n * sizeof(double));
  if (!g || !Bsq) {
    free(g); free(Bsq);
    return DFJK_ORACLE_ERR_ALLOC;
  }
  for (int P = 0; P < naux; P++) {
    unpack(nao, Bp + (size_t)P * npair, Bsq);
    for (size_t e1 = 0; e1 < n; e1++)
      for (size_t e2 = 0; e2 < n; e2++)
        for (size_t e3 = 0; e3 < n; e3++)
          for (size_t e4 = 0; e4 < n; e4++)
            g[((e1 * n + e2) * n + e3) * n + e4] += Bsq[e1 * n + e2] * Bsq[e3 * n + e4];
  }
  for (int p1 = 0; p1 < nmo; p1++)
    for (int p2 = 0; p2 < nmo; p2++)
      for (int a1 = 0; a1 < nact; a1++)
        for (int a2 = 0; a2 < nact; a2++) {
          double s20 = 0.0, s21 = 0.0;
          for (size_t e1 = 0; e1 < n; e1++)
            for (size_t e2 = 0; e2 < n; e2++)
              for (size_t e3 = 0; e3 < n; e3++)
                for (size_t e4 = 0; e4 < n; e4++) {
                  const double gv = g[((e1 * n + e2) * n + e3) * n + e4];
                  s20 += M[e1 * nmo + p1] * M[e2 * nmo + p2] * M[e3 * nmo + a0 + a1] * M[e4 * nmo + a0 + a2] * gv;
                  s21 += M[e1 * nmo + p1] * M[e2 * nmo + a0 + a1] * M[e3 * nmo + p2] * M[e4 * nmo + a0 + a2] * gv;
                }
          if (ppaa) ppaa[(((size_t)p1 * nmo + p2) * nact + a1) * nact + a2] = s20;
          if (papa) papa[(((size_t)p1 * nact + a1) * nmo + p2) * nact + a2] = s21;
        }
  free(g); free(Bsq);
  return DFJK_ORACLE_OK;
}

/*
 * Single elements of Eq. 20 and Eq. 21 straight from the definitions, for parity at sizes where
 * the full outputs (nmo^2 nact^2 entries over naux slices) are too slow to form on the host:
 *   bmo^P[p][q] = sum_{e1} sum_{e2} M[e1][p] b^P[e1][e2] M[e2][q]                      (Eq. 18-19)
 *   ppaa_v[t] = sum_P bmo^P[p1][p2] bmo^P[a0+a1][a0+a2]   at (p1,p2,a1,a2) = sample t   (Eq. 20)
 *   papa_v[t] = sum_P bmo^P[p1][a0+a1] bmo^P[p2][a0+a2]   at (p1,a1,p2,a2) = the same four numbers
 *               read in papa's index order                                             (Eq. 21)
 * i.e. sample t = (p1, p2, a1, a2) addresses ppaa[p1][p2][a1][a2] and papa[p1][a1][p2][a2].
 * The packed triangle is read in place (no unpack), e1 and e2 ascending, then P ascending.
 * OpenMP splits the aux slices; the per-slice terms are summed afterwards in ascending P.
 * Pinned against dfjk_oracle_ao2mo at small sizes (tests/test_ao2mo_oracle_pins.py).
 */
static double packed_at(const double* BpP, int e1, int e2) {
  return e1 >= e2 ? BpP[(size_t)e1 * (e1 + 1) / 2 + e2] : BpP[(size_t)e2 * (e2 + 1) / 2 + e1];
}

static double bmo_at(int nao, int nmo, const double* M, const double* BpP, int p, int q) {
  double s = 0.0;
  for (int e1 = 0; e1 < nao; e1++) {
    double y = 0.0;
    for (int e2 = 0; e2 < nao; e2++) y += packed_at(BpP, e1, e2) * M[(size_t)e2 * nmo + q];
    s += M[(size_t)e1 * nmo + p] * y;
  }
  return s;
}

int dfjk_oracle_ao2mo_sample(int naux, int nao, int nmo, int a0, int nact, const double* M, const double* Bp,
                             int nsample, const int* sp1, const int* sp2, const int* sa1, const int* sa2,
                             double* ppaa_v, double* papa_v) {
  if (naux < 0 || nao < 1 || nmo < 1 || nact < 1 || a0 < 0 || a0 + nact > nmo || nsample < 0 || !M || !Bp)
    return DFJK_ORACLE_ERR_ARG;
  for (int t = 0; t < nsample; t++)
    if (sp1[t] < 0 || sp1[t] >= nmo || sp2[t] < 0 || sp2[t] >= nmo || sa1[t] < 0 || sa1[t] >= nact ||
        sa2[t] < 0 || sa2[t] >= nact)
      return DFJK_ORACLE_ERR_ARG;
  const size_t npair = (size_t)nao * (nao + 1) / 2;
  const size_t nterm = (size_t)(nsample > 0 ? nsample : 1) * (size_t)(naux > 0 ? naux : 1);
  double* t20 = (double*)malloc(nterm * sizeof(double));
  double* t21 = (double*)malloc(nterm * sizeof(double));
  if (!t20 || !t21) {
    free(t20); free(t21);
    return DFJK_ORACLE_ERR_ALLOC;
  }
#pragma omp parallel for schedule(dynamic)
  for (int P = 0; P < naux; P++) {
    const double* BpP = Bp + (size_t)P * npair;
    for (int t = 0; t < nsample; t++) {
      const int p1 = sp1[t], p2 = sp2[t], a1 = a0 + sa1[t], a2 = a0 + sa2[t];
      if (ppaa_v) t20[(size_t)t * naux + P] = bmo_at(nao, nmo, M, BpP, p1, p2) * bmo_at(nao, nmo, M, BpP, a1, a2);
      if (papa_v) t21[(size_t)t * naux + P] = bmo_at(nao, nmo, M, BpP, p1, a1) * bmo_at(nao, nmo, M, BpP, p2, a2);
    }
  }
  for (int t = 0; t < nsample; t++) {
    double s20 = 0.0, s21 = 0.0;
    for (int P = 0; P < naux; P++) {
      if (ppaa_v) s20 += t20[(size_t)t * naux + P];
      if (papa_v) s21 += t21[(size_t)t * naux + P];
    }
    if (ppaa_v) ppaa_v[t] = s20;
    if (papa_v) papa_v[t] = s21;
  }
  free(t20); free(t21);
  return DFJK_ORACLE_OK;
}
