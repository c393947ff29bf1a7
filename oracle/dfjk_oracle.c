/*
 * dfjk_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the density-fitted Coulomb/exchange (JK) build of
 * arxiv 2505.03755 (Eq. 12-17), written from the definitions so a reader can
 * check it against the paper by eye.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path (paper_2505_03755_b200/csrc), and neither side
 * includes the other.
 *
 * Conventions (rows R1-R13):
 *   - Bp is the packed Cholesky tensor b^P_{mu nu} "stored in triangular form of size
 *     Naux*Nao(Nao+1)/2": aux index P slowest, then the row-major lower triangle
 *     idx(mu,nu) = mu(mu+1)/2 + nu for mu >= nu.  b^P is symmetric in (mu,nu) (Eq. 12, real AOs).
 *   - C_s is nao x nocc_s row-major, occ_s has nocc_s entries; D_s = C_s diag(occ_s) C_s^T.
 *     The sets are concatenated:  C = [C_0 | C_1 | ...] block after block, occ likewise.
 *   - J and K are nset x nao x nao row-major, full squares; raw J[D_s], K[D_s] with no 1/2 and no
 *     subtraction (Eq. 13 is left to the caller).
 *
 * No symmetry shortcut, no packed-weight trick, no sqrt(occ) folding, no blocking over P, no
 * tiling: every sum runs over the full index range in ascending order.  OpenMP splits OUTPUT
 * rows only, so every output element is summed in the same order whatever the thread count.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force 4-index contraction (Eq. 12 + the
 * index pattern of Eq. 5), closed forms (B=I, rank-one, diagonal, C=I),
 * invariants (symmetry, linearity, Tr(DJ) = sum rho^2, Tr(DK) = sum_P ||C'^T B_P C'||_F^2,
 * C-form == D-form), an independent numpy.einsum evaluation, and SURVEY.md 8(c)'s recorded
 * values for the tiny config.  No function here is "parity unpinned".
 */
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define DFJK_ORACLE_OK 0
#define DFJK_ORACLE_ERR_ARG 1
#define DFJK_ORACLE_ERR_ALLOC 2

int dfjk_oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* Step 1 ("unpacked to the square-matrix form"): one aux slice of the packed
 * tensor -> full symmetric nao x nao matrix Bsq[mu][nu] = Bsq[nu][mu] = Bp_P[mu(mu+1)/2+nu]. */
void dfjk_oracle_unpack_slice(int nao, const double* BpP, double* Bsq) {
  for (int mu = 0; mu < nao; mu++)
    for (int nu = 0; nu <= mu; nu++) {
      double v = BpP[(size_t)mu * (mu + 1) / 2 + nu];
      Bsq[(size_t)mu * nao + nu] = v;
      Bsq[(size_t)nu * nao + mu] = v;
    }
}

/* Step 2: D[mu][nu] = sum_i occ_i C[mu][i] C[nu][i]   (density of one set; the "density matrix"
 * input of the JK call). */
void dfjk_oracle_density(int nao, int nocc, const double* C, const double* occ, double* D) {
#pragma omp parallel for schedule(static)
  for (int mu = 0; mu < nao; mu++)
    for (int nu = 0; nu < nao; nu++) {
      double s = 0.0;
      for (int i = 0; i < nocc; i++) s += occ[i] * C[(size_t)mu * nocc + i] * C[(size_t)nu * nocc + i];
      D[(size_t)mu * nao + nu] = s;
    }
}

/*
 * The JK call ("the input is a density matrix and the ... Cholesky vectors and the
 * output is J and K"), C-form of K:
 *   rho[s][P]   = sum_{mu,nu} Bsq_P[mu][nu] D_s[mu][nu]                      (Eq. 14)
 *   J_s[mu][nu] = sum_P rho[s][P] Bsq_P[mu][nu]                              (Eq. 15)
 *   X[mu][i]    = sum_lam Bsq_P[mu][lam] C_s[lam][i]          (Eq. 16 with gamma = C occ C^T; the
 *                                                              half-transform of Eq. 18)
 *   K_s[mu][nu] = sum_P sum_i occ_i X[mu][i] X[nu][i]                        (Eq. 17)
 * P ascending everywhere.  J, K may be NULL (skipped); rho_out (nset x naux) may be NULL.
 */
int dfjk_oracle_get_jk(int naux, int nao, int nset, const int* nocc, const double* C,
                       const double* occ, const double* Bp, double* J, double* K, double* rho_out) {
  if (naux < 0 || nao <= 0 || nset <= 0 || !nocc || !Bp) return DFJK_ORACLE_ERR_ARG;
  const size_t n2 = (size_t)nao * nao, npair = (size_t)nao * (nao + 1) / 2;
  int nocc_max = 0;
  size_t ctot = 0;
  for (int s = 0; s < nset; s++) {
    if (nocc[s] < 0) return DFJK_ORACLE_ERR_ARG;
    if (nocc[s] > nocc_max) nocc_max = nocc[s];
    ctot += (size_t)nocc[s];
  }
  if (ctot > 0 && (!C || !occ)) return DFJK_ORACLE_ERR_ARG;
  double* Bsq = (double*)malloc(n2 * sizeof(double));
  double* D = (double*)malloc(n2 * (size_t)nset * sizeof(double));
  double* X = (double*)malloc((size_t)nao * (size_t)(nocc_max > 0 ? nocc_max : 1) * sizeof(double));
  double* rowsum = (double*)malloc((size_t)nao * sizeof(double));
  if (!Bsq || !D || !X || !rowsum) { free(Bsq); free(D); free(X); free(rowsum); return DFJK_ORACLE_ERR_ALLOC; }

  /* densities of every set */
  {
    size_t coff = 0, ooff = 0;
    for (int s = 0; s < nset; s++) {
      dfjk_oracle_density(nao, nocc[s], C + coff, occ + ooff, D + n2 * s);
      coff += (size_t)nao * nocc[s];
      ooff += (size_t)nocc[s];
    }
  }
  if (J) memset(J, 0, n2 * (size_t)nset * sizeof(double));
  if (K) memset(K, 0, n2 * (size_t)nset * sizeof(double));

  for (int P = 0; P < naux; P++) {
    dfjk_oracle_unpack_slice(nao, Bp + (size_t)P * npair, Bsq);
    size_t coff = 0, ooff = 0;
    for (int s = 0; s < nset; s++) {
      const double* Cs = C + coff;
      const double* os = occ + ooff;
      const double* Ds = D + n2 * s;
      const int no = nocc[s];
      if (J || rho_out) {
        /* Eq. 14 over the full square: row sums (rows split over threads), then rows ascending */
#pragma omp parallel for schedule(static)
        for (int mu = 0; mu < nao; mu++) {
          double r = 0.0;
          for (int nu = 0; nu < nao; nu++) r += Bsq[(size_t)mu * nao + nu] * Ds[(size_t)mu * nao + nu];
          rowsum[mu] = r;
        }
        double rho = 0.0;
        for (int mu = 0; mu < nao; mu++) rho += rowsum[mu];
        if (rho_out) rho_out[(size_t)s * naux + P] = rho;
        if (J) {
          /* Eq. 15 */
          double* Js = J + n2 * s;
#pragma omp parallel for schedule(static)
          for (int mu = 0; mu < nao; mu++)
            for (int nu = 0; nu < nao; nu++) Js[(size_t)mu * nao + nu] += rho * Bsq[(size_t)mu * nao + nu];
        }
      }
      if (K && no > 0) {
        double* Ks = K + n2 * s;
        /* half-transform X = Bsq_P C_s */
#pragma omp parallel for schedule(static)
        for (int mu = 0; mu < nao; mu++) {
          double* x = X + (size_t)mu * no;
          for (int i = 0; i < no; i++) x[i] = 0.0;
          for (int lam = 0; lam < nao; lam++) {
            const double b = Bsq[(size_t)mu * nao + lam];
            const double* c = Cs + (size_t)lam * no;
            for (int i = 0; i < no; i++) x[i] += b * c[i];
          }
        }
        /* K += X occ X^T, every (mu,nu) of the full square */
#pragma omp parallel for schedule(static)
        for (int mu = 0; mu < nao; mu++) {
          const double* xm = X + (size_t)mu * no;
          for (int nu = 0; nu < nao; nu++) {
            const double* xn = X + (size_t)nu * no;
            double t = 0.0;
#pragma omp simd reduction(+ : t)
            for (int i = 0; i < no; i++) t += os[i] * xm[i] * xn[i];
            Ks[(size_t)mu * nao + nu] += t;
          }
        }
      }
      coff += (size_t)nao * no;
      ooff += (size_t)no;
    }
  }
  free(Bsq); free(D); free(X); free(rowsum);
  return DFJK_ORACLE_OK;
}

/*
 * D-form of K, literally Eq. 16 then Eq. 17 with the nao x nao density:
 *   V[mu][sig]  = sum_lam Bsq_P[mu][lam] D[lam][sig]
 *   K[mu][nu]  += sum_sig V[mu][sig] Bsq_P[nu][sig]
 * One set, density given (any symmetric or non-symmetric D).  O(naux nao^3): tiny/small only.
 */
int dfjk_oracle_get_k_dform(int naux, int nao, const double* D, const double* Bp, double* K) {
  if (naux < 0 || nao <= 0 || !D || !Bp || !K) return DFJK_ORACLE_ERR_ARG;
  const size_t n2 = (size_t)nao * nao, npair = (size_t)nao * (nao + 1) / 2;
  double* Bsq = (double*)malloc(n2 * sizeof(double));
  double* V = (double*)malloc(n2 * sizeof(double));
  if (!Bsq || !V) { free(Bsq); free(V); return DFJK_ORACLE_ERR_ALLOC; }
  memset(K, 0, n2 * sizeof(double));
  for (int P = 0; P < naux; P++) {
    dfjk_oracle_unpack_slice(nao, Bp + (size_t)P * npair, Bsq);
#pragma omp parallel for schedule(static)
    for (int mu = 0; mu < nao; mu++) {
      double* v = V + (size_t)mu * nao;
      for (int sig = 0; sig < nao; sig++) v[sig] = 0.0;
      for (int lam = 0; lam < nao; lam++) {
        const double b = Bsq[(size_t)mu * nao + lam];
        for (int sig = 0; sig < nao; sig++) v[sig] += b * D[(size_t)lam * nao + sig];
      }
    }
#pragma omp parallel for schedule(static)
    for (int mu = 0; mu < nao; mu++)
      for (int nu = 0; nu < nao; nu++) {
        double t = 0.0;
        for (int sig = 0; sig < nao; sig++) t += V[(size_t)mu * nao + sig] * Bsq[(size_t)nu * nao + sig];
        K[(size_t)mu * nao + nu] += t;
      }
  }
  free(Bsq); free(V);
  return DFJK_ORACLE_OK;
}

/*
 * Brute force through the 4-index integrals (tiny shapes only, O(naux nao^4) work, nao^4 memory):
 *   G[m1][m2][m3][m4] = g^{m1 m3}_{m2 m4} = sum_P b^P_{m1 m2} b^P_{m3 m4}          (Eq. 12)
 *   J[m1][m2] = sum_{m3,m4} g^{m1 m3}_{m2 m4} D[m3][m4]      (first term of Eq. 5)
 *   K[m1][m2] = sum_{m3,m4} g^{m1 m3}_{m4 m2} D[m3][m4]      (second term of Eq. 5)
 * One set, density given.
 */
int dfjk_oracle_bruteforce(int naux, int nao, const double* D, const double* Bp, double* J, double* K) {
  if (naux < 0 || nao <= 0 || nao > 24 || !D || !Bp || !J || !K) return DFJK_ORACLE_ERR_ARG;
  const size_t n = (size_t)nao, n2 = n * n, npair = n * (n + 1) / 2;
  double* Bsq = (double*)malloc(n2 * (size_t)(naux > 0 ? naux : 1) * sizeof(double));
  double* G = (double*)malloc(n2 * n2 * sizeof(double));
  if (!Bsq || !G) { free(Bsq); free(G); return DFJK_ORACLE_ERR_ALLOC; }
  for (int P = 0; P < naux; P++) dfjk_oracle_unpack_slice(nao, Bp + (size_t)P * npair, Bsq + n2 * P);
  for (size_t m1 = 0; m1 < n; m1++)
    for (size_t m2 = 0; m2 < n; m2++)
      for (size_t m3 = 0; m3 < n; m3++)
        for (size_t m4 = 0; m4 < n; m4++) {
          double g = 0.0;
          for (int P = 0; P < naux; P++) g += Bsq[n2 * P + m1 * n + m2] * Bsq[n2 * P + m3 * n + m4];
          G[((m1 * n + m2) * n + m3) * n + m4] = g;
        }
  for (size_t m1 = 0; m1 < n; m1++)
    for (size_t m2 = 0; m2 < n; m2++) {
      double j = 0.0, k = 0.0;
      for (size_t m3 = 0; m3 < n; m3++)
        for (size_t m4 = 0; m4 < n; m4++) {
          j += G[((m1 * n + m2) * n + m3) * n + m4] * D[m3 * n + m4];
          k += G[((m1 * n + m4) * n + m3) * n + m2] * D[m3 * n + m4];
        }
      J[m1 * n + m2] = j;
      K[m1 * n + m2] = k;
    }
  free(Bsq); free(G);
  return DFJK_ORACLE_OK;
}

/* element (mu,nu) of the unpacked slice, read in place from the packed row */
static double slice_at(const double* BpP, int mu, int nu) {
  return mu >= nu ? BpP[(size_t)mu * (mu + 1) / 2 + nu] : BpP[(size_t)nu * (nu + 1) / 2 + mu];
}

/*
 * Single output elements, one by one from the definitions (for parity at sizes where the full
 * oracle takes minutes).  For sample t = (set[t], mu[t], nu[t]):
 *   Jv[t] = sum_P rho[s][P] Bsq_P[mu][nu],  rho[s][P] = sum over the full square (Eq. 14-15)
 *   Kv[t] = sum_P sum_i occ_i x_mu[i] x_nu[i],  x_m[i] = sum_lam Bsq_P[m][lam] C_s[lam][i] (Eq. 16-17)
 * Threads split P; the per-P terms are stored and added in ascending P afterwards.
 * Jv or Kv may be NULL.
 */
int dfjk_oracle_sample(int naux, int nao, int nset, const int* nocc, const double* C, const double* occ,
                       const double* Bp, int nsample, const int* sset, const int* smu, const int* snu,
                       double* Jv, double* Kv) {
  if (naux < 0 || nao <= 0 || nset <= 0 || !nocc || !Bp || nsample < 0) return DFJK_ORACLE_ERR_ARG;
  const size_t n2 = (size_t)nao * nao, npair = (size_t)nao * (nao + 1) / 2;
  size_t* coff = (size_t*)malloc(sizeof(size_t) * (size_t)nset);
  size_t* ooff = (size_t*)malloc(sizeof(size_t) * (size_t)nset);
  int nocc_max = 1;
  {
    size_t c = 0, o = 0;
    for (int s = 0; s < nset; s++) {
      coff[s] = c; ooff[s] = o;
      c += (size_t)nao * nocc[s]; o += (size_t)nocc[s];
      if (nocc[s] > nocc_max) nocc_max = nocc[s];
    }
  }
  for (int t = 0; t < nsample; t++)
    if (sset[t] < 0 || sset[t] >= nset || smu[t] < 0 || smu[t] >= nao || snu[t] < 0 || snu[t] >= nao) {
      free(coff); free(ooff);
      return DFJK_ORACLE_ERR_ARG;
    }
  double* term = (double*)malloc(sizeof(double) * (size_t)(nsample > 0 ? nsample : 1) * (size_t)(naux > 0 ? naux : 1));
  if (Jv) {
    double* D = (double*)malloc(n2 * (size_t)nset * sizeof(double));
    double* rho = (double*)malloc(sizeof(double) * (size_t)nset * (size_t)(naux > 0 ? naux : 1));
    for (int s = 0; s < nset; s++) dfjk_oracle_density(nao, nocc[s], C + coff[s], occ + ooff[s], D + n2 * s);
#pragma omp parallel for schedule(static)
    for (int P = 0; P < naux; P++) {
      const double* BpP = Bp + (size_t)P * npair;
      for (int s = 0; s < nset; s++) {
        double r = 0.0;
        for (int mu = 0; mu < nao; mu++)
          for (int nu = 0; nu < nao; nu++) r += slice_at(BpP, mu, nu) * D[n2 * s + (size_t)mu * nao + nu];
        rho[(size_t)s * naux + P] = r;
      }
    }
    for (int t = 0; t < nsample; t++) {
      double j = 0.0;
      for (int P = 0; P < naux; P++)
        j += rho[(size_t)sset[t] * naux + P] * slice_at(Bp + (size_t)P * npair, smu[t], snu[t]);
      Jv[t] = j;
    }
    free(D); free(rho);
  }
  if (Kv) {
#pragma omp parallel
    {
      double* xm = (double*)malloc(sizeof(double) * (size_t)nocc_max);
      double* xn = (double*)malloc(sizeof(double) * (size_t)nocc_max);
#pragma omp for schedule(static)
      for (int P = 0; P < naux; P++) {
        const double* BpP = Bp + (size_t)P * npair;
        for (int t = 0; t < nsample; t++) {
          const int s = sset[t], no = nocc[s];
          const double* Cs = C + coff[s];
          const double* os = occ + ooff[s];
          for (int i = 0; i < no; i++) { xm[i] = 0.0; xn[i] = 0.0; }
          for (int lam = 0; lam < nao; lam++) {
            const double bm = slice_at(BpP, smu[t], lam), bn = slice_at(BpP, snu[t], lam);
            for (int i = 0; i < no; i++) {
              xm[i] += bm * Cs[(size_t)lam * no + i];
              xn[i] += bn * Cs[(size_t)lam * no + i];
            }
          }
          double k = 0.0;
          for (int i = 0; i < no; i++) k += os[i] * xm[i] * xn[i];
          term[(size_t)t * naux + P] = k;
        }
      }
      free(xm); free(xn);
    }
    for (int t = 0; t < nsample; t++) {
      double k = 0.0;
      for (int P = 0; P < naux; P++) k += term[(size_t)t * naux + P];
      Kv[t] = k;
    }
  }
  free(term); free(coff); free(ooff);
  return DFJK_ORACLE_OK;
}
