/* colour.c — TEST INFRASTRUCTURE (see oracle.h).  SURVEY.md §8(c) C4 "Colour matrix":
 *   CF_{s s'} = sum_{a_1..a_n, i, j} [ (T^{a_s1} ... T^{a_sn})_{ij} ]^* (T^{a_s'1} ... T^{a_s'n})_{ij}
 * built numerically from the 8 Gell-Mann matrices.  Permutations in lexicographic order.
 * brute: loop over every pair (s,s') and every adjoint tuple (the definition, n <= 4).
 * streamed: for each adjoint tuple build all n! products once and add the Gram contribution
 * (same sum, other loop order).  Pins: tests/test_oracle_colour.py (N C_F^n diagonal, integer
 * tables of SURVEY C8, symmetry, rank, brute == streamed).
 */
#include "oracle_internal.h"

static int next_perm(int* a, int n) {
  int i = n - 2; while (i >= 0 && a[i] > a[i + 1]) --i;
  if (i < 0) return 0;
  int j = n - 1; while (a[j] < a[i]) --j;
  int t = a[i]; a[i] = a[j]; a[j] = t;
  for (int l = i + 1, r = n - 1; l < r; ++l, --r) { t = a[l]; a[l] = a[r]; a[r] = t; }
  return 1;
}
int oracle_all_perms(int n, int perms[][5]) {       /* lexicographic; returns n! */
  int a[5]; for (int i = 0; i < n; ++i) a[i] = i;
  int k = 0;
  do { for (int i = 0; i < n; ++i) perms[k][i] = a[i]; ++k; } while (next_perm(a, n));
  return k;
}
static void string_product(cplx T[8][3][3], const int* adj, const int* perm, int n, cplx out[3][3]) {
  cplx acc[3][3] = {{1,0,0},{0,1,0},{0,0,1}};
  for (int k = 0; k < n; ++k) {
    cplx (*t)[3] = T[adj[perm[k]]];
    cplx nxt[3][3];
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
      cplx s = 0; for (int l = 0; l < 3; ++l) s += acc[i][l] * t[l][j]; nxt[i][j] = s;
    }
    memcpy(acc, nxt, sizeof(acc));
  }
  memcpy(out, acc, sizeof(acc));
}

int oracle_colour_matrix(int n, double* CF, int brute) {
  if (n < 1 || n > 5) return -1;
  static int perms[120][5];
  int np = oracle_all_perms(n, perms);
  cplx T[8][3][3]; oracle_gellmann_T(T);
  int64_t ntuple = 1; for (int i = 0; i < n; ++i) ntuple *= 8;
  for (int i = 0; i < np * np; ++i) CF[i] = 0;
  if (brute) {
    for (int s = 0; s < np; ++s) for (int sp = 0; sp < np; ++sp) {
      cplx tot = 0;
      for (int64_t t = 0; t < ntuple; ++t) {
        int adj[5]; int64_t r = t; for (int i = 0; i < n; ++i) { adj[i] = (int)(r % 8); r /= 8; }
        cplx A[3][3], B[3][3];
        string_product(T, adj, perms[s], n, A);
        string_product(T, adj, perms[sp], n, B);
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) tot += conj(A[i][j]) * B[i][j];
      }
      CF[s * np + sp] = (double)R_CREAL(tot);
    }
    return 0;
  }
  real* acc = (real*)calloc((size_t)np * np, sizeof(real));
  #pragma omp parallel
  {
    real* loc = (real*)calloc((size_t)np * np, sizeof(real));
    cplx (*prod)[3][3] = malloc(sizeof(cplx) * 9 * np);
    #pragma omp for schedule(static)
    for (int64_t t = 0; t < ntuple; ++t) {
      int adj[5]; int64_t r = t; for (int i = 0; i < n; ++i) { adj[i] = (int)(r % 8); r /= 8; }
      for (int s = 0; s < np; ++s) string_product(T, adj, perms[s], n, prod[s]);
      for (int s = 0; s < np; ++s) for (int sp = 0; sp < np; ++sp) {
        cplx tot = 0;
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) tot += conj(prod[s][i][j]) * prod[sp][i][j];
        loc[s * np + sp] += R_CREAL(tot);
      }
    }
    #pragma omp critical
    for (int i = 0; i < np * np; ++i) acc[i] += loc[i];
    free(loc); free(prod);
  }
  for (int i = 0; i < np * np; ++i) CF[i] = (double)acc[i];
  free(acc);
  return 0;
}
