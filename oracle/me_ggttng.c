/* me_ggttng.c — TEST INFRASTRUCTURE (see oracle.h).  g g -> t t~ + (n-2) g, n = 2..5 gluons
 * (processes named at PAPER.md:139; leading order, fixed couplings PAPER.md:141).
 *   C4  colour-ordered Berends-Giele recursion + colour matrix  -> oracle_me_ggttng (the oracle)
 *   C5  colour-dressed recursion with explicit f^{abc}, T^a and brute-force colour sums
 *       -> oracle_me_ggttng_dressed (independent second route, pins every sign of C4)
 *   C5  gg -> tt~ written out by hand (3 diagrams, 2 flows) -> oracle_me_ggtt_explicit
 * Formulas are those of SURVEY.md §8(c) C4/C5, in that notation: gluon momenta P_i incoming,
 * j(s) ordered gluon current, Psibar(s) ordered quark-line current, A_sigma partial amplitude.
 * Pins: tests/test_oracle_me.py — Combridge closed form, C4 == C5, Ward identity, Bose symmetry,
 * Lorentz invariance, SURVEY Appendix A worked values (cross-check).
 */
#include "oracle_internal.h"
#include <stdio.h>

int oracle_all_perms(int n, int perms[][5]);

#define MAXG 5
#define NKEY 32768            /* ordered tuples of <= 5 gluons, digits 1..5 base 8 */

typedef struct {
  int n;                      /* gluons in total */
  real gs, mt;
  vec4c P[MAXG];              /* incoming gluon momenta */
  vec4c e[MAXG];              /* polarisations (eps incoming, eps* outgoing) */
  vec4c pt;                   /* top momentum (outgoing) */
  vec4c ubar, v;              /* ubar(p_t), v(p_tbar) */
  vec4c jmemo[NKEY];  unsigned char jdone[NKEY];
  vec4c qmemo[NKEY];  unsigned char qdone[NKEY];
} bg_t;

static int key_of(const int* s, int k) { int key = 0, mul = 1; for (int i = 0; i < k; ++i) { key += (s[i] + 1) * mul; mul *= 8; } return key; }
static vec4c Psum(const bg_t* b, const int* s, int k) { vec4c r = v_zero(); for (int i = 0; i < k; ++i) r = v_add(r, b->P[s[i]]); return r; }

/* ordered gluon current j(s), s = (s_1..s_k)  [C4] */
static vec4c jcur(bg_t* b, const int* s, int k) {
  if (k == 1) return b->e[s[0]];
  int key = key_of(s, k);
  if (b->jdone[key]) return b->jmemo[key];
  vec4c Ps = Psum(b, s, k), mPs = v_scale(-1, Ps), r = v_zero();
  for (int a = 1; a <= k - 1; ++a) {                      /* A = s[1..a], B = s[a+1..k] */
    vec4c PA = Psum(b, s, a), PB = Psum(b, s + a, k - a);
    vec4c jA = jcur(b, s, a), jB = jcur(b, s + a, k - a);
    vec4c t = oracle_V3(&PA, &jA, &PB, &jB, &mPs);
    r = v_add(r, v_scale(-b->gs, t));
  }
  for (int a = 1; a < k; ++a) for (int c = a + 1; c < k; ++c) {   /* A=s[1..a], B=s[a+1..c], C=s[c+1..k] */
    vec4c jA = jcur(b, s, a), jB = jcur(b, s + a, c - a), jC = jcur(b, s + c, k - c);
    cplx AB = mdot_cc(&jA, &jB), BC = mdot_cc(&jB, &jC), AC = mdot_cc(&jA, &jC);
    for (int m = 0; m < 4; ++m)
      r.c[m] += -b->gs * b->gs * (AB * jC.c[m] + BC * jA.c[m] - 2 * AC * jB.c[m]);
  }
  cplx P2 = mdot_cc(&Ps, &Ps);
  r = v_scale(1 / P2, r);
  b->jmemo[key] = r; b->jdone[key] = 1;
  return r;
}
/* row spinor  X . (i g_s jslash) */
static vec4c times_vertex(const bg_t* b, const vec4c* row, const vec4c* j) {
  mat4c sl = oracle_slash(j);
  vec4c r = row_times_mat(row, &sl);
  return v_scale(I * b->gs, r);
}
/* ordered quark-line current Psibar(s) for a prefix s of the ordering  [C4] */
static vec4c qcur(bg_t* b, const int* s, int k) {
  if (k == 0) return b->ubar;
  int key = key_of(s, k);
  if (b->qdone[key]) return b->qmemo[key];
  vec4c acc = v_zero();
  for (int a = 0; a <= k - 1; ++a) {
    vec4c prev = qcur(b, s, a), j = jcur(b, s + a, k - a);
    acc = v_add(acc, times_vertex(b, &prev, &j));
  }
  vec4c q = v_sub(b->pt, Psum(b, s, k));
  mat4c num = m_add_scaled_identity(oracle_slash(&q), b->mt);
  cplx den = mdot_cc(&q, &q) - b->mt * b->mt;
  vec4c r = row_times_mat(&acc, &num);
  r = v_scale(I / den, r);
  b->qmemo[key] = r; b->qdone[key] = 1;
  return r;
}
static cplx partial_amp(bg_t* b, const int* sigma) {
  cplx A = 0; int n = b->n;
  for (int a = 0; a <= n - 1; ++a) {
    vec4c prev = qcur(b, sigma, a), j = jcur(b, sigma + a, n - a);
    vec4c t = times_vertex(b, &prev, &j);
    A += row_times_col(&t, &b->v);
  }
  return A;
}

/* colour matrices, built once per n (not thread-safe on first call: drivers call it serially) */
static double* g_CF[6] = {0,0,0,0,0,0};
static const double* colour_matrix_cached(int n) {
  if (!g_CF[n]) {
    int np = 1; for (int i = 2; i <= n; ++i) np *= i;
    double* cf = (double*)malloc(sizeof(double) * np * np);
    oracle_colour_matrix(n, cf, 0);
    g_CF[n] = cf;
  }
  return g_CF[n];
}

static void setup_externals(bg_t* b, int nfinal, const double* p, const oracle_params_t* par,
                            int h, int ward_which) {
  int n = 2 + nfinal, npar = n + 2;
  b->n = n;
  b->gs = R_SQRT(4 * R_PI * (real)par->alpha_s);
  b->mt = par->mt;
  memset(b->jdone, 0, sizeof(b->jdone)); memset(b->qdone, 0, sizeof(b->qdone));
  real q[4];
  for (int g = 0; g < n; ++g) {
    int ipar = (g < 2) ? g : g + 2;
    int lam = ((h >> (npar - 1 - ipar)) & 1) ? 1 : -1;
    for (int m = 0; m < 4; ++m) q[m] = p[4 * ipar + m];
    vec4c eps = oracle_eps(q, lam);
    if (g < 2) { b->P[g] = v_from_real(q); b->e[g] = eps; }
    else       { b->P[g] = v_scale(-1, v_from_real(q)); b->e[g] = oracle_conj(&eps); }
    if (g == ward_which) b->e[g] = b->P[g];
  }
  int lt = ((h >> (npar - 1 - 2)) & 1) ? 1 : -1, ltb = ((h >> (npar - 1 - 3)) & 1) ? 1 : -1;
  for (int m = 0; m < 4; ++m) q[m] = p[8 + m];
  b->pt = v_from_real(q);
  vec4c u = oracle_u(q, b->mt, lt); b->ubar = oracle_bar(&u);
  for (int m = 0; m < 4; ++m) q[m] = p[12 + m];
  b->v = oracle_v(q, b->mt, ltb);
}

static double me_c4(int nfinal, const double* p, const oracle_params_t* par, double* hel_out, int ward_which) {
  int n = 2 + nfinal, npar = n + 2, nhel = 1 << npar;
  if (n < 2 || n > 5) return -1;
  int perms[120][5];               /* per call (threads of oracle_me_batch each fill their own copy) */
  oracle_all_perms(n, perms);
  int np = 1; for (int i = 2; i <= n; ++i) np *= i;
  const double* CF = colour_matrix_cached(n);
  real denom = 256; for (int i = 2; i <= nfinal; ++i) denom *= i;     /* 2*2*8*8*(n-2)!  (A3) */
  bg_t* b = (bg_t*)malloc(sizeof(bg_t));
  cplx A[120];
  real total = 0;
  for (int h = 0; h < nhel; ++h) {
    setup_externals(b, nfinal, p, par, h, ward_which);
    for (int s = 0; s < np; ++s) A[s] = partial_amp(b, perms[s]);
    real mh = 0;
    for (int s = 0; s < np; ++s) for (int sp = 0; sp < np; ++sp)
      mh += R_CREAL(conj(A[s]) * (real)CF[s * np + sp] * A[sp]);
    if (hel_out) hel_out[h] = (double)(mh / denom);
    total += mh;
  }
  free(b);
  return (double)(total / denom);
}
double oracle_me_ggttng(int nfinal, const double* p, const oracle_params_t* par, double* hel_out) {
  return me_c4(nfinal, p, par, hel_out, -1);
}
double oracle_me_ggttng_ward(int nfinal, const double* p, const oracle_params_t* par, int which) {
  return me_c4(nfinal, p, par, NULL, which);
}

/* ---------------- C5: gg -> tt~ by hand ---------------- */
double oracle_me_ggtt_explicit(const double* p, const oracle_params_t* par) {
  real gs = R_SQRT(4 * R_PI * (real)par->alpha_s), m = par->mt;
  real q[4];
  real total = 0;
  for (int h = 0; h < 16; ++h) {
    int l1 = (h & 8) ? 1 : -1, l2 = (h & 4) ? 1 : -1, lt = (h & 2) ? 1 : -1, ltb = (h & 1) ? 1 : -1;
    for (int i = 0; i < 4; ++i) q[i] = p[i];
    vec4c p1 = v_from_real(q), e1 = oracle_eps(q, l1);
    for (int i = 0; i < 4; ++i) q[i] = p[4 + i];
    vec4c p2 = v_from_real(q), e2 = oracle_eps(q, l2);
    for (int i = 0; i < 4; ++i) q[i] = p[8 + i];
    vec4c pt = v_from_real(q), u = oracle_u(q, m, lt), ubar = oracle_bar(&u);
    for (int i = 0; i < 4; ++i) q[i] = p[12 + i];
    vec4c v = oracle_v(q, m, ltb);
    vec4c p12 = v_add(p1, p2), mp12 = v_scale(-1, p12);
    cplx s = mdot_cc(&p12, &p12);
    vec4c J = oracle_V3(&p1, &e1, &p2, &e2, &mp12);
    mat4c e1s = oracle_slash(&e1), e2s = oracle_slash(&e2), Js = oracle_slash(&J);
    vec4c qt = v_sub(pt, p1), qu = v_sub(pt, p2);
    mat4c nt = m_add_scaled_identity(oracle_slash(&qt), m), nu = m_add_scaled_identity(oracle_slash(&qu), m);
    cplx dt = mdot_cc(&qt, &qt) - m * m, du = mdot_cc(&qu, &qu) - m * m;
    vec4c r;
    /* ubar e1slash (qtslash+m) e2slash v */
    r = row_times_mat(&ubar, &e1s); r = row_times_mat(&r, &nt); r = row_times_mat(&r, &e2s);
    cplx tch = row_times_col(&r, &v) / dt;
    r = row_times_mat(&ubar, &e2s); r = row_times_mat(&r, &nu); r = row_times_mat(&r, &e1s);
    cplx uch = row_times_col(&r, &v) / du;
    r = row_times_mat(&ubar, &Js);
    cplx sch = row_times_col(&r, &v) / s;
    cplx jamp1 = -I * gs * gs * tch - I * gs * gs * sch;
    cplx jamp2 = -I * gs * gs * uch + I * gs * gs * sch;
    real a11 = R_CREAL(conj(jamp1) * jamp1), a22 = R_CREAL(conj(jamp2) * jamp2), a12 = R_CREAL(conj(jamp1) * jamp2);
    total += (16 * a11 + 16 * a22 - 2 * 2 * a12) / 3;
  }
  return (double)(total / 256);
}

/* ---------------- C5: colour-dressed recursion, explicit colour indices ---------------- */
typedef struct { cplx c[8][4]; unsigned char nz[8]; } dcur;       /* J^{a,mu}(S) */
typedef struct { cplx c[3][4]; } qrow;                              /* Psibar_{k}(S), fixed top colour i */

double oracle_me_ggttng_dressed(int nfinal, const double* p, const oracle_params_t* par) {
  int n = 2 + nfinal, npar = n + 2, nhel = 1 << npar, nsub = 1 << n, full = nsub - 1;
  if (n < 2 || n > 4) return -1;
  cplx T[8][3][3]; oracle_gellmann_T(T);
  /* f^{abc} = -2i Tr([T^a,T^b] T^c) */
  static real f[8][8][8];
  for (int a = 0; a < 8; ++a) for (int b2 = 0; b2 < 8; ++b2) for (int c = 0; c < 8; ++c) {
    cplx tr = 0;
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k)
      tr += (T[a][i][j] * T[b2][j][k] - T[b2][i][j] * T[a][j][k]) * T[c][k][i];
    f[a][b2][c] = R_CREAL(-2 * I * tr);
  }
  bg_t* b = (bg_t*)malloc(sizeof(bg_t));
  dcur* J = (dcur*)malloc(sizeof(dcur) * nsub);
  qrow (*Q)[3] = malloc(sizeof(qrow) * 3 * nsub);                   /* Q[S][i] */
  real denom = 256; for (int i = 2; i <= nfinal; ++i) denom *= i;
  int64_t ncol = 1; for (int i = 0; i < n; ++i) ncol *= 8;
  real total = 0;
  for (int h = 0; h < nhel; ++h) {
    setup_externals(b, nfinal, p, par, h, -1);
    real gs = b->gs;
    vec4c PS[32];
    for (int S = 1; S < nsub; ++S) { PS[S] = v_zero(); for (int g = 0; g < n; ++g) if (S >> g & 1) PS[S] = v_add(PS[S], b->P[g]); }
    for (int64_t ic = 0; ic < ncol; ++ic) {
      int col[4]; { int64_t r = ic; for (int g = 0; g < n; ++g) { col[g] = (int)(r % 8); r /= 8; } }
      /* gluon currents by subset, in increasing popcount order (numeric order suffices: subsets < S) */
      for (int S = 1; S < nsub; ++S) {
        dcur* out = &J[S]; memset(out, 0, sizeof(*out));
        if ((S & (S - 1)) == 0) {
          int g = 0; while (!((S >> g) & 1)) ++g;
          for (int m = 0; m < 4; ++m) out->c[col[g]][m] = b->e[g].c[m];
          out->nz[col[g]] = 1; continue;
        }
        vec4c mP = v_scale(-1, PS[S]);
        int low = S & -S;
        /* unordered 2-partitions {A,B}: A contains the lowest element */
        for (int A = S; A > 0; A = (A - 1) & S) {
          if (!(A & low) || A == S) continue;
          int B = S ^ A;
          for (int a = 0; a < 8; ++a) if (J[A].nz[a]) for (int bb = 0; bb < 8; ++bb) if (J[B].nz[bb]) {
            vec4c ja, jb; memcpy(ja.c, J[A].c[a], sizeof(ja.c)); memcpy(jb.c, J[B].c[bb], sizeof(jb.c));
            vec4c t = oracle_V3(&PS[A], &ja, &PS[B], &jb, &mP);
            for (int c = 0; c < 8; ++c) if (f[a][bb][c] != 0) {
              for (int m = 0; m < 4; ++m) out->c[c][m] += gs * f[a][bb][c] * t.c[m];   /* vertex g f^{abc} V3 */
              out->nz[c] = 1;
            }
          }
        }
        /* unordered 3-partitions {A,B,C}: A has the lowest element, B the lowest of the rest */
        for (int A = S; A > 0; A = (A - 1) & S) {
          if (!(A & low) || A == S) continue;
          int R = S ^ A; int lowR = R & -R;
          for (int B = R; B > 0; B = (B - 1) & R) {
            if (!(B & lowR) || B == R) continue;
            int C = R ^ B;
            for (int a = 0; a < 8; ++a) if (J[A].nz[a]) for (int bb = 0; bb < 8; ++bb) if (J[B].nz[bb])
            for (int c = 0; c < 8; ++c) if (J[C].nz[c]) {
              vec4c ea, eb, ec; memcpy(ea.c, J[A].c[a], sizeof(ea.c)); memcpy(eb.c, J[B].c[bb], sizeof(eb.c)); memcpy(ec.c, J[C].c[c], sizeof(ec.c));
              cplx ab = mdot_cc(&ea, &eb), ac = mdot_cc(&ea, &ec), bc = mdot_cc(&eb, &ec);
              for (int d = 0; d < 8; ++d) {
                real c1 = 0, c2 = 0, c3 = 0;
                for (int e = 0; e < 8; ++e) {
                  c1 += f[a][bb][e] * f[c][d][e];      /* f^{abe} f^{cde} */
                  c2 += f[a][c][e] * f[bb][d][e];      /* f^{ace} f^{bde} */
                  c3 += f[a][d][e] * f[bb][c][e];      /* f^{ade} f^{bce} */
                }
                if (c1 == 0 && c2 == 0 && c3 == 0) continue;
                for (int m = 0; m < 4; ++m) {
                  cplx t1 = ac * eb.c[m] - bc * ea.c[m];   /* g^{mu rho}g^{nu sigma} - g^{mu sigma}g^{nu rho} */
                  cplx t2 = ab * ec.c[m] - bc * ea.c[m];   /* g^{mu nu}g^{rho sigma} - g^{mu sigma}g^{nu rho} */
                  cplx t3 = ab * ec.c[m] - ac * eb.c[m];   /* g^{mu nu}g^{rho sigma} - g^{mu rho}g^{nu sigma} */
                  out->c[d][m] += (-I * gs * gs) * (c1 * t1 + c2 * t2 + c3 * t3);
                }
                out->nz[d] = 1;
              }
            }
          }
        }
        cplx P2 = mdot_cc(&PS[S], &PS[S]);
        for (int a = 0; a < 8; ++a) for (int m = 0; m < 4; ++m) out->c[a][m] *= (-I / P2);   /* propagator -i g/P^2 */
      }
      /* quark line by subset of absorbed gluons */
      for (int i = 0; i < 3; ++i) { memset(&Q[0][i], 0, sizeof(qrow)); for (int m = 0; m < 4; ++m) Q[0][i].c[i][m] = b->ubar.c[m]; }
      cplx Mij[3][3]; memset(Mij, 0, sizeof(Mij));
      for (int S = 1; S < nsub; ++S) {
        for (int i = 0; i < 3; ++i) {
          qrow acc; memset(&acc, 0, sizeof(acc));
          for (int A = S; A > 0; A = (A - 1) & S) {
            int prev = S ^ A;
            for (int a = 0; a < 8; ++a) if (J[A].nz[a]) {
              vec4c ja; memcpy(ja.c, J[A].c[a], sizeof(ja.c));
              mat4c sl = oracle_slash(&ja);
              for (int k = 0; k < 3; ++k) {
                vec4c row; memcpy(row.c, Q[prev][i].c[k], sizeof(row.c));
                vec4c r = row_times_mat(&row, &sl);
                for (int l = 0; l < 3; ++l) if (T[a][k][l] != 0)
                  for (int m = 0; m < 4; ++m) acc.c[l][m] += I * gs * T[a][k][l] * r.c[m];   /* i g T^a gamma^mu */
              }
            }
          }
          if (S == full) {
            for (int l = 0; l < 3; ++l) { vec4c row; memcpy(row.c, acc.c[l], sizeof(row.c)); Mij[i][l] = row_times_col(&row, &b->v); }
          } else {
            vec4c q = v_sub(b->pt, PS[S]);
            mat4c num = m_add_scaled_identity(oracle_slash(&q), b->mt);
            cplx den = mdot_cc(&q, &q) - b->mt * b->mt;
            for (int l = 0; l < 3; ++l) {
              vec4c row; memcpy(row.c, acc.c[l], sizeof(row.c));
              vec4c r = row_times_mat(&row, &num);
              for (int m = 0; m < 4; ++m) Q[S][i].c[l][m] = (I / den) * r.c[m];
            }
          }
        }
      }
      for (int i = 0; i < 3; ++i) for (int l = 0; l < 3; ++l) total += R_CREAL(conj(Mij[i][l]) * Mij[i][l]);
    }
  }
  free(b); free(J); free(Q);
  return (double)(total / denom);
}

/* ---------------- batch driver ---------------- */
#ifdef _OPENMP
#include <omp.h>
#endif
int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
int oracle_me_batch(int proc, const double* momenta, int64_t nevt, const oracle_params_t* par,
                    double* me_out, int nthreads) {
  if (proc < 0 || proc > 4) return -1;
  int npar = (proc == 0) ? 4 : proc + 3;
  if (proc >= 1) colour_matrix_cached(proc + 1);      /* build serially before the parallel loop */
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
  nthreads = 1;
#endif
  #pragma omp parallel for schedule(dynamic, 4) num_threads(nthreads)
  for (int64_t ie = 0; ie < nevt; ++ie) {
    const double* p = momenta + (size_t)ie * npar * 4;
    me_out[ie] = (proc == 0) ? oracle_me_eemumu(p, par, NULL) : oracle_me_ggttng(proc - 1, p, par, NULL);
  }
  return 0;
}
