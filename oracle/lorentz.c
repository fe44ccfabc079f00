/* lorentz.c — TEST INFRASTRUCTURE (see oracle.h).  Conventions C1 of SURVEY.md §8(c):
 * metric diag(+,-,-,-); chiral gamma matrices; helicity spinors u, v; massless polarisation
 * vectors; Gell-Mann matrices.  Pins (tests/test_oracle_lorentz.py): Clifford algebra,
 * Dirac equation, completeness sums, transversality, normalisation, [T^a,T^b] = i f T, Tr = 1/2.
 */
#include "oracle_internal.h"

const real oracle_metric[4] = {1, -1, -1, -1};

void oracle_gamma_mat(int mu, mat4c* g) {
  /* gamma^0 = [[0,1],[1,0]], gamma^i = [[0,sigma^i],[-sigma^i,0]] in 2x2 blocks */
  memset(g, 0, sizeof(*g));
  cplx sig[2][2];
  real sgn_lower;
  if (mu == 0)      { sig[0][0]=1; sig[0][1]=0;  sig[1][0]=0; sig[1][1]=1;  sgn_lower = 1; }
  else if (mu == 1) { sig[0][0]=0; sig[0][1]=1;  sig[1][0]=1; sig[1][1]=0;  sgn_lower = -1; }
  else if (mu == 2) { sig[0][0]=0; sig[0][1]=-I; sig[1][0]=I; sig[1][1]=0;  sgn_lower = -1; }
  else              { sig[0][0]=1; sig[0][1]=0;  sig[1][0]=0; sig[1][1]=-1; sgn_lower = -1; }
  for (int i = 0; i < 2; ++i) for (int j = 0; j < 2; ++j) {
    g->m[i][2 + j] = sig[i][j];               /* upper-right block */
    g->m[2 + i][j] = sgn_lower * sig[i][j];   /* lower-left block  */
  }
}

mat4c oracle_slash(const vec4c* a) {
  mat4c r; memset(&r, 0, sizeof(r));
  for (int mu = 0; mu < 4; ++mu) {
    mat4c g; oracle_gamma_mat(mu, &g);
    for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j)
      r.m[i][j] += oracle_metric[mu] * a->c[mu] * g.m[i][j];
  }
  return r;
}
mat4c m_add_scaled_identity(mat4c a, cplx s) { for (int i = 0; i < 4; ++i) a.m[i][i] += s; return a; }
vec4c row_times_mat(const vec4c* row, const mat4c* m) {
  vec4c r = v_zero();
  for (int j = 0; j < 4; ++j) for (int i = 0; i < 4; ++i) r.c[j] += row->c[i] * m->m[i][j];
  return r;
}
vec4c mat_times_col(const mat4c* m, const vec4c* col) {
  vec4c r = v_zero();
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) r.c[i] += m->m[i][j] * col->c[j];
  return r;
}
cplx row_times_col(const vec4c* row, const vec4c* col) {
  cplx r = 0; for (int i = 0; i < 4; ++i) r += row->c[i] * col->c[i]; return r;
}
vec4c oracle_conj(const vec4c* a) { vec4c r; for (int i = 0; i < 4; ++i) r.c[i] = conj(a->c[i]); return r; }

/* two-component helicity eigenvector chi_lambda(p) */
static void chi(const real p[4], int lambda, cplx out[2]) {
  real pabs = R_SQRT(p[1]*p[1] + p[2]*p[2] + p[3]*p[3]);
  if (pabs + p[3] <= 0 || (p[1] == 0 && p[2] == 0 && p[3] < 0)) {     /* pz = -|p| */
    if (lambda > 0) { out[0] = 0;  out[1] = 1; }
    else            { out[0] = -1; out[1] = 0; }
    return;
  }
  real norm = R_SQRT(2 * pabs * (pabs + p[3]));
  if (lambda > 0) { out[0] = (pabs + p[3]) / norm;      out[1] = (p[1] + I * p[2]) / norm; }
  else            { out[0] = (-p[1] + I * p[2]) / norm; out[1] = (pabs + p[3]) / norm; }
}
static void omegas(const real p[4], real m, real* wplus, real* wminus) {
  real pabs = R_SQRT(p[1]*p[1] + p[2]*p[2] + p[3]*p[3]);
  if (m == 0) { *wplus = R_SQRT(2 * p[0]); *wminus = 0; }              /* exact massless branch */
  else        { *wplus = R_SQRT(p[0] + pabs); *wminus = R_SQRT(p[0] - pabs); }
}
vec4c oracle_u(const real p[4], real m, int lambda) {
  real wp, wm; omegas(p, m, &wp, &wm);
  cplx x[2]; chi(p, lambda, x);
  real w_minus_lam = (lambda > 0) ? wm : wp;   /* omega_{-lambda} */
  real w_lam       = (lambda > 0) ? wp : wm;   /* omega_{lambda}  */
  vec4c r; r.c[0] = w_minus_lam * x[0]; r.c[1] = w_minus_lam * x[1];
           r.c[2] = w_lam * x[0];       r.c[3] = w_lam * x[1];
  return r;
}
vec4c oracle_v(const real p[4], real m, int lambda) {
  real wp, wm; omegas(p, m, &wp, &wm);
  cplx x[2]; chi(p, -lambda, x);               /* chi_{-lambda} */
  real w_minus_lam = (lambda > 0) ? wm : wp;
  real w_lam       = (lambda > 0) ? wp : wm;
  vec4c r; r.c[0] = -lambda * w_lam * x[0];      r.c[1] = -lambda * w_lam * x[1];
           r.c[2] = lambda * w_minus_lam * x[0]; r.c[3] = lambda * w_minus_lam * x[1];
  return r;
}
vec4c oracle_bar(const vec4c* psi) {           /* psi^dagger gamma^0: swaps upper and lower halves */
  mat4c g0; oracle_gamma_mat(0, &g0);
  vec4c d = oracle_conj(psi);
  return row_times_mat(&d, &g0);
}
vec4c oracle_eps(const real k[4], int lambda) {
  real kabs = R_SQRT(k[1]*k[1] + k[2]*k[2] + k[3]*k[3]);
  real kt = R_SQRT(k[1]*k[1] + k[2]*k[2]);
  real e1[4], e2[4];
  if (kt == 0) {
    e1[0]=0; e1[1]=1; e1[2]=0; e1[3]=0;
    e2[0]=0; e2[1]=0; e2[2]=(k[3] >= 0 ? 1 : -1); e2[3]=0;
  } else {
    e1[0]=0; e1[1]=k[1]*k[3]/(kabs*kt); e1[2]=k[2]*k[3]/(kabs*kt); e1[3]=-kt/kabs;
    e2[0]=0; e2[1]=-k[2]/kt;            e2[2]=k[1]/kt;             e2[3]=0;
  }
  vec4c r; real rs2 = R_SQRT((real)2);
  for (int i = 0; i < 4; ++i) r.c[i] = (-lambda * e1[i] - I * e2[i]) / rs2;
  return r;
}
vec4c oracle_V3(const vec4c* p1, const vec4c* e1, const vec4c* p2, const vec4c* e2, const vec4c* p3) {
  vec4c p12 = v_sub(*p1, *p2), p23 = v_sub(*p2, *p3), p31 = v_sub(*p3, *p1);
  cplx e1e2 = mdot_cc(e1, e2), a = mdot_cc(&p23, e1), b = mdot_cc(&p31, e2);
  vec4c r;
  for (int i = 0; i < 4; ++i) r.c[i] = e1e2 * p12.c[i] + e2->c[i] * a + e1->c[i] * b;
  return r;
}

void oracle_gellmann_T(cplx T[8][3][3]) {
  memset(T, 0, sizeof(cplx) * 72);
  real h = (real)0.5, s3 = R_SQRT((real)3);
  T[0][0][1] = h;      T[0][1][0] = h;                    /* lambda1 */
  T[1][0][1] = -I * h; T[1][1][0] = I * h;                /* lambda2 */
  T[2][0][0] = h;      T[2][1][1] = -h;                   /* lambda3 */
  T[3][0][2] = h;      T[3][2][0] = h;                    /* lambda4 */
  T[4][0][2] = -I * h; T[4][2][0] = I * h;                /* lambda5 */
  T[5][1][2] = h;      T[5][2][1] = h;                    /* lambda6 */
  T[6][1][2] = -I * h; T[6][2][1] = I * h;                /* lambda7 */
  T[7][0][0] = h / s3; T[7][1][1] = h / s3; T[7][2][2] = -2 * h / s3;   /* lambda8 */
}

/* ---- exported views for the pins ---- */
static void pack(const vec4c* a, double out[8]) {
  for (int i = 0; i < 4; ++i) { out[2*i] = (double)R_CREAL(a->c[i]); out[2*i+1] = (double)R_CIMAG(a->c[i]); }
}
static void toreal(const double p[4], real q[4]) { for (int i = 0; i < 4; ++i) q[i] = p[i]; }
void oracle_spinor_u(const double p[4], double m, int lambda, double out[8]) { real q[4]; toreal(p,q); vec4c r = oracle_u(q, m, lambda); pack(&r, out); }
void oracle_spinor_v(const double p[4], double m, int lambda, double out[8]) { real q[4]; toreal(p,q); vec4c r = oracle_v(q, m, lambda); pack(&r, out); }
void oracle_polvec(const double k[4], int lambda, double out[8]) { real q[4]; toreal(k,q); vec4c r = oracle_eps(q, lambda); pack(&r, out); }
void oracle_gamma(int mu, double out[32]) {
  mat4c g; oracle_gamma_mat(mu, &g);
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) {
    out[2*(4*i+j)] = (double)R_CREAL(g.m[i][j]); out[2*(4*i+j)+1] = (double)R_CIMAG(g.m[i][j]);
  }
}
