/* me_eemumu.c — TEST INFRASTRUCTURE (see oracle.h).  SURVEY.md §8(c) C3: e+(p1) e-(p2) -> mu+(p3)
 * mu-(p4), photon + Z s-channel, explicit Feynman rules, written out term by term
 * (process named at PAPER.md:45 and PAPER.md:139).  Pin: closed form of SURVEY C8
 * (tests/test_oracle_me.py), incl. the printed value 6.167834679019e-3 at cos(theta)=0.5.
 */
#include "oracle_internal.h"

double oracle_me_eemumu(const double* p, const oracle_params_t* par, double* hel_out) {
  real P[4][4];
  for (int i = 0; i < 4; ++i) for (int m = 0; m < 4; ++m) P[i][m] = p[4 * i + m];
  real e = R_SQRT(4 * R_PI / (real)par->alpha_ew_inv);
  real sw2 = par->sw2, sw = R_SQRT(sw2), cw = R_SQRT(1 - sw2);
  real gz = e / (2 * sw * cw);
  real gV = -(real)0.5 + 2 * sw2, gA = -(real)0.5;
  real gL = -gz * (gV + gA), gR = -gz * (gV - gA);
  real mz = par->mz, gamz = par->gamma_z;
  real s = 0;
  { real q[4]; for (int m = 0; m < 4; ++m) q[m] = P[0][m] + P[1][m];
    s = q[0]*q[0] - q[1]*q[1] - q[2]*q[2] - q[3]*q[3]; }
  cplx prop_a = -I / s;
  cplx prop_z = -I / (s - mz * mz + I * mz * gamz);
  /* chiral projectors in this representation: P_L = upper two components, P_R = lower two */
  mat4c chir; memset(&chir, 0, sizeof(chir));
  chir.m[0][0] = gL; chir.m[1][1] = gL; chir.m[2][2] = gR; chir.m[3][3] = gR;
  real total = 0;
  for (int h = 0; h < 16; ++h) {
    int l1 = (h & 8) ? 1 : -1, l2 = (h & 4) ? 1 : -1, l3 = (h & 2) ? 1 : -1, l4 = (h & 1) ? 1 : -1;
    vec4c v1 = oracle_v(P[0], 0, l1), vbar1 = oracle_bar(&v1);    /* incoming antifermion: vbar */
    vec4c u2 = oracle_u(P[1], 0, l2);                              /* incoming fermion: u       */
    vec4c v3 = oracle_v(P[2], 0, l3);                              /* outgoing antifermion: v   */
    vec4c u4 = oracle_u(P[3], 0, l4), ubar4 = oracle_bar(&u4);     /* outgoing fermion: ubar    */
    cplx M = 0;
    for (int mu = 0; mu < 4; ++mu) {
      mat4c g; oracle_gamma_mat(mu, &g);
      /* gamma_mu (lower index) = metric * gamma^mu ; sum_mu g^{mu mu} X^mu Y^mu */
      vec4c t;
      /* photon: (ie)^2 (vbar1 gamma^mu u2)(ubar4 gamma^mu v3) g_{mu mu} (-i/s) */
      t = mat_times_col(&g, &u2); cplx a_e = row_times_col(&vbar1, &t);
      t = mat_times_col(&g, &v3); cplx a_m = row_times_col(&ubar4, &t);
      M += oracle_metric[mu] * (I * e) * (I * e) * a_e * a_m * prop_a;
      /* Z: (i)^2 (vbar1 gamma^mu (gL PL + gR PR) u2)(ubar4 gamma^mu (gL PL + gR PR) v3) (-i)/(s-MZ^2+i MZ GZ) */
      vec4c cu2 = mat_times_col(&chir, &u2), cv3 = mat_times_col(&chir, &v3);
      t = mat_times_col(&g, &cu2); cplx z_e = row_times_col(&vbar1, &t);
      t = mat_times_col(&g, &cv3); cplx z_m = row_times_col(&ubar4, &t);
      M += oracle_metric[mu] * (I) * (I) * z_e * z_m * prop_z;
    }
    real m2 = R_CREAL(M) * R_CREAL(M) + R_CIMAG(M) * R_CIMAG(M);
    if (hel_out) hel_out[h] = (double)(m2 / 4);
    total += m2;
  }
  return (double)(total / 4);
}
