/* me_qchannel.c — TEST INFRASTRUCTURE (see oracle.h).
 *
 * Quark channels of p p -> t t~ + jets ("pp -> t t~ 0-2 j"): every tree-level QCD
 * process with the top line, ONE massless quark line of another flavour and ng <= 2 gluons, in any crossing:
 *     q q~ -> t t~ (g (g)),  q g -> t t~ q (g),  g q~ -> t t~ q~ (g),  g g -> t t~ q q~,  ...
 * Method: the Feynman rules written out as an off-shell recursion with EXPLICIT colour indices and explicit factors
 * of i (the colour-dressed route C5 of me_ggttng.c, extended by the second quark line):
 *     quark-gluon vertex  i g T^a_{kl} gamma^mu        quark propagator  i (qslash + m)/(q^2 - m^2)
 *     three-gluon vertex  g f^{abc} V3                 gluon propagator  -i g_{mu nu}/P^2
 *     four-gluon vertex   -i g^2 [f f (g g - g g) + 2 more]
 * Elements of the recursion: the gluons and the light-quark PAIR.  J^{a,mu}(S) is the off-shell gluon current of the
 * element subset S; when S holds the pair, the current has one more source term, Vbar(S1) i g gamma^mu T^a U(S2) summed
 * over the splits S1 + S2 of the gluons of S between the two ends of the light line (U, Vbar: the light line's
 * off-shell spinors with the gluon sets absorbed).  The top line then absorbs gluon currents exactly as in C5.
 * |M|^2 = sum over every external colour and helicity of |M|^2, divided by the initial-state spin and colour
 * multiplicities and by k! for k identical final gluons (A3).
 *
 * Process string `spec`, one character per particle in process order (two incoming first; 't' and 'T' at positions
 * 2 and 3): 'q' light quark, 'Q' light antiquark, 'g' gluon.  Examples: "qQtT", "qQtTg", "qgtTq", "gQtTQ", "qQtTgg".
 * Helicity index as everywhere: bit (npar-1-i) of h set <=> particle i has lambda = +1.
 *
 * Pins (tests/test_oracle_qchannel.py): the textbook closed form of q q~ -> t t~ (absolute normalisation, colour
 * average), the Ward identity on every gluon of every process (relative signs between diagram classes), the
 * initial-state collinear limits q -> q g and g -> q q~ onto the closed form (every 1-jet process) and of
 * q q~ -> t t~ g g onto q q~ -> t t~ g, C- and beam-exchange symmetries.  The other 2-jet crossings (q g -> t t~ q g,
 * g g -> t t~ q q~, ...) run the same code with other external spinors; their own pins are the Ward identities.
 */
#include "oracle_internal.h"

#define MAXEL 4                       /* ng <= 3 gluons + the pair */
typedef struct { cplx c[8][4]; unsigned char nz[8]; } gcur;   /* J^{a,mu}; nz[a] = 0: component a is identically zero */
typedef struct { cplx c[3][4]; } qcur;          /* spinor with a fundamental colour index */

typedef struct {
  int npar, ng, gpart[3];             /* gluon element -> particle index */
  int pin, pout;                      /* particle at the start / end of the light line's fermion flow */
  int in_is_u, out_is_ubar;           /* start: u (incoming q) or v (outgoing Q); end: ubar (outgoing q) or vbar (incoming Q) */
  real denom;
} qspec;

static int parse_spec(const char* spec, qspec* s) {
  int n = (int)strlen(spec);
  if (n < 4 || n > 7 || spec[2] != 't' || spec[3] != 'T') return -1;
  s->npar = n; s->ng = 0; s->pin = s->pout = -1;
  real denom = 1; int nfg = 0;
  for (int i = 0; i < n; ++i) {
    char c = spec[i]; int incoming = i < 2;
    if (i == 2 || i == 3) continue;
    if (c == 'g') { if (s->ng == 3) return -1; s->gpart[s->ng++] = i; if (incoming) denom *= 16; else ++nfg; }
    else if (c == 'q' || c == 'Q') {
      int start = (c == 'q') == incoming;          /* incoming quark or outgoing antiquark start the fermion flow */
      if (start) { if (s->pin >= 0) return -1; s->pin = i; s->in_is_u = incoming; }
      else       { if (s->pout >= 0) return -1; s->pout = i; s->out_is_ubar = !incoming; }
      if (incoming) denom *= 6;
    } else return -1;
  }
  if (s->pin < 0 || s->pout < 0) return -1;
  for (int k = 2; k <= nfg; ++k) denom *= k;
  s->denom = denom;
  return 0;
}

static inline vec4c col_of(const cplx c[4]) { vec4c r; memcpy(r.c, c, sizeof(r.c)); return r; }

double oracle_me_qchannel(const char* spec, const double* p, const oracle_params_t* par, double* hel_out, int ward_which) {
  qspec s;
  if (parse_spec(spec, &s) != 0) return -1;
  const int npar = s.npar, ng = s.ng, nel = ng + 1, PAIR = 1 << ng, nsub = 1 << nel, full = nsub - 1, ngsub = 1 << ng;
  const int nhel = 1 << npar;
  const real gs = R_SQRT(4 * R_PI * (real)par->alpha_s), mt = par->mt;
  cplx T[8][3][3]; oracle_gellmann_T(T);
  real f[8][8][8];                    /* f^{abc} = -2i Tr([T^a,T^b] T^c) */
  for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {
    cplx tr = 0;
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k)
      tr += (T[a][i][j] * T[b][j][k] - T[b][i][j] * T[a][j][k]) * T[c][k][i];
    f[a][b][c] = R_CREAL(-2 * I * tr);
  }
  /* f^{abe} f^{cde}, tabulated once (the three colour structures of the four-gluon vertex are ff[a][b][c][d],
   * ff[a][c][b][d], ff[a][d][b][c]); the four gamma matrices */
  static real ff[8][8][8][8];
  #pragma omp critical(qchannel_ff)
  {
    for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) for (int d = 0; d < 8; ++d) {
      real v = 0; for (int e = 0; e < 8; ++e) v += f[a][b][e] * f[c][d][e];
      ff[a][b][c][d] = v;
    }
  }
  mat4c gmat[4]; for (int mu = 0; mu < 4; ++mu) oracle_gamma_mat(mu, &gmat[mu]);
  real q[4];
  real total = 0;
  int64_t ngcol = 1; for (int g = 0; g < ng; ++g) ngcol *= 8;
  for (int h = 0; h < nhel; ++h) {
    #define LAM(i) (((h >> (npar - 1 - (i))) & 1) ? 1 : -1)
    /* ---- external wavefunctions and incoming momenta of the elements ---- */
    vec4c P[MAXEL], eps[3];
    for (int g = 0; g < ng; ++g) {
      int ip = s.gpart[g];
      for (int m = 0; m < 4; ++m) q[m] = p[4 * ip + m];
      vec4c e = oracle_eps(q, LAM(ip));
      if (ip < 2) { P[g] = v_from_real(q); eps[g] = e; }
      else        { P[g] = v_scale(-1, v_from_real(q)); eps[g] = oracle_conj(&e); }
      if (g == ward_which) eps[g] = P[g];
    }
    for (int m = 0; m < 4; ++m) q[m] = p[4 * s.pin + m];
    vec4c psi_in = s.in_is_u ? oracle_u(q, 0, LAM(s.pin)) : oracle_v(q, 0, LAM(s.pin));
    vec4c f_in = v_scale(s.in_is_u ? 1 : -1, v_from_real(q));          /* momentum carried along the fermion arrow */
    for (int m = 0; m < 4; ++m) q[m] = p[4 * s.pout + m];
    vec4c w = s.out_is_ubar ? oracle_u(q, 0, LAM(s.pout)) : oracle_v(q, 0, LAM(s.pout));
    vec4c psi_out = oracle_bar(&w);
    vec4c f_out = v_scale(s.out_is_ubar ? 1 : -1, v_from_real(q));
    P[ng] = v_sub(f_in, f_out);                                         /* what the pair brings into the rest */
    for (int m = 0; m < 4; ++m) q[m] = p[8 + m];
    vec4c pt = v_from_real(q), ut = oracle_u(q, mt, LAM(2)), ubar = oracle_bar(&ut);
    for (int m = 0; m < 4; ++m) q[m] = p[12 + m];
    vec4c vtb = oracle_v(q, mt, LAM(3));
    vec4c PS[1 << MAXEL];
    for (int S = 0; S < nsub; ++S) { PS[S] = v_zero(); for (int e = 0; e < nel; ++e) if (S >> e & 1) PS[S] = v_add(PS[S], P[e]); }
    real mh = 0;
    for (int64_t ic = 0; ic < ngcol; ++ic) {
      int col[3] = {0, 0, 0}; { int64_t r = ic; for (int g = 0; g < ng; ++g) { col[g] = (int)(r % 8); r /= 8; } }
      for (int cin = 0; cin < 3; ++cin) for (int cout = 0; cout < 3; ++cout) {
        gcur J[1 << MAXEL]; qcur U[8], V[8], Q[1 << MAXEL];
        /* ---- light line: U(G) column at the start, Vbar(G) row at the end, G = set of absorbed gluons.  They need the
         * pure-gluon currents J(G), which are built first (subsets without the pair). ---- */
        for (int pass = 0; pass < 2; ++pass) {
          for (int S = 1; S < nsub; ++S) {
            if (((S & PAIR) != 0) != (pass == 1)) continue;
            gcur* out = &J[S]; memset(out, 0, sizeof(*out));
            if (S < PAIR && (S & (S - 1)) == 0) {                       /* external gluon */
              int g = 0; while (!((S >> g) & 1)) ++g;
              for (int m = 0; m < 4; ++m) out->c[col[g]][m] = eps[g].c[m];
              out->nz[col[g]] = 1;
              continue;
            }
            if (S & PAIR) {                                             /* source: the light line emits the gluon */
              int G = S ^ PAIR;
              for (int G1 = G;; G1 = (G1 - 1) & G) {
                int G2 = G ^ G1;
                for (int mu = 0; mu < 4; ++mu) {
                  const mat4c gm = gmat[mu];
                  for (int a = 0; a < 8; ++a) {
                    cplx acc = 0;
                    for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) if (T[a][k][l] != 0) {
                      vec4c row = col_of(V[G1].c[k]), cl = col_of(U[G2].c[l]);
                      vec4c r = row_times_mat(&row, &gm);
                      acc += T[a][k][l] * row_times_col(&r, &cl);
                    }
                    out->c[a][mu] += I * gs * acc;                      /* i g T^a gamma^mu (upper index mu) */
                    out->nz[a] = 1;
                  }
                }
                if (G1 == 0) break;
              }
            }
            vec4c mP = v_scale(-1, PS[S]);
            int low = S & -S;
            for (int A = S; A > 0; A = (A - 1) & S) {                   /* three-gluon vertex, unordered {A,B} */
              if (!(A & low) || A == S) continue;
              int B = S ^ A;
              for (int a = 0; a < 8; ++a) if (J[A].nz[a]) for (int b = 0; b < 8; ++b) if (J[B].nz[b]) {
                vec4c ja = col_of(J[A].c[a]), jb = col_of(J[B].c[b]);
                vec4c t = oracle_V3(&PS[A], &ja, &PS[B], &jb, &mP);
                for (int c = 0; c < 8; ++c) if (f[a][b][c] != 0) {
                  for (int m = 0; m < 4; ++m) out->c[c][m] += gs * f[a][b][c] * t.c[m];
                  out->nz[c] = 1;
                }
              }
            }
            for (int A = S; A > 0; A = (A - 1) & S) {                   /* four-gluon vertex, unordered {A,B,C} */
              if (!(A & low) || A == S) continue;
              int R = S ^ A, lowR = R & -R;
              for (int B = R; B > 0; B = (B - 1) & R) {
                if (!(B & lowR) || B == R) continue;
                int C = R ^ B;
                for (int a = 0; a < 8; ++a) if (J[A].nz[a]) for (int b = 0; b < 8; ++b) if (J[B].nz[b])
                for (int c = 0; c < 8; ++c) if (J[C].nz[c]) {
                  vec4c ea = col_of(J[A].c[a]), eb = col_of(J[B].c[b]), ec = col_of(J[C].c[c]);
                  cplx ab = mdot_cc(&ea, &eb), ac = mdot_cc(&ea, &ec), bc = mdot_cc(&eb, &ec);
                  for (int d = 0; d < 8; ++d) {
                    real c1 = ff[a][b][c][d], c2 = ff[a][c][b][d], c3 = ff[a][d][b][c];
                    if (c1 == 0 && c2 == 0 && c3 == 0) continue;
                    for (int m = 0; m < 4; ++m) {
                      cplx t1 = ac * eb.c[m] - bc * ea.c[m];
                      cplx t2 = ab * ec.c[m] - bc * ea.c[m];
                      cplx t3 = ab * ec.c[m] - ac * eb.c[m];
                      out->c[d][m] += (-I * gs * gs) * (c1 * t1 + c2 * t2 + c3 * t3);
                    }
                    out->nz[d] = 1;
                  }
                }
              }
            }
            cplx P2 = mdot_cc(&PS[S], &PS[S]);
            for (int a = 0; a < 8; ++a) for (int m = 0; m < 4; ++m) out->c[a][m] *= (-I / P2);
          }
          if (pass == 0) {
            /* light line after the pure-gluon currents: U(G) = i qslash/q^2 sum_A i g T^a Jslash^a(A) U(G \ A), q = f_in + P_G */
            memset(&U[0], 0, sizeof(qcur)); memset(&V[0], 0, sizeof(qcur));
            for (int m = 0; m < 4; ++m) { U[0].c[cin][m] = psi_in.c[m]; V[0].c[cout][m] = psi_out.c[m]; }
            for (int G = 1; G < ngsub; ++G) {
              qcur accu, accv; memset(&accu, 0, sizeof(accu)); memset(&accv, 0, sizeof(accv));
              for (int A = G; A > 0; A = (A - 1) & G) {
                int prev = G ^ A;
                for (int a = 0; a < 8; ++a) if (J[A].nz[a]) {
                  vec4c ja = col_of(J[A].c[a]);
                  mat4c sl = oracle_slash(&ja);
                  for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) if (T[a][k][l] != 0) {
                    vec4c cl = col_of(U[prev].c[l]);
                    vec4c r = mat_times_col(&sl, &cl);
                    for (int m = 0; m < 4; ++m) accu.c[k][m] += I * gs * T[a][k][l] * r.c[m];
                    vec4c row = col_of(V[prev].c[k]);
                    vec4c r2 = row_times_mat(&row, &sl);
                    for (int m = 0; m < 4; ++m) accv.c[l][m] += I * gs * T[a][k][l] * r2.c[m];
                  }
                }
              }
              vec4c qu = v_add(f_in, PS[G]), qv = v_sub(f_out, PS[G]);
              mat4c nu = oracle_slash(&qu), nv = oracle_slash(&qv);
              cplx du = mdot_cc(&qu, &qu), dv = mdot_cc(&qv, &qv);
              for (int k = 0; k < 3; ++k) {
                vec4c cl = col_of(accu.c[k]); vec4c r = mat_times_col(&nu, &cl);
                for (int m = 0; m < 4; ++m) U[G].c[k][m] = (I / du) * r.c[m];
                vec4c row = col_of(accv.c[k]); vec4c r2 = row_times_mat(&row, &nv);
                for (int m = 0; m < 4; ++m) V[G].c[k][m] = (I / dv) * r2.c[m];
              }
            }
          }
        }
        /* ---- top line: Q(S) row with colour index, S = absorbed elements; closes on v(tb) when S is everything ---- */
        for (int ci = 0; ci < 3; ++ci) {          /* colour of the top quark */
        memset(&Q[0], 0, sizeof(qcur));
        for (int m = 0; m < 4; ++m) Q[0].c[ci][m] = ubar.c[m];
        for (int S = 1; S < nsub; ++S) {
          qcur acc; memset(&acc, 0, sizeof(acc));
          for (int A = S; A > 0; A = (A - 1) & S) {
            int prev = S ^ A;
            for (int a = 0; a < 8; ++a) if (J[A].nz[a]) {
              vec4c ja = col_of(J[A].c[a]);
              mat4c sl = oracle_slash(&ja);
              for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) if (T[a][k][l] != 0) {
                vec4c row = col_of(Q[prev].c[k]);
                vec4c r = row_times_mat(&row, &sl);
                for (int m = 0; m < 4; ++m) acc.c[l][m] += I * gs * T[a][k][l] * r.c[m];
              }
            }
          }
          if (S == full) {
            for (int l = 0; l < 3; ++l) { vec4c row = col_of(acc.c[l]); cplx M = row_times_col(&row, &vtb); mh += R_CREAL(conj(M) * M); }
          } else {
            vec4c qq = v_sub(pt, PS[S]);
            mat4c num = m_add_scaled_identity(oracle_slash(&qq), mt);
            cplx den = mdot_cc(&qq, &qq) - mt * mt;
            for (int l = 0; l < 3; ++l) {
              vec4c row = col_of(acc.c[l]); vec4c r = row_times_mat(&row, &num);
              for (int m = 0; m < 4; ++m) Q[S].c[l][m] = (I / den) * r.c[m];
            }
          }
        }
        }
      }
    }
    if (hel_out) hel_out[h] = (double)(mh / s.denom);
    total += mh;
    #undef LAM
  }
  return (double)(total / s.denom);
}

int oracle_me_qchannel_batch(const char* spec, const double* momenta, int64_t nevt, const oracle_params_t* par,
                             double* me_out, int nthreads) {
  qspec s;
  if (parse_spec(spec, &s) != 0) return -1;
#ifdef _OPENMP
  if (nthreads <= 0) nthreads = oracle_num_threads();
#else
  nthreads = 1;
#endif
  #pragma omp parallel for schedule(dynamic, 1) num_threads(nthreads)
  for (int64_t ie = 0; ie < nevt; ++ie)
    me_out[ie] = oracle_me_qchannel(spec, momenta + (size_t)ie * s.npar * 4, par, NULL, -1);
  return 0;
}
