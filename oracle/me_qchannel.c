/* me_qchannel.c — TEST INFRASTRUCTURE (see oracle.h).
 *
 * Quark channels of p p -> t t~ + jets ("pp -> t t~ 0-2 j"): every tree-level QCD
 * process with the top line, one or two massless quark lines and gluons (gluons + light lines <= 4), any crossing:
 *     q q~ -> t t~ (g (g)),  q g -> t t~ q (g),  g q~ -> t t~ q~ (g),  g g -> t t~ q q~,
 *     q q~ -> t t~ r r~,  q r -> t t~ q r,  q q~ -> t t~ q q~,  q q -> t t~ q q,  ...
 * Method: the Feynman rules written out as an off-shell recursion with EXPLICIT colour indices and explicit factors
 * of i (the colour-dressed route C5 of me_ggttng.c, extended by the light quark lines):
 *     quark-gluon vertex  i g T^a_{kl} gamma^mu        quark propagator  i (qslash + m)/(q^2 - m^2)
 *     three-gluon vertex  g f^{abc} V3                 gluon propagator  -i g_{mu nu}/P^2
 *     four-gluon vertex   -i g^2 [f f (g g - g g) + 2 more]
 * Elements of the recursion: the gluons and one PAIR per light line.  J^{a,mu}(S) is the off-shell gluon current of the
 * element subset S; when S holds the pair of line l the current has one more source term,
 * Vbar_l(S1) i g gamma^mu T^a U_l(S2) summed over the splits S1 + S2 of the rest of S between the two ends of that line
 * (U_l, Vbar_l: the line's off-shell spinors with element sets absorbed — gluons, or the other line's pair through its
 * gluon current).  Subsets are visited in increasing numeric order, which respects every dependency.  The top line
 * then absorbs gluon currents exactly as in C5.
 * Two lines of the SAME flavour: the amplitude is M(starts paired with ends one way) - M(the other way) (Fermi
 * statistics), combined colour by colour and helicity by helicity before squaring.
 * |M|^2 = sum over every external colour and helicity, divided by the initial-state spin and colour multiplicities
 * and by k! for k identical final-state particles (A3).
 *
 * Process string `spec`, one character per particle in process order (two incoming first; 't' and 'T' at positions
 * 2 and 3): 'q' / 'Q' light quark / antiquark, 'r' / 'R' quark / antiquark of a second light flavour, 'g' gluon.
 * Examples: "qQtT", "qQtTg", "qgtTq", "gQtTQ", "qQtTgg", "qQtTrR", "qrtTqr", "qQtTqQ", "qqtTqq".
 * Helicity index as everywhere: bit (npar-1-i) of h set <=> particle i has lambda = +1.
 *
 * Pins (tests/test_oracle_qchannel.py): the textbook closed form of q q~ -> t t~ (absolute normalisation, colour
 * average), the Ward identity on every gluon of every process (relative signs between diagram classes), the
 * initial-state collinear limits q -> q g and g -> q q~ onto the closed form (every 1-jet process) and of
 * q q~ -> t t~ g g, q g -> t t~ q g and g g -> t t~ q q~ onto the 1-jet processes, C- and beam-exchange symmetries for
 * the mirrored crossings.  Two light lines: see the test file's header; the SIGN of the interference between the two pairings of the
 * same-flavour processes is a reading with no pin of its own ("parity unpinned" for that term).
 */
#include "oracle_internal.h"

#define MAXEL 4                       /* gluons + light lines */
#define MAXSUB (1 << MAXEL)
typedef struct { cplx c[8][4]; unsigned char nz[8]; } gcur;   /* J^{a,mu}; nz[a] = 0: component a is identically zero */
typedef struct { cplx c[3][4]; } qcur;          /* spinor with a fundamental colour index */

typedef struct {
  int npar, ng, gpart[3];             /* gluon element -> particle index */
  int nl;                             /* light lines */
  int npairing;                       /* 1, or 2 for two lines of the same flavour */
  int start[2][2], end[2][2];         /* [pairing][line]: particles at the start / end of the line's fermion flow */
  real sign[2];                       /* relative sign of the pairing */
  real denom;
} qspec;

/* start of a fermion flow: incoming quark (u) or outgoing antiquark (v); end: outgoing quark (ubar) or incoming antiquark (vbar) */
static int is_start(char c, int incoming) { return ((c == 'q' || c == 'r') ? 1 : 0) == incoming; }

static int parse_spec(const char* spec, qspec* s) {
  int n = (int)strlen(spec);
  if (n < 4 || n > 8 || spec[2] != 't' || spec[3] != 'T') return -1;
  s->npar = n; s->ng = 0;
  int st[2][2], en[2][2], nst[2] = {0, 0}, nen[2] = {0, 0};
  real denom = 1;
  int nfinal[5] = {0, 0, 0, 0, 0};                 /* g q Q r R among the final particles */
  for (int i = 0; i < n; ++i) {
    char c = spec[i]; int incoming = i < 2;
    if (i == 2 || i == 3) continue;
    if (c == 'g') { if (s->ng == 3) return -1; s->gpart[s->ng++] = i; if (incoming) denom *= 16; else ++nfinal[0]; }
    else if (c == 'q' || c == 'Q' || c == 'r' || c == 'R') {
      int fl = (c == 'r' || c == 'R');
      if (is_start(c, incoming)) { if (nst[fl] == 2) return -1; st[fl][nst[fl]++] = i; }
      else                       { if (nen[fl] == 2) return -1; en[fl][nen[fl]++] = i; }
      if (incoming) denom *= 6;
      else ++nfinal[c == 'q' ? 1 : c == 'Q' ? 2 : c == 'r' ? 3 : 4];
    } else return -1;
  }
  if (nst[0] != nen[0] || nst[1] != nen[1] || nst[0] == 0) return -1;
  s->npairing = 1; s->sign[0] = 1; s->sign[1] = -1;
  if (nst[0] == 1 && nst[1] == 0) { s->nl = 1; s->start[0][0] = st[0][0]; s->end[0][0] = en[0][0]; }
  else if (nst[0] == 1 && nst[1] == 1) {
    s->nl = 2;
    s->start[0][0] = st[0][0]; s->end[0][0] = en[0][0];
    s->start[0][1] = st[1][0]; s->end[0][1] = en[1][0];
  } else if (nst[0] == 2 && nst[1] == 0) {           /* same flavour twice: both ways of pairing starts with ends */
    s->nl = 2; s->npairing = 2;
    for (int k = 0; k < 2; ++k) {
      s->start[k][0] = st[0][0]; s->start[k][1] = st[0][1];
      s->end[k][0] = en[0][k]; s->end[k][1] = en[0][1 - k];
    }
  } else return -1;
  if (s->ng + s->nl > MAXEL) return -1;
  for (int t = 0; t < 5; ++t) for (int k = 2; k <= nfinal[t]; ++k) denom *= k;
  s->denom = denom;
  return 0;
}

static inline vec4c col_of(const cplx c[4]) { vec4c r; memcpy(r.c, c, sizeof(r.c)); return r; }

typedef struct {                      /* helicity- and colour-independent tables */
  cplx T[8][3][3];
  real f[8][8][8], ff[8][8][8][8];
  mat4c gmat[4];
  real gs, mt;
} qtab;

static void make_tables(qtab* t, const oracle_params_t* par) {
  t->gs = R_SQRT(4 * R_PI * (real)par->alpha_s); t->mt = par->mt;
  oracle_gellmann_T(t->T);
  for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {     /* f^{abc} = -2i Tr([T^a,T^b] T^c) */
    cplx tr = 0;
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k)
      tr += (t->T[a][i][j] * t->T[b][j][k] - t->T[b][i][j] * t->T[a][j][k]) * t->T[c][k][i];
    t->f[a][b][c] = R_CREAL(-2 * I * tr);
  }
  /* f^{abe} f^{cde}: the three colour structures of the four-gluon vertex are ff[a][b][c][d], ff[a][c][b][d], ff[a][d][b][c] */
  for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) for (int d = 0; d < 8; ++d) {
    real v = 0; for (int e = 0; e < 8; ++e) v += t->f[a][b][e] * t->f[c][d][e];
    t->ff[a][b][c][d] = v;
  }
  for (int mu = 0; mu < 4; ++mu) oracle_gamma_mat(mu, &t->gmat[mu]);
}

typedef struct {                      /* external wavefunctions of one helicity configuration */
  vec4c Pg[3], eps[3];                /* gluons: incoming momentum, polarisation */
  vec4c psi[8], flow[8];              /* light-quark particles: spinor (column at a start, row at an end) and the momentum
                                         carried along the fermion arrow (+p for quarks, -p for antiquarks) */
  vec4c pt, ubar, vtb;
} qext;

/* M[i][l], i / l = colour of the top / antitop: the amplitude of one pairing for fixed colours of the other externals */
static void amplitude(const qspec* s, const qtab* t, const qext* x, int pairing, const int* gcol, const int* qcolour,
                      cplx M[3][3]) {
  const int ng = s->ng, nl = s->nl, nel = ng + nl, nsub = 1 << nel, full = nsub - 1;
  const real gs = t->gs, mt = t->mt;
  vec4c P[MAXEL], PS[MAXSUB];
  for (int g = 0; g < ng; ++g) P[g] = x->Pg[g];
  for (int l = 0; l < nl; ++l)        /* what the pair brings into the rest: f_in - f_out */
    P[ng + l] = v_sub(x->flow[s->start[pairing][l]], x->flow[s->end[pairing][l]]);
  for (int S = 0; S < nsub; ++S) { PS[S] = v_zero(); for (int e = 0; e < nel; ++e) if (S >> e & 1) PS[S] = v_add(PS[S], P[e]); }
  gcur J[MAXSUB]; qcur U[2][MAXSUB], V[2][MAXSUB], Q[MAXSUB];
  for (int l = 0; l < nl; ++l) {
    memset(&U[l][0], 0, sizeof(qcur)); memset(&V[l][0], 0, sizeof(qcur));
    const int ps = s->start[pairing][l], pe = s->end[pairing][l];
    for (int m = 0; m < 4; ++m) { U[l][0].c[qcolour[ps]][m] = x->psi[ps].c[m]; V[l][0].c[qcolour[pe]][m] = x->psi[pe].c[m]; }
  }
  for (int S = 1; S < nsub; ++S) {
    /* ---- gluon current of the element set S ---- */
    gcur* out = &J[S]; memset(out, 0, sizeof(*out));
    if (S < (1 << ng) && (S & (S - 1)) == 0) {                          /* external gluon */
      int g = 0; while (!((S >> g) & 1)) ++g;
      for (int m = 0; m < 4; ++m) out->c[gcol[g]][m] = x->eps[g].c[m];
      out->nz[gcol[g]] = 1;
    } else {
      for (int l = 0; l < nl; ++l) if (S >> (ng + l) & 1) {             /* source: light line l emits the gluon */
        const int G = S ^ (1 << (ng + l));
        for (int G1 = G;; G1 = (G1 - 1) & G) {
          const int G2 = G ^ G1;
          for (int mu = 0; mu < 4; ++mu) for (int a = 0; a < 8; ++a) {
            cplx acc = 0;
            for (int k = 0; k < 3; ++k) for (int c = 0; c < 3; ++c) if (t->T[a][k][c] != 0) {
              vec4c row = col_of(V[l][G1].c[k]), cl = col_of(U[l][G2].c[c]);
              vec4c r = row_times_mat(&row, &t->gmat[mu]);
              acc += t->T[a][k][c] * row_times_col(&r, &cl);
            }
            out->c[a][mu] += I * gs * acc;                              /* i g T^a gamma^mu (upper index mu) */
            out->nz[a] = 1;
          }
          if (G1 == 0) break;
        }
      }
      vec4c mP = v_scale(-1, PS[S]);
      const int low = S & -S;
      for (int A = S; A > 0; A = (A - 1) & S) {                         /* three-gluon vertex, unordered {A,B} */
        if (!(A & low) || A == S) continue;
        const int B = S ^ A;
        for (int a = 0; a < 8; ++a) if (J[A].nz[a]) for (int b = 0; b < 8; ++b) if (J[B].nz[b]) {
          vec4c ja = col_of(J[A].c[a]), jb = col_of(J[B].c[b]);
          vec4c v3 = oracle_V3(&PS[A], &ja, &PS[B], &jb, &mP);
          for (int c = 0; c < 8; ++c) if (t->f[a][b][c] != 0) {
            for (int m = 0; m < 4; ++m) out->c[c][m] += gs * t->f[a][b][c] * v3.c[m];
            out->nz[c] = 1;
          }
        }
      }
      for (int A = S; A > 0; A = (A - 1) & S) {                         /* four-gluon vertex, unordered {A,B,C} */
        if (!(A & low) || A == S) continue;
        const int R = S ^ A, lowR = R & -R;
        for (int B = R; B > 0; B = (B - 1) & R) {
          if (!(B & lowR) || B == R) continue;
          const int C = R ^ B;
          for (int a = 0; a < 8; ++a) if (J[A].nz[a]) for (int b = 0; b < 8; ++b) if (J[B].nz[b])
          for (int c = 0; c < 8; ++c) if (J[C].nz[c]) {
            vec4c ea = col_of(J[A].c[a]), eb = col_of(J[B].c[b]), ec = col_of(J[C].c[c]);
            cplx ab = mdot_cc(&ea, &eb), ac = mdot_cc(&ea, &ec), bc = mdot_cc(&eb, &ec);
            for (int d = 0; d < 8; ++d) {
              real c1 = t->ff[a][b][c][d], c2 = t->ff[a][c][b][d], c3 = t->ff[a][d][b][c];
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
    /* ---- the light lines that do not own an element of S absorb it:
     *      U_l(S) = i qslash/q^2 sum_A i g T^a Jslash^a(A) U_l(S \ A),  q = f_in + P_S;  Vbar_l(S) likewise, q = f_out - P_S ---- */
    for (int l = 0; l < nl; ++l) {
      if (S >> (ng + l) & 1) continue;
      qcur accu, accv; memset(&accu, 0, sizeof(accu)); memset(&accv, 0, sizeof(accv));
      for (int A = S; A > 0; A = (A - 1) & S) {
        const int prev = S ^ A;
        for (int a = 0; a < 8; ++a) if (J[A].nz[a]) {
          vec4c ja = col_of(J[A].c[a]);
          mat4c sl = oracle_slash(&ja);
          for (int k = 0; k < 3; ++k) for (int c = 0; c < 3; ++c) if (t->T[a][k][c] != 0) {
            vec4c cl = col_of(U[l][prev].c[c]);
            vec4c r = mat_times_col(&sl, &cl);
            for (int m = 0; m < 4; ++m) accu.c[k][m] += I * gs * t->T[a][k][c] * r.c[m];
            vec4c row = col_of(V[l][prev].c[k]);
            vec4c r2 = row_times_mat(&row, &sl);
            for (int m = 0; m < 4; ++m) accv.c[c][m] += I * gs * t->T[a][k][c] * r2.c[m];
          }
        }
      }
      vec4c qu = v_add(x->flow[s->start[pairing][l]], PS[S]), qv = v_sub(x->flow[s->end[pairing][l]], PS[S]);
      mat4c nu = oracle_slash(&qu), nv = oracle_slash(&qv);
      cplx du = mdot_cc(&qu, &qu), dv = mdot_cc(&qv, &qv);
      for (int k = 0; k < 3; ++k) {
        vec4c cl = col_of(accu.c[k]); vec4c r = mat_times_col(&nu, &cl);
        for (int m = 0; m < 4; ++m) U[l][S].c[k][m] = (I / du) * r.c[m];
        vec4c row = col_of(accv.c[k]); vec4c r2 = row_times_mat(&row, &nv);
        for (int m = 0; m < 4; ++m) V[l][S].c[k][m] = (I / dv) * r2.c[m];
      }
    }
  }
  /* ---- top line: Q(S) row with colour index, S = absorbed elements; closes on v(tb) when S is everything ---- */
  for (int ci = 0; ci < 3; ++ci) {
  memset(&Q[0], 0, sizeof(qcur));
  for (int m = 0; m < 4; ++m) Q[0].c[ci][m] = x->ubar.c[m];
  for (int S = 1; S < nsub; ++S) {
    qcur acc; memset(&acc, 0, sizeof(acc));
    for (int A = S; A > 0; A = (A - 1) & S) {
      const int prev = S ^ A;
      for (int a = 0; a < 8; ++a) if (J[A].nz[a]) {
        vec4c ja = col_of(J[A].c[a]);
        mat4c sl = oracle_slash(&ja);
        for (int k = 0; k < 3; ++k) for (int c = 0; c < 3; ++c) if (t->T[a][k][c] != 0) {
          vec4c row = col_of(Q[prev].c[k]);
          vec4c r = row_times_mat(&row, &sl);
          for (int m = 0; m < 4; ++m) acc.c[c][m] += I * gs * t->T[a][k][c] * r.c[m];
        }
      }
    }
    if (S == full) {
      for (int c = 0; c < 3; ++c) { vec4c row = col_of(acc.c[c]); M[ci][c] = row_times_col(&row, &x->vtb); }
    } else {
      vec4c qq = v_sub(x->pt, PS[S]);
      mat4c num = m_add_scaled_identity(oracle_slash(&qq), mt);
      cplx den = mdot_cc(&qq, &qq) - mt * mt;
      for (int c = 0; c < 3; ++c) {
        vec4c row = col_of(acc.c[c]); vec4c r = row_times_mat(&row, &num);
        for (int m = 0; m < 4; ++m) Q[S].c[c][m] = (I / den) * r.c[m];
      }
    }
  }
  }
}

/* pauli != 0: only the helicity and colour configurations in which the two identical final-state quarks (particles 4 and 5)
 * are in the same spin and colour state are summed (diagnostic for the Pauli-principle pin) */
static double me_q(const char* spec, const double* p, const oracle_params_t* par, double* hel_out, int ward_which, int pauli) {
  qspec s;
  if (parse_spec(spec, &s) != 0) return -1;
  const int npar = s.npar, ng = s.ng, nhel = 1 << npar;
  qtab* t = (qtab*)malloc(sizeof(qtab));
  make_tables(t, par);
  int qpart[4], nq = 0;               /* the light-quark particles */
  for (int i = 0; i < npar; ++i) if (spec[i] == 'q' || spec[i] == 'Q' || spec[i] == 'r' || spec[i] == 'R') qpart[nq++] = i;
  int64_t ngcol = 1; for (int g = 0; g < ng; ++g) ngcol *= 8;
  int nqcol = 1; for (int i = 0; i < nq; ++i) nqcol *= 3;
  real q[4];
  real total = 0;
  for (int h = 0; h < nhel; ++h) {
    #define LAM(i) (((h >> (npar - 1 - (i))) & 1) ? 1 : -1)
    if (pauli && LAM(4) != LAM(5)) { if (hel_out) hel_out[h] = 0; continue; }
    qext x;
    for (int g = 0; g < ng; ++g) {
      int ip = s.gpart[g];
      for (int m = 0; m < 4; ++m) q[m] = p[4 * ip + m];
      vec4c e = oracle_eps(q, LAM(ip));
      if (ip < 2) { x.Pg[g] = v_from_real(q); x.eps[g] = e; }
      else        { x.Pg[g] = v_scale(-1, v_from_real(q)); x.eps[g] = oracle_conj(&e); }
      if (g == ward_which) x.eps[g] = x.Pg[g];
    }
    for (int k = 0; k < nq; ++k) {
      int ip = qpart[k], incoming = ip < 2, quark = (spec[ip] == 'q' || spec[ip] == 'r');
      for (int m = 0; m < 4; ++m) q[m] = p[4 * ip + m];
      vec4c w = (quark ? oracle_u(q, 0, LAM(ip)) : oracle_v(q, 0, LAM(ip)));
      /* incoming quark u, outgoing antiquark v: columns;  outgoing quark ubar, incoming antiquark vbar: rows */
      x.psi[ip] = is_start(spec[ip], incoming) ? w : oracle_bar(&w);
      x.flow[ip] = v_scale(quark ? 1 : -1, v_from_real(q));
    }
    for (int m = 0; m < 4; ++m) q[m] = p[8 + m];
    x.pt = v_from_real(q);
    { vec4c ut = oracle_u(q, t->mt, LAM(2)); x.ubar = oracle_bar(&ut); }
    for (int m = 0; m < 4; ++m) q[m] = p[12 + m];
    x.vtb = oracle_v(q, t->mt, LAM(3));
    real mh = 0;
    for (int64_t ic = 0; ic < ngcol; ++ic) {
      int gcol[3] = {0, 0, 0}; { int64_t r = ic; for (int g = 0; g < ng; ++g) { gcol[g] = (int)(r % 8); r /= 8; } }
      for (int iq = 0; iq < nqcol; ++iq) {
        int qcolour[8] = {0, 0, 0, 0, 0, 0, 0, 0}; { int r = iq; for (int k = 0; k < nq; ++k) { qcolour[qpart[k]] = r % 3; r /= 3; } }
        if (pauli && qcolour[4] != qcolour[5]) continue;
        cplx M[3][3]; memset(M, 0, sizeof(M));
        for (int k = 0; k < s.npairing; ++k) {
          cplx Mk[3][3];
          amplitude(&s, t, &x, k, gcol, qcolour, Mk);
          for (int i = 0; i < 3; ++i) for (int c = 0; c < 3; ++c) M[i][c] += s.sign[k] * Mk[i][c];
        }
        for (int i = 0; i < 3; ++i) for (int c = 0; c < 3; ++c) mh += R_CREAL(conj(M[i][c]) * M[i][c]);
      }
    }
    if (hel_out) hel_out[h] = (double)(mh / s.denom);
    total += mh;
    #undef LAM
  }
  free(t);
  return (double)(total / s.denom);
}

double oracle_me_qchannel(const char* spec, const double* p, const oracle_params_t* par, double* hel_out, int ward_which) {
  return me_q(spec, p, par, hel_out, ward_which, 0);
}
/* Pauli principle (pin of the relative sign of the two pairings): for two identical final-state quarks with the same
 * momentum, helicity and colour the amplitude vanishes.  Returns the part of |M|^2 (same normalisation) from the
 * configurations with equal helicity and colour of particles 4 and 5; the caller passes p4 = p5.  -1 unless the
 * process ends in two identical (anti)quarks. */
double oracle_me_qchannel_pauli(const char* spec, const double* p, const oracle_params_t* par) {
  if (strlen(spec) != 6 || spec[4] != spec[5] || (spec[4] != 'q' && spec[4] != 'Q')) return -1;
  return me_q(spec, p, par, NULL, -1, 1);
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
