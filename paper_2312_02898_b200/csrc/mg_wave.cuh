// mg_wave.cuh — device routines for the event-parallel helicity-amplitude kernels (K3, K4, K5 of
// SURVEY.md §8(a); "compute probability amplitudes ('matrix elements')"
// "identical for every event ... almost branch free").  One thread owns one event; every object below
// lives in that thread's registers.  Conventions:
//   metric (+,-,-,-), momenta (E,px,py,pz); Weyl (chiral) gamma matrices, so for a 4-vector a
//       aslash = [[0, M-(a)], [M+(a), 0]],  M+-(a) = a0 +- a.sigma  (2x2 blocks);
//   gluons carry *incoming* momenta P (P = +p for beams, -p for final-state gluons);
//   colour-ordered vertex functions with the coupling and phases stripped:
//       ggg   : j(A,B)   = -V3(P_A,j_A; P_B,j_B; -P_A-P_B) / P^2
//       gggg  : j(A,M,C) = -[(A.M) C + (M.C) A - 2 (A.C) M] / P^2
//       quark : Lbar' = -Lbar jslash (qslash + m)/(q^2 - m^2),  R' = -(qslash + m) jslash R/(q^2 - m^2)
//   (each vertex carries g_s, each quark vertex/propagator pair i*i = -1, the closing vertex one common
//    factor i; |M|^2 is multiplied by g_s^{2n} once at the end.)
// T is double (MG_FP64) or float (MG_FP32).  Nothing here is shared with oracle/.
#pragma once
#ifndef MG_DEV
#define MG_DEV __device__ __forceinline__
#endif

namespace mgw {

template <class T> struct W4 {   // four complex components
  T r[4];
  T i[4];
};
template <class T> struct P4 {   // real 4-vector
  T c[4];
};
template <class T> struct C1 {   // one complex number
  T r, i;
};

template <class T> MG_DEV T rsq(T x);
template <> MG_DEV double rsq<double>(double x) { return sqrt(x); }
template <> MG_DEV float rsq<float>(float x) { return sqrtf(x); }

template <class T> MG_DEV P4<T> padd(const P4<T>& a, const P4<T>& b) {
  P4<T> o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.c[m] = a.c[m] + b.c[m];
  return o;
}
template <class T> MG_DEV P4<T> psub(const P4<T>& a, const P4<T>& b) {
  P4<T> o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.c[m] = a.c[m] - b.c[m];
  return o;
}
template <class T, class S> MG_DEV P4<T> pcast(const P4<S>& a) {
  P4<T> o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.c[m] = T(a.c[m]);
  return o;
}
template <class T> MG_DEV T pdot(const P4<T>& a, const P4<T>& b) {
  return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3];
}

// ---------------------------------------------------------------------------------------------
// K3: external wavefunctions
// ---------------------------------------------------------------------------------------------

// Gluon polarisation vector for physical momentum k, lambda = +-1 (circular, helicity basis):
//   eps(k,lambda) = (-lambda e1 - i e2)/sqrt2, e1 = (0, kx kz, ky kz, -kT^2)/(|k| kT), e2 = (0,-ky,kx,0)/kT.
// conj = false: incoming (eps); conj = true: outgoing (eps*).
template <class T> MG_DEV void ext_gluon(const P4<T>& k, int lambda, bool conj, W4<T>& e) {
  const T rs2 = T(0.70710678118654752440);
  T kt2 = k.c[1] * k.c[1] + k.c[2] * k.c[2];
  T sl = (lambda > 0) ? -rs2 : rs2;      // -lambda/sqrt2
  T si = conj ? rs2 : -rs2;              // coefficient of e2 in the imaginary part
  e.r[0] = T(0); e.i[0] = T(0);
  if (kt2 == T(0)) {
    e.r[1] = sl; e.r[2] = T(0); e.r[3] = T(0);
    e.i[1] = T(0); e.i[2] = (k.c[3] >= T(0)) ? si : -si; e.i[3] = T(0);
  } else {
    T kk = rsq(kt2 + k.c[3] * k.c[3]);
    T kt = rsq(kt2);
    T ikt = T(1) / kt;
    T ikk = T(1) / kk;
    T a = sl * k.c[3] * ikk * ikt;
    e.r[1] = a * k.c[1];
    e.r[2] = a * k.c[2];
    e.r[3] = -sl * kt * ikk;
    e.i[1] = -si * k.c[2] * ikt;
    e.i[2] = si * k.c[1] * ikt;
    e.i[3] = T(0);
  }
}

// Two-component helicity eigenspinors chi_+(p), chi_-(p) (unit norm).
template <class T> MG_DEV void chi_pm(const P4<T>& p, T pp, C1<T> cp[2], C1<T> cm[2]) {
  // |p| + pz without cancellation for backward momenta: (|p| + pz)(|p| - pz) = kT^2
  const T kt2 = p.c[1] * p.c[1] + p.c[2] * p.c[2];
  T s = (p.c[3] >= T(0)) ? pp + p.c[3] : kt2 / (pp - p.c[3]);
  if (pp == T(0)) {                       // at rest: quantise along +z
    cp[0] = {T(1), T(0)}; cp[1] = {T(0), T(0)};
    cm[0] = {T(0), T(0)}; cm[1] = {T(1), T(0)};
  } else if (s <= T(0)) {                 // along -z
    cp[0] = {T(0), T(0)}; cp[1] = {T(1), T(0)};
    cm[0] = {T(-1), T(0)}; cm[1] = {T(0), T(0)};
  } else {
    T nn = T(1) / rsq(T(2) * pp * s);
    cp[0] = {s * nn, T(0)};              cp[1] = {p.c[1] * nn, p.c[2] * nn};
    cm[0] = {-p.c[1] * nn, p.c[2] * nn}; cm[1] = {s * nn, T(0)};
  }
}

// Outgoing fermion: row spinor ubar(p,lambda) = u^dagger gamma^0, u = (w_{-l} chi_l, w_l chi_l),
// w_+- = sqrt(E +- |p|) (w_- = 0 exactly if m == 0).
template <class T> MG_DEV void ext_ubar(const P4<T>& p, T m, int lambda, W4<T>& o) {
  T pp = rsq(p.c[1] * p.c[1] + p.c[2] * p.c[2] + p.c[3] * p.c[3]);
  T wp = rsq(p.c[0] + pp);
  T wm = (m == T(0)) ? T(0) : m / wp;     // sqrt(E-|p|) = m / sqrt(E+|p|), no cancellation
  C1<T> cp[2], cm[2];
  chi_pm(p, pp, cp, cm);
  const C1<T>* ch = (lambda > 0) ? cp : cm;
  T wl = (lambda > 0) ? wp : wm;          // w_{lambda}
  T wo = (lambda > 0) ? wm : wp;          // w_{-lambda}
  // ubar = (conj(u_lower), conj(u_upper)) = (w_l chi^*, w_{-l} chi^*)
  o.r[0] = wl * ch[0].r; o.i[0] = -wl * ch[0].i;
  o.r[1] = wl * ch[1].r; o.i[1] = -wl * ch[1].i;
  o.r[2] = wo * ch[0].r; o.i[2] = -wo * ch[0].i;
  o.r[3] = wo * ch[1].r; o.i[3] = -wo * ch[1].i;
}

// Outgoing antifermion: column spinor v(p,lambda) = (-l w_l chi_{-l}, l w_{-l} chi_{-l}).
template <class T> MG_DEV void ext_v(const P4<T>& p, T m, int lambda, W4<T>& o) {
  T pp = rsq(p.c[1] * p.c[1] + p.c[2] * p.c[2] + p.c[3] * p.c[3]);
  T wp = rsq(p.c[0] + pp);
  T wm = (m == T(0)) ? T(0) : m / wp;
  C1<T> cp[2], cm[2];
  chi_pm(p, pp, cp, cm);
  const C1<T>* ch = (lambda > 0) ? cm : cp;   // chi_{-lambda}
  T wl = (lambda > 0) ? wp : wm;
  T wo = (lambda > 0) ? wm : wp;
  T a = (lambda > 0) ? -wl : wl;              // -lambda w_lambda
  T b = (lambda > 0) ? wo : -wo;              //  lambda w_{-lambda}
  o.r[0] = a * ch[0].r; o.i[0] = a * ch[0].i;
  o.r[1] = a * ch[1].r; o.i[1] = a * ch[1].i;
  o.r[2] = b * ch[0].r; o.i[2] = b * ch[0].i;
  o.r[3] = b * ch[1].r; o.i[3] = b * ch[1].i;
}
// Incoming fermion u(p,lambda) (column) and incoming antifermion vbar(p,lambda) (row) — used by the
// e+ e- -> mu+ mu- kernel (massless beams, but written for general m).
template <class T> MG_DEV void ext_u(const P4<T>& p, T m, int lambda, W4<T>& o) {
  T pp = rsq(p.c[1] * p.c[1] + p.c[2] * p.c[2] + p.c[3] * p.c[3]);
  T wp = rsq(p.c[0] + pp);
  T wm = (m == T(0)) ? T(0) : m / wp;
  C1<T> cp[2], cm[2];
  chi_pm(p, pp, cp, cm);
  const C1<T>* ch = (lambda > 0) ? cp : cm;
  T wl = (lambda > 0) ? wp : wm;
  T wo = (lambda > 0) ? wm : wp;
  o.r[0] = wo * ch[0].r; o.i[0] = wo * ch[0].i;
  o.r[1] = wo * ch[1].r; o.i[1] = wo * ch[1].i;
  o.r[2] = wl * ch[0].r; o.i[2] = wl * ch[0].i;
  o.r[3] = wl * ch[1].r; o.i[3] = wl * ch[1].i;
}
template <class T> MG_DEV void ext_vbar(const P4<T>& p, T m, int lambda, W4<T>& o) {
  W4<T> v;
  ext_v(p, m, lambda, v);
  // vbar = v^dagger gamma^0 = (conj(v_lower), conj(v_upper))
  o.r[0] = v.r[2]; o.i[0] = -v.i[2];
  o.r[1] = v.r[3]; o.i[1] = -v.i[3];
  o.r[2] = v.r[0]; o.i[2] = -v.i[0];
  o.r[3] = v.r[1]; o.i[3] = -v.i[1];
}

// ---------------------------------------------------------------------------------------------
// K4: internal currents
// ---------------------------------------------------------------------------------------------

// complex Minkowski product a.b (no conjugation)
template <class T> MG_DEV C1<T> wdot(const W4<T>& a, const W4<T>& b) {
  C1<T> d;
  d.r = a.r[0] * b.r[0] - a.i[0] * b.i[0];
  d.i = a.r[0] * b.i[0] + a.i[0] * b.r[0];
#pragma unroll
  for (int m = 1; m < 4; ++m) {
    d.r = d.r - a.r[m] * b.r[m] + a.i[m] * b.i[m];
    d.i = d.i - a.r[m] * b.i[m] - a.i[m] * b.r[m];
  }
  return d;
}
// real 4-vector . complex 4-vector
template <class T> MG_DEV C1<T> pwdot(const P4<T>& p, const W4<T>& b) {
  C1<T> d;
  d.r = p.c[0] * b.r[0] - p.c[1] * b.r[1] - p.c[2] * b.r[2] - p.c[3] * b.r[3];
  d.i = p.c[0] * b.i[0] - p.c[1] * b.i[1] - p.c[2] * b.i[2] - p.c[3] * b.i[3];
  return d;
}

// ggg -> off-shell gluon.  j = s * V3(PA,jA; PB,jB; -(PA+PB)),  s = -1/(PA+PB)^2 (passed in):
//   V3^mu = (jA.jB)(PA-PB)^mu + jB^mu ((2PB+PA).jA) - jA^mu ((2PA+PB).jB)
template <class T>
MG_DEV void cur_v3(const P4<T>& PA, const W4<T>& jA, const P4<T>& PB, const W4<T>& jB, T s, W4<T>& o) {
  C1<T> d = wdot(jA, jB);
  P4<T> qa, qb;
#pragma unroll
  for (int m = 0; m < 4; ++m) { qa.c[m] = T(2) * PB.c[m] + PA.c[m]; qb.c[m] = T(2) * PA.c[m] + PB.c[m]; }
  C1<T> a = pwdot(qa, jA);
  C1<T> b = pwdot(qb, jB);
  d.r *= s; d.i *= s; a.r *= s; a.i *= s; b.r *= -s; b.i *= -s;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    T dp = PA.c[m] - PB.c[m];
    o.r[m] = d.r * dp + a.r * jB.r[m] - a.i * jB.i[m] + b.r * jA.r[m] - b.i * jA.i[m];
    o.i[m] = d.i * dp + a.r * jB.i[m] + a.i * jB.r[m] + b.r * jA.i[m] + b.i * jA.r[m];
  }
}

// gggg kinematic structure with M in the middle:  j = s * [(A.M) C + (M.C) A - 2 (A.C) M],  s = -1/P^2.
template <class T>
MG_DEV void cur_k(const W4<T>& A, const W4<T>& M, const W4<T>& C, T s, W4<T>& o) {
  C1<T> am = wdot(A, M), mc = wdot(M, C), ac = wdot(A, C);
  am.r *= s; am.i *= s; mc.r *= s; mc.i *= s; ac.r *= T(-2) * s; ac.i *= T(-2) * s;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    o.r[m] = am.r * C.r[m] - am.i * C.i[m] + mc.r * A.r[m] - mc.i * A.i[m] + ac.r * M.r[m] - ac.i * M.i[m];
    o.i[m] = am.r * C.i[m] + am.i * C.r[m] + mc.r * A.i[m] + mc.i * A.r[m] + ac.r * M.i[m] + ac.i * M.r[m];
  }
}

// 2x2 blocks of aslash for a complex vector a:  M+ = [[a0+a3, a1-i a2],[a1+i a2, a0-a3]],
//                                               M- = [[a0-a3,-a1+i a2],[-a1-i a2, a0+a3]].
template <class T> struct M2 { C1<T> m00, m01, m10, m11; };
template <class T> MG_DEV void slash_blocks(const W4<T>& a, M2<T>& mp, M2<T>& mm) {
  mp.m00 = {a.r[0] + a.r[3], a.i[0] + a.i[3]};
  mp.m11 = {a.r[0] - a.r[3], a.i[0] - a.i[3]};
  mp.m01 = {a.r[1] + a.i[2], a.i[1] - a.r[2]};   // a1 - i a2
  mp.m10 = {a.r[1] - a.i[2], a.i[1] + a.r[2]};   // a1 + i a2
  mm.m00 = mp.m11; mm.m11 = mp.m00;
  mm.m01 = {-mp.m01.r, -mp.m01.i};
  mm.m10 = {-mp.m10.r, -mp.m10.i};
}
#define MG_CMUL_R(x, y) ((x).r * (y).r - (x).i * (y).i)
#define MG_CMUL_I(x, y) ((x).r * (y).i + (x).i * (y).r)

// row (x0,x1) times 2x2
template <class T> MG_DEV void row2(const C1<T>& x0, const C1<T>& x1, const M2<T>& m, C1<T>& y0, C1<T>& y1) {
  y0.r = MG_CMUL_R(x0, m.m00) + MG_CMUL_R(x1, m.m10);
  y0.i = MG_CMUL_I(x0, m.m00) + MG_CMUL_I(x1, m.m10);
  y1.r = MG_CMUL_R(x0, m.m01) + MG_CMUL_R(x1, m.m11);
  y1.i = MG_CMUL_I(x0, m.m01) + MG_CMUL_I(x1, m.m11);
}
// 2x2 times column (x0,x1)
template <class T> MG_DEV void col2(const M2<T>& m, const C1<T>& x0, const C1<T>& x1, C1<T>& y0, C1<T>& y1) {
  y0.r = MG_CMUL_R(m.m00, x0) + MG_CMUL_R(m.m01, x1);
  y0.i = MG_CMUL_I(m.m00, x0) + MG_CMUL_I(m.m01, x1);
  y1.r = MG_CMUL_R(m.m10, x0) + MG_CMUL_R(m.m11, x1);
  y1.i = MG_CMUL_I(m.m10, x0) + MG_CMUL_I(m.m11, x1);
}

// Quark-line step from the top side (row spinor):  o = s * L jslash (qslash + m),  s = -1/(q^2-m^2).
// quark-line steps with the helicity-independent propagator factors prepared once per event:
//   qp = s (q0 + q3), qm = s (q0 - q3), sq1 = s q1, sq2 = s q2, ms = s m
template <class T> MG_DEV void cur_lqp(const W4<T>& L, const W4<T>& j, T qp, T qm, T sq1, T sq2, T ms, W4<T>& o);
template <class T> MG_DEV void cur_rqp(const W4<T>& R, const W4<T>& j, T qp, T qm, T sq1, T sq2, T ms, W4<T>& o);
template <class T>
MG_DEV void cur_lq(const W4<T>& L, const W4<T>& j, const P4<T>& q, T m, T s, W4<T>& o) {
  cur_lqp(L, j, s * (q.c[0] + q.c[3]), s * (q.c[0] - q.c[3]), s * q.c[1], s * q.c[2], m * s, o);
}
template <class T>
MG_DEV void cur_lqp(const W4<T>& L, const W4<T>& j, T qp, T qm, T sq1, T sq2, T ms, W4<T>& o) {
  M2<T> mp, mm;
  slash_blocks(j, mp, mm);
  C1<T> lu0 = {L.r[0], L.i[0]}, lu1 = {L.r[1], L.i[1]}, ll0 = {L.r[2], L.i[2]}, ll1 = {L.r[3], L.i[3]};
  C1<T> tu0, tu1, tl0, tl1;
  row2(ll0, ll1, mp, tu0, tu1);      // (L jslash)_U = L_L M+(j)
  row2(lu0, lu1, mm, tl0, tl1);      // (L jslash)_L = L_U M-(j)
  // times (qslash + m), q real:  res_U = t_L M+(q) + m t_U ; res_L = t_U M-(q) + m t_L
  // M+(q) = [[qp, q1 - i q2],[q1 + i q2, qm]]
  o.r[0] = ms * tu0.r + tl0.r * qp + tl1.r * sq1 - tl1.i * sq2;
  o.i[0] = ms * tu0.i + tl0.i * qp + tl1.i * sq1 + tl1.r * sq2;
  o.r[1] = ms * tu1.r + tl1.r * qm + tl0.r * sq1 + tl0.i * sq2;
  o.i[1] = ms * tu1.i + tl1.i * qm + tl0.i * sq1 - tl0.r * sq2;
  // M-(q) = [[qm, -q1 + i q2],[-q1 - i q2, qp]]
  o.r[2] = ms * tl0.r + tu0.r * qm - tu1.r * sq1 + tu1.i * sq2;
  o.i[2] = ms * tl0.i + tu0.i * qm - tu1.i * sq1 - tu1.r * sq2;
  o.r[3] = ms * tl1.r + tu1.r * qp - tu0.r * sq1 - tu0.i * sq2;
  o.i[3] = ms * tl1.i + tu1.i * qp - tu0.i * sq1 + tu0.r * sq2;
}

// Quark-line step from the antitop side (column spinor):  o = s * (qslash + m) jslash R,  s = -1/(q^2-m^2).
template <class T>
MG_DEV void cur_rq(const W4<T>& R, const W4<T>& j, const P4<T>& q, T m, T s, W4<T>& o) {
  cur_rqp(R, j, s * (q.c[0] + q.c[3]), s * (q.c[0] - q.c[3]), s * q.c[1], s * q.c[2], m * s, o);
}
template <class T>
MG_DEV void cur_rqp(const W4<T>& R, const W4<T>& j, T qp, T qm, T sq1, T sq2, T ms, W4<T>& o) {
  M2<T> mp, mm;
  slash_blocks(j, mp, mm);
  C1<T> ru0 = {R.r[0], R.i[0]}, ru1 = {R.r[1], R.i[1]}, rl0 = {R.r[2], R.i[2]}, rl1 = {R.r[3], R.i[3]};
  C1<T> tu0, tu1, tl0, tl1;
  col2(mm, rl0, rl1, tu0, tu1);      // (jslash R)_U = M-(j) R_L
  col2(mp, ru0, ru1, tl0, tl1);      // (jslash R)_L = M+(j) R_U
  // (qslash + m) t:  res_U = M-(q) t_L + m t_U ; res_L = M+(q) t_U + m t_L
  // M-(q) = [[qm, -q1 + i q2],[-q1 - i q2, qp]]
  o.r[0] = ms * tu0.r + qm * tl0.r - sq1 * tl1.r - sq2 * tl1.i;
  o.i[0] = ms * tu0.i + qm * tl0.i - sq1 * tl1.i + sq2 * tl1.r;
  o.r[1] = ms * tu1.r + qp * tl1.r - sq1 * tl0.r + sq2 * tl0.i;
  o.i[1] = ms * tu1.i + qp * tl1.i - sq1 * tl0.i - sq2 * tl0.r;
  // M+(q) = [[qp, q1 - i q2],[q1 + i q2, qm]]
  o.r[2] = ms * tl0.r + qp * tu0.r + sq1 * tu1.r + sq2 * tu1.i;
  o.i[2] = ms * tl0.i + qp * tu0.i + sq1 * tu1.i - sq2 * tu1.r;
  o.r[3] = ms * tl1.r + qm * tu1.r + sq1 * tu0.r - sq2 * tu0.i;
  o.i[3] = ms * tl1.i + qm * tu1.i + sq1 * tu0.i + sq2 * tu0.r;
}

// ---------------------------------------------------------------------------------------------
// K5: amplitudes.  The closing quark-gluon vertex  L jslash R = B_mu j^mu  with the bilinear
// B_mu = L gamma_mu R (index lowered) shared by every diagram that closes on the same (L, R).
// ---------------------------------------------------------------------------------------------
template <class T> MG_DEV void bilinear(const W4<T>& L, const W4<T>& R, W4<T>& B) {
  C1<T> a0 = {L.r[0], L.i[0]}, a1 = {L.r[1], L.i[1]}, c0 = {L.r[2], L.i[2]}, c1 = {L.r[3], L.i[3]};
  C1<T> d0 = {R.r[0], R.i[0]}, d1 = {R.r[1], R.i[1]}, b0 = {R.r[2], R.i[2]}, b1 = {R.r[3], R.i[3]};
  // upper-row x lower-column products (a b) and lower-row x upper-column products (c d)
  T ab00r = MG_CMUL_R(a0, b0), ab00i = MG_CMUL_I(a0, b0), ab11r = MG_CMUL_R(a1, b1), ab11i = MG_CMUL_I(a1, b1);
  T ab01r = MG_CMUL_R(a0, b1), ab01i = MG_CMUL_I(a0, b1), ab10r = MG_CMUL_R(a1, b0), ab10i = MG_CMUL_I(a1, b0);
  T cd00r = MG_CMUL_R(c0, d0), cd00i = MG_CMUL_I(c0, d0), cd11r = MG_CMUL_R(c1, d1), cd11i = MG_CMUL_I(c1, d1);
  T cd01r = MG_CMUL_R(c0, d1), cd01i = MG_CMUL_I(c0, d1), cd10r = MG_CMUL_R(c1, d0), cd10i = MG_CMUL_I(c1, d0);
  // B^0 = a.b + c.d ; B^3 = (a0b0 - a1b1) - (c0d0 - c1d1) ; B^1 = (a0b1 + a1b0) - (c0d1 + c1d0)
  // B^2 = -i (a0b1 - a1b0) + i (c0d1 - c1d0).   Stored with lowered index: B_0 = B^0, B_k = -B^k.
  B.r[0] = ab00r + ab11r + cd00r + cd11r;
  B.i[0] = ab00i + ab11i + cd00i + cd11i;
  B.r[3] = -(ab00r - ab11r) + (cd00r - cd11r);
  B.i[3] = -(ab00i - ab11i) + (cd00i - cd11i);
  B.r[1] = -(ab01r + ab10r) + (cd01r + cd10r);
  B.i[1] = -(ab01i + ab10i) + (cd01i + cd10i);
  // -B^2 = i (ab01 - ab10) - i (cd01 - cd10) = i * z, z = (ab01-ab10) - (cd01-cd10): re = -Im z, im = Re z
  T zr = (ab01r - ab10r) - (cd01r - cd10r), zi = (ab01i - ab10i) - (cd01i - cd10i);
  B.r[2] = -zi;
  B.i[2] = zr;
}
// quark pair -> off-shell gluon (quark channels, gen/quark.py):  j^mu = s * L gamma^mu R  (index raised), s = -1/P^2
template <class T> MG_DEV void cur_pair(const W4<T>& L, const W4<T>& R, T s, W4<T>& o) {
  W4<T> B;
  bilinear(L, R, B);
  o.r[0] = s * B.r[0];
  o.i[0] = s * B.i[0];
#pragma unroll
  for (int m = 1; m < 4; ++m) { o.r[m] = -s * B.r[m]; o.i[m] = -s * B.i[m]; }
}
// plain (already index-lowered) contraction  sum_mu B_mu j^mu
template <class T> MG_DEV C1<T> contract(const W4<T>& B, const W4<T>& j) {
  C1<T> d;
  d.r = B.r[0] * j.r[0] - B.i[0] * j.i[0];
  d.i = B.r[0] * j.i[0] + B.i[0] * j.r[0];
#pragma unroll
  for (int m = 1; m < 4; ++m) {
    d.r = d.r + B.r[m] * j.r[m] - B.i[m] * j.i[m];
    d.i = d.i + B.r[m] * j.i[m] + B.i[m] * j.r[m];
  }
  return d;
}

// Chiral halves of the bilinear (config 1, Z couplings):  BL_mu = L gamma_mu P_L R,  BR_mu = L gamma_mu P_R R
// (P_L = upper two components in the Weyl basis); index lowered as in bilinear().
template <class T> MG_DEV void bilinear_lr(const W4<T>& L, const W4<T>& R, W4<T>& BL, W4<T>& BR) {
  C1<T> a0 = {L.r[0], L.i[0]}, a1 = {L.r[1], L.i[1]}, c0 = {L.r[2], L.i[2]}, c1 = {L.r[3], L.i[3]};
  C1<T> d0 = {R.r[0], R.i[0]}, d1 = {R.r[1], R.i[1]}, b0 = {R.r[2], R.i[2]}, b1 = {R.r[3], R.i[3]};
  T ab00r = MG_CMUL_R(a0, b0), ab00i = MG_CMUL_I(a0, b0), ab11r = MG_CMUL_R(a1, b1), ab11i = MG_CMUL_I(a1, b1);
  T ab01r = MG_CMUL_R(a0, b1), ab01i = MG_CMUL_I(a0, b1), ab10r = MG_CMUL_R(a1, b0), ab10i = MG_CMUL_I(a1, b0);
  T cd00r = MG_CMUL_R(c0, d0), cd00i = MG_CMUL_I(c0, d0), cd11r = MG_CMUL_R(c1, d1), cd11i = MG_CMUL_I(c1, d1);
  T cd01r = MG_CMUL_R(c0, d1), cd01i = MG_CMUL_I(c0, d1), cd10r = MG_CMUL_R(c1, d0), cd10i = MG_CMUL_I(c1, d0);
  BR.r[0] = ab00r + ab11r;      BR.i[0] = ab00i + ab11i;
  BR.r[3] = -(ab00r - ab11r);   BR.i[3] = -(ab00i - ab11i);
  BR.r[1] = -(ab01r + ab10r);   BR.i[1] = -(ab01i + ab10i);
  BR.r[2] = -(ab01i - ab10i);   BR.i[2] = (ab01r - ab10r);
  BL.r[0] = cd00r + cd11r;      BL.i[0] = cd00i + cd11i;
  BL.r[3] = (cd00r - cd11r);    BL.i[3] = (cd00i - cd11i);
  BL.r[1] = (cd01r + cd10r);    BL.i[1] = (cd01i + cd10i);
  BL.r[2] = (cd01i - cd10i);    BL.i[2] = -(cd01r - cd10r);
}
// Minkowski product of two index-lowered complex vectors
template <class T> MG_DEV C1<T> mink(const W4<T>& a, const W4<T>& b) { return wdot(a, b); }

}  // namespace mgw
