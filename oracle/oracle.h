/* oracle.h — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, scalar CPU oracle for the hot path of arXiv:2312.02898 ("Madgraph5_aMC@NLO on
 * GPUs and vector CPUs"): RAMBO batch -> per-event tree-level |M|^2 summed over helicities and
 * colours ("compute probability amplitudes ('matrix elements') for a given
 * collision"; PAPER.md:47 RAMBO; PAPER.md:139 process list e+e- -> mu+mu-, gg -> tt~ + 0..3 g;
 * PAPER.md:141 leading order, fixed couplings).  The paper prints no formulas; every formula
 * here is a reading listed in SURVEY.md §8(c) C1..C7 and restated in DESIGN.md §3.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code, table or constant generator with the CUDA path
 * (paper_2312_02898_b200/): different algorithm (colour-ordered Berends-Giele recursion plus
 * explicit Gell-Mann colour sums, instead of Feynman diagrams + colour-flow JAMPs).
 *
 * Build twice: -DORACLE_LONG_DOUBLE (adjudication, x87 80-bit) and default double (timing).
 * Parity pins: tests/test_oracle_*.py (closed forms, invariants, brute force).  Functions with
 * no independent pin say "parity unpinned" below (none at present for fp64).
 */
#ifndef ORACLE_H
#define ORACLE_H
#include <stdint.h>
#include <complex.h>

#ifdef ORACLE_LONG_DOUBLE
typedef long double real;
typedef long double _Complex cplx;
#define R_SQRT sqrtl
#define R_FABS fabsl
#define R_LOG  logl
#define R_SIN  sinl
#define R_COS  cosl
#define R_CREAL creall
#define R_CIMAG cimagl
#define R_PI 3.14159265358979323846264338327950288L
#else
typedef double real;
typedef double _Complex cplx;
#define R_SQRT sqrt
#define R_FABS fabs
#define R_LOG  log
#define R_SIN  sin
#define R_COS  cos
#define R_CREAL creal
#define R_CIMAG cimag
#define R_PI 3.14159265358979323846264338327950288
#endif

/* physics parameters.  Plain doubles on the interface. */
typedef struct {
  double alpha_s;      /* 0.118 */
  double alpha_ew_inv; /* 132.507 */
  double sw2;          /* sin^2(theta_W); A1 reading 0.22224649... derived by caller */
  double mz, gamma_z;  /* 91.188, 2.4414 */
  double mt;           /* 173.0 ; Gamma_t = 0 (A2) */
} oracle_params_t;

/* ---- C6 R1: Philox4x32-10 ---- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* ---- C6 R2: RAMBO.  momenta layout [nevt][2+nfinal][4] (E,px,py,pz), weights [nevt] or NULL.
 * returns 0, or -1 if sqrt_s <= sum(masses). */
int oracle_rambo(uint64_t seed, int64_t first_event, int64_t nevt, int nfinal,
                 const double* masses_final, double sqrt_s, double* momenta, double* weights);

/* ---- C1: external wavefunctions (exposed for the Dirac/completeness pins) ---- */
void oracle_spinor_u(const double p[4], double m, int lambda, double out_re_im[8]);
void oracle_spinor_v(const double p[4], double m, int lambda, double out_re_im[8]);
void oracle_polvec  (const double k[4], int lambda, double out_re_im[8]);
void oracle_gamma   (int mu, double out_re_im[32]);          /* 4x4 row-major */

/* ---- C4: colour matrix from explicit Gell-Mann matrices; CF is n! x n! row-major,
 * permutations in lexicographic order.  brute != 0: definition over every (sigma,sigma') pair
 * (n <= 4 in practice); brute == 0: same sum streamed as a Gram matrix over adjoint tuples. */
int oracle_colour_matrix(int n, double* CF, int brute);

/* ---- matrix elements.  p: [npar][4] physical momenta, process order.  Returns the
 * spin/colour-averaged, identical-particle-divided |M|^2 (A3).  hel_out: NULL or [nhel]
 * per-helicity colour-summed |M_h|^2 / denominator (helicity index: bit (npar-1-i) of h set
 * <=> particle i has lambda=+1). ---- */
double oracle_me_eemumu(const double* p, const oracle_params_t* par, double* hel_out);        /* C3 */
double oracle_me_ggttng(int nfinal_gluons, const double* p, const oracle_params_t* par,
                        double* hel_out);                                                       /* C4 */
/* C5: independent colour-dressed route (explicit f^{abc}, explicit colour sums).  n_gluons<=4 */
double oracle_me_ggttng_dressed(int nfinal_gluons, const double* p, const oracle_params_t* par);
/* C5: gg -> tt~, three diagrams written out by hand with CF = 1/3 [[16,-2],[-2,16]] */
double oracle_me_ggtt_explicit(const double* p, const oracle_params_t* par);
/* Ward-identity probe (C8 pin ii): same as C4 but external gluon `which` (0-based among gluons,
 * process order: 2 beam gluons then final ones) has its polarisation replaced by its momentum. */
double oracle_me_ggttng_ward(int nfinal_gluons, const double* p, const oracle_params_t* par, int which);

/* ---- quark channels of p p -> t t~ + jets: top line + one massless quark line of another
 * flavour + up to 2 gluons, any crossing.  spec: one character per particle in process order ('q' quark, 'Q' antiquark,
 * 'g' gluon, "tT" at positions 2-3), e.g. "qQtT", "qQtTg", "qgtTq", "gQtTQ", "qQtTgg", "qgtTqg", "ggtTqQ".
 * Colour-dressed Feynman rules with explicit colour sums (me_qchannel.c).  ward_which >= 0: gluon number ward_which
 * (in process order among the gluons) has its polarisation replaced by its momentum; -1: physical. ---- */
double oracle_me_qchannel(const char* spec, const double* p, const oracle_params_t* par, double* hel_out, int ward_which);
double oracle_me_qchannel_pauli(const char* spec, const double* p, const oracle_params_t* par);   /* see me_qchannel.c */
int oracle_me_qchannel_batch(const char* spec, const double* momenta, int64_t nevt, const oracle_params_t* par,
                             double* me_out, int nthreads);

/* batch drivers (OpenMP over events) for parity and the cpu_baseline timing.
 * proc: 0 = e+e- -> mu+mu-, 1..4 = gg -> tt~ + (proc-1) g.  momenta [nevt][npar][4]. */
int oracle_me_batch(int proc, const double* momenta, int64_t nevt, const oracle_params_t* par,
                    double* me_out, int nthreads);
int oracle_num_threads(void);

/* ---- batch-unweighting primitive (PAPER.md:99-:103): prod_i = w_i * me_i rounded once to double (single != 0: to
 * float), out3 = (max_i, sum_i, sum_i prod_i^2) of the products; prod_out may be NULL.  Pinned by closed forms
 * (arithmetic series) and by the exactness of the maximum (tests/test_oracle_weight.py). ---- */
int oracle_weight_max(const double* me, const double* w, int64_t n, int single, double* prod_out, double* out3);
#endif
