/* oracle_internal.h — TEST INFRASTRUCTURE (see oracle.h).  Shared by the oracle's own .c files only. */
#ifndef ORACLE_INTERNAL_H
#define ORACLE_INTERNAL_H
#include "oracle.h"
#include <math.h>
#include <string.h>
#include <stdlib.h>

typedef struct { cplx c[4]; } vec4c;      /* complex Lorentz vector (contravariant) or spinor */
typedef struct { cplx m[4][4]; } mat4c;

extern const real oracle_metric[4];       /* diag(+,-,-,-)  (C1) */
void  oracle_gamma_mat(int mu, mat4c* g); /* chiral/HELAS representation (C1) */

static inline cplx mdot_cc(const vec4c* a, const vec4c* b) {   /* Minkowski product, NO conjugation */
  return a->c[0]*b->c[0] - a->c[1]*b->c[1] - a->c[2]*b->c[2] - a->c[3]*b->c[3];
}
static inline vec4c v_from_real(const real p[4]) { vec4c r; for (int i=0;i<4;++i) r.c[i]=p[i]; return r; }
static inline vec4c v_add(vec4c a, vec4c b) { vec4c r; for (int i=0;i<4;++i) r.c[i]=a.c[i]+b.c[i]; return r; }
static inline vec4c v_sub(vec4c a, vec4c b) { vec4c r; for (int i=0;i<4;++i) r.c[i]=a.c[i]-b.c[i]; return r; }
static inline vec4c v_scale(cplx s, vec4c a) { vec4c r; for (int i=0;i<4;++i) r.c[i]=s*a.c[i]; return r; }
static inline vec4c v_zero(void) { vec4c r; for (int i=0;i<4;++i) r.c[i]=0; return r; }

mat4c oracle_slash(const vec4c* a);                               /* gamma^mu a_mu */
mat4c m_add_scaled_identity(mat4c a, cplx s);                      /* a + s*1 */
vec4c row_times_mat(const vec4c* row, const mat4c* m);             /* (row spinor) . M */
vec4c mat_times_col(const mat4c* m, const vec4c* col);             /* M . (column spinor) */
cplx  row_times_col(const vec4c* row, const vec4c* col);

vec4c oracle_u(const real p[4], real m, int lambda);               /* u(p,lambda)   (C1) */
vec4c oracle_v(const real p[4], real m, int lambda);               /* v(p,lambda)   (C1) */
vec4c oracle_bar(const vec4c* psi);                                /* psi^dagger gamma^0 */
vec4c oracle_eps(const real k[4], int lambda);                     /* eps(k,lambda) (C1) */
vec4c oracle_conj(const vec4c* a);

/* V3^mu(p1,e1;p2,e2;p3) = (e1.e2)(p1-p2)^mu + e2^mu((p2-p3).e1) + e1^mu((p3-p1).e2)   (C4) */
vec4c oracle_V3(const vec4c* p1, const vec4c* e1, const vec4c* p2, const vec4c* e2, const vec4c* p3);

/* SU(3): Gell-Mann T^a = lambda^a/2, a = 0..7 (C4) */
void oracle_gellmann_T(cplx T[8][3][3]);
#endif
