/* weight.c — oracle of the batch-unweighting primitive (TEST INFRASTRUCTURE; see oracle.h).
 * PAPER.md:99-:103 (§3): "weights from Jacobian terms and PDFs are transferred to the GPU, and multiplied with the
 * matrix elements that are already in GPU memory ... The maximum of these weights is computed in parallel".
 * Plain definition: prod_i = fl(w_i * me_i) (one rounding, the precision of me), then max_i, sum_i, sum_i prod_i^2 of
 * the products, the sums accumulated in `real` (long double in the adjudication build) in index order. */
#include <math.h>
#include "oracle.h"

int oracle_weight_max(const double* me, const double* w, int64_t n, int single, double* prod_out, double* out3) {
  real mx = -INFINITY, su = 0, s2 = 0;
  for (int64_t i = 0; i < n; ++i) {
    double p = w[i] * me[i];
    if (single) p = (double)(float)p;
    if (prod_out) prod_out[i] = p;
    if ((real)p > mx) mx = (real)p;
    su += (real)p;
    s2 += (real)p * (real)p;
  }
  out3[0] = (double)mx; out3[1] = (double)su; out3[2] = (double)s2;
  return 0;
}
