/* philox_rambo.c — TEST INFRASTRUCTURE (see oracle.h).  The sampler half of the oracle.
 * Follows SURVEY.md §8(c) C6 step by step (the paper only names RAMBO and a "multi-event random
 * number generator", Fig. 1b).
 *   R1  Philox4x32-10, Salmon et al. SC'11, written out from the round definition.
 *   R2  RAMBO, Kleiss-Stirling-Ellis 1986, steps 1..6 in the order of C6.
 * Pins: tests/test_oracle_sampler.py (known-answer vectors; conservation, on-shellness,
 * closed-form massless weight, massive n=2 weight = (pi/2) beta, n=3 Dalitz mean).
 */
#include "oracle.h"
#include <math.h>
#include <stdlib.h>

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
    uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;   /* key schedule, applied before the next round */
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

static real factorial(int n) { real f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

int oracle_rambo(uint64_t seed, int64_t first_event, int64_t nevt, int nfinal,
                 const double* masses_final, double sqrt_s, double* momenta, double* weights) {
  const int n = nfinal, npar = nfinal + 2;
  real w = sqrt_s, summ = 0;
  int massive = 0;
  for (int i = 0; i < n; ++i) { summ += masses_final[i]; if (masses_final[i] != 0.0) massive = 1; }
  if (!(w > summ)) return -1;
  /* step 4: massless weight  W0 = (pi/2)^(n-1) w^(2n-4) / ((n-1)! (n-2)!)   (no (2pi)^(4-3n)) */
  real W0 = 1;
  for (int i = 0; i < n - 1; ++i) W0 *= R_PI / 2;
  for (int i = 0; i < 2 * n - 4; ++i) W0 *= w;
  W0 /= factorial(n - 1) * factorial(n - 2);

  for (int64_t ie = 0; ie < nevt; ++ie) {
    uint64_t ievt = (uint64_t)(first_event + ie);
    real q[8][4], p[8][4];
    /* step 1: isotropic massless q_i from 4 uniforms per final particle */
    for (int i = 0; i < n; ++i) {
      uint32_t ctr[4] = { (uint32_t)ievt, (uint32_t)(ievt >> 32), (uint32_t)i, 0u };
      uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
      uint32_t x[4];
      oracle_philox4x32_10(ctr, key, x);
      real u[4];
      for (int m = 0; m < 4; ++m) u[m] = ((real)x[m] + (real)0.5) / (real)4294967296.0;
      real c = 2 * u[0] - 1, s = R_SQRT(1 - c * c), phi = 2 * R_PI * u[1];
      real q0 = -R_LOG(u[2] * u[3]);
      q[i][0] = q0; q[i][1] = q0 * s * R_COS(phi); q[i][2] = q0 * s * R_SIN(phi); q[i][3] = q0 * c;
    }
    /* step 2 */
    real Q[4] = {0, 0, 0, 0};
    for (int i = 0; i < n; ++i) for (int m = 0; m < 4; ++m) Q[m] += q[i][m];
    real M = R_SQRT(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
    real b[3] = { -Q[1] / M, -Q[2] / M, -Q[3] / M };
    real x = w / M, gam = Q[0] / M, a = 1 / (1 + gam);
    /* step 3 */
    for (int i = 0; i < n; ++i) {
      real bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
      p[i][0] = x * (gam * q[i][0] + bq);
      for (int m = 0; m < 3; ++m) p[i][m + 1] = x * (q[i][m + 1] + b[m] * q[i][0] + a * bq * b[m]);
    }
    real W = W0;
    /* step 5: massive rescaling, Newton, fixed 6 iterations, no early exit */
    if (massive) {
      real xi = R_SQRT(1 - (summ / w) * (summ / w));
      for (int it = 0; it < 6; ++it) {
        real sumE = 0, der = 0;
        for (int i = 0; i < n; ++i) {
          real mi = masses_final[i];
          real Ei = R_SQRT(mi * mi + xi * xi * p[i][0] * p[i][0]);
          sumE += Ei; der += p[i][0] * p[i][0] / Ei;
        }
        xi = xi - (sumE - w) / (xi * der);
      }
      real prod = 1, sum2 = 0;
      for (int i = 0; i < n; ++i) {
        real mi = masses_final[i];
        real Ei = R_SQRT(mi * mi + xi * xi * p[i][0] * p[i][0]);
        real kabs = xi * p[i][0];               /* |k_i| = xi |p_i| = xi p_i^0 (massless p) */
        p[i][0] = Ei; p[i][1] *= xi; p[i][2] *= xi; p[i][3] *= xi;
        prod *= kabs / Ei; sum2 += kabs * kabs / Ei;
      }
      real xipow = 1;
      for (int i = 0; i < 2 * n - 3; ++i) xipow *= xi;
      W = W0 * xipow * prod / sum2 * w;
    }
    /* step 6: beams */
    double* out = momenta + (size_t)ie * npar * 4;
    out[0] = (double)(w / 2); out[1] = 0; out[2] = 0; out[3] = (double)(w / 2);
    out[4] = (double)(w / 2); out[5] = 0; out[6] = 0; out[7] = (double)(-w / 2);
    for (int i = 0; i < n; ++i) for (int m = 0; m < 4; ++m) out[8 + 4 * i + m] = (double)p[i][m];
    if (weights) weights[ie] = (double)W;
  }
  return 0;
}
