// mg_rambo.cu — K1 + K2 of SURVEY.md §8(a): device Philox4x32-10 and the RAMBO flat phase-space sampler
// (Fig. 1b "multi-event random number and phase-space generator"; "RAMBO ...
// ideal to quickly generate a batch of test events").  One thread = one event; the only HBM traffic is the
// AoSoA momentum write (32 B x npar per event, coalesced: a warp writes 1 KiB contiguous per particle), so
// this kernel is HBM-write-bound.  Always fp64.
//
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), stream mapping of DESIGN.md §3 (R1):
//   key = (seed_lo, seed_hi), counter = (ievt_lo, ievt_hi, ifinal, 0), u_m = (x_m + 0.5) 2^-32.
// RAMBO (Kleiss, Stirling, Ellis 1986), steps R2.1-R2.6 of DESIGN.md §3.
#include <cuda_runtime.h>
#include <stdint.h>
#include "mg_internal.h"

namespace {

constexpr int MAXF = 6;

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t out[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
    c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

__global__ void philox_raw_kernel(uint32_t k0, uint32_t k1, long long first_event, long long nevt, int nfinal,
                                  uint32_t* __restrict__ out) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nevt * nfinal) return;
  const unsigned long long gi = (unsigned long long)(first_event + t / nfinal);
  uint32_t x[4];
  philox4x32_10((uint32_t)gi, (uint32_t)(gi >> 32), (uint32_t)(t % nfinal), 0u, k0, k1, x);
  reinterpret_cast<uint4*>(out)[t] = make_uint4(x[0], x[1], x[2], x[3]);
}

struct RamboArgs {
  double masses[MAXF];
  double sqrt_s, w0;      // w0: massless weight constant
  uint32_t k0, k1;
  int nfinal, npar, any_massive;
  long long first_event, nevt;
};

template <int NF>
__global__ void __launch_bounds__(256) rambo_kernel(RamboArgs a, double* __restrict__ mom, double* __restrict__ wgt) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= a.nevt) return;
  const unsigned long long gi = (unsigned long long)(a.first_event + i);
  double q[NF][4];
  double Q0 = 0, Q1 = 0, Q2 = 0, Q3 = 0;
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    uint32_t x[4];
    philox4x32_10((uint32_t)gi, (uint32_t)(gi >> 32), (uint32_t)f, 0u, a.k0, a.k1, x);
    const double u1 = ((double)x[0] + 0.5) * 2.3283064365386963e-10;
    const double u2 = ((double)x[1] + 0.5) * 2.3283064365386963e-10;
    const double u3 = ((double)x[2] + 0.5) * 2.3283064365386963e-10;
    const double u4 = ((double)x[3] + 0.5) * 2.3283064365386963e-10;
    const double c = 2.0 * u1 - 1.0;
    const double s = sqrt(1.0 - c * c);
    const double phi = 6.283185307179586476925286766559 * u2;
    const double q0 = -log(u3 * u4);
    double sp, cp;
    sincos(phi, &sp, &cp);
    q[f][0] = q0; q[f][1] = q0 * s * cp; q[f][2] = q0 * s * sp; q[f][3] = q0 * c;
    Q0 += q[f][0]; Q1 += q[f][1]; Q2 += q[f][2]; Q3 += q[f][3];
  }
  const double M = sqrt(Q0 * Q0 - Q1 * Q1 - Q2 * Q2 - Q3 * Q3);
  const double b1 = -Q1 / M, b2 = -Q2 / M, b3 = -Q3 / M;
  const double x = a.sqrt_s / M, g = Q0 / M, aa = 1.0 / (1.0 + g);
  double p[NF][4];
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const double bq = b1 * q[f][1] + b2 * q[f][2] + b3 * q[f][3];
    p[f][0] = x * (g * q[f][0] + bq);
    p[f][1] = x * (q[f][1] + b1 * q[f][0] + aa * bq * b1);
    p[f][2] = x * (q[f][2] + b2 * q[f][0] + aa * bq * b2);
    p[f][3] = x * (q[f][3] + b3 * q[f][0] + aa * bq * b3);
  }
  double weight = a.w0;
  if (a.any_massive) {
    double sm = 0;
#pragma unroll
    for (int f = 0; f < NF; ++f) sm += a.masses[f];
    const double r = sm / a.sqrt_s;
    double xi = sqrt(1.0 - r * r);
#pragma unroll 1
    for (int it = 0; it < 6; ++it) {     // fixed 6 Newton iterations, no early exit
      double se = 0, sd = 0;
#pragma unroll
      for (int f = 0; f < NF; ++f) {
        const double e = sqrt(a.masses[f] * a.masses[f] + xi * xi * p[f][0] * p[f][0]);
        se += e;
        sd += p[f][0] * p[f][0] / e;
      }
      xi = xi - (se - a.sqrt_s) / (xi * sd);
    }
    double prod = 1.0, ssum = 0.0;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const double e = sqrt(a.masses[f] * a.masses[f] + xi * xi * p[f][0] * p[f][0]);
      p[f][0] = e; p[f][1] *= xi; p[f][2] *= xi; p[f][3] *= xi;
      const double k2 = p[f][1] * p[f][1] + p[f][2] * p[f][2] + p[f][3] * p[f][3];
      prod *= sqrt(k2) / e;
      ssum += k2 / e;
    }
    weight = a.w0 * pow(xi, (double)(2 * NF - 3)) * prod / ssum * a.sqrt_s;
  }
  if (wgt) wgt[i] = weight;
  // AoSoA write: mom[page][ipar][lane][4]
  const long long page = i / MG_NEPP_I;
  const int lane = (int)(i % MG_NEPP_I);
  double2* base = reinterpret_cast<double2*>(mom + (page * a.npar * MG_NEPP_I + lane) * 4);
  const int stride = MG_NEPP_I * 2;   // double2 units per particle
  const double h = 0.5 * a.sqrt_s;
  base[0] = make_double2(h, 0.0);           base[1] = make_double2(0.0, h);
  base[stride] = make_double2(h, 0.0);      base[stride + 1] = make_double2(0.0, -h);
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    base[(2 + f) * stride] = make_double2(p[f][0], p[f][1]);
    base[(2 + f) * stride + 1] = make_double2(p[f][2], p[f][3]);
  }
}

}  // namespace

cudaError_t mg_launch_rambo(int nfinal, const double* masses, double sqrt_s, uint64_t seed, long long first_event,
                            long long nevt, double* mom, double* wgt, cudaStream_t st) {
  RamboArgs a;
  a.nfinal = nfinal; a.npar = nfinal + 2; a.sqrt_s = sqrt_s;
  a.k0 = (uint32_t)seed; a.k1 = (uint32_t)(seed >> 32);
  a.first_event = first_event; a.nevt = nevt;
  a.any_massive = 0;
  for (int f = 0; f < MAXF; ++f) { a.masses[f] = f < nfinal ? masses[f] : 0.0; if (a.masses[f] != 0.0) a.any_massive = 1; }
  // W0 = (pi/2)^(n-1) w^(2n-4) / ((n-1)! (n-2)!)
  double w0 = 1.0, f1 = 1.0, f2 = 1.0;
  for (int k = 1; k <= nfinal - 1; ++k) { w0 *= 1.5707963267948966; f1 *= k; }
  for (int k = 1; k <= nfinal - 2; ++k) f2 *= k;
  for (int k = 0; k < 2 * nfinal - 4; ++k) w0 *= sqrt_s;
  a.w0 = w0 / (f1 * f2);
  if (nevt <= 0) return cudaSuccess;
  const int block = 256;
  const unsigned grid = (unsigned)((nevt + block - 1) / block);
  switch (nfinal) {
    case 2: rambo_kernel<2><<<grid, block, 0, st>>>(a, mom, wgt); break;
    case 3: rambo_kernel<3><<<grid, block, 0, st>>>(a, mom, wgt); break;
    case 4: rambo_kernel<4><<<grid, block, 0, st>>>(a, mom, wgt); break;
    case 5: rambo_kernel<5><<<grid, block, 0, st>>>(a, mom, wgt); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t mg_launch_philox_raw(uint64_t seed, long long first_event, long long nevt, int nfinal, uint32_t* out,
                                 cudaStream_t st) {
  const long long n = nevt * nfinal;
  if (n <= 0) return cudaSuccess;
  philox_raw_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>((uint32_t)seed, (uint32_t)(seed >> 32), first_event, nevt,
                                                                 nfinal, out);
  return cudaGetLastError();
}
