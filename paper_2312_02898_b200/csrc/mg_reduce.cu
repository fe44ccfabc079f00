// mg_reduce.cu — the two small device reductions next to the matrix-element kernels:
//   * helicity-probe statistics (K8): per helicity h, sum over the probe events of |M_h|^2 and of
//     | |M_h|^2 - |M_hbar|^2 | with hbar = all helicities flipped (decides the good-helicity list and whether the
//     helicity-flip symmetry may be used; mg_api.cu);
//   * the batch-unweighting primitive of PAPER.md:99-:103 (§3: "weights from Jacobian terms and PDFs are transferred
//     to the GPU, and multiplied with the matrix elements that are already in GPU memory ... The maximum of these
//     weights is computed in parallel"): me[i] <- w[i] * me[i] in place, plus max, sum and sum of squares of the
//     products.  HBM-bound: 8 B weight + 8 B |M|^2 read + 8 B written per event (fp64).
// Both reductions have a fixed shape (fixed chunk per block, fixed tree inside a block, one final block that adds the
// partials in index order), so results are bit-reproducible.
#include "mg_internal.h"

namespace {

constexpr int RB = 256;   // threads per block of every reduction here

template <class T>
__global__ void __launch_bounds__(RB) probe_stats_kernel(const T* __restrict__ perhel, long long nevt, int nhel,
                                                         double* __restrict__ out /* [2][nhel] */) {
  __shared__ double s0[RB], s1[RB];
  const int h = blockIdx.x, hb = nhel - 1 - h;
  double a = 0.0, d = 0.0;
  for (long long i = threadIdx.x; i < nevt; i += RB) {
    const double x = (double)perhel[(long long)h * nevt + i], y = (double)perhel[(long long)hb * nevt + i];
    a += x;
    d += fabs(x - y);
  }
  s0[threadIdx.x] = a; s1[threadIdx.x] = d;
  __syncthreads();
  for (int off = RB / 2; off > 0; off >>= 1) {
    if (threadIdx.x < off) { s0[threadIdx.x] += s0[threadIdx.x + off]; s1[threadIdx.x] += s1[threadIdx.x + off]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[h] = s0[0]; out[nhel + h] = s1[0]; }
}

// stage 1: block b handles elements [b * chunk, (b + 1) * chunk): product in place, block-level (max, sum, sum sq)
template <class T>
__global__ void __launch_bounds__(RB) weight_stage1(T* __restrict__ me, const double* __restrict__ w, long long n, long long chunk,
                                                    double* __restrict__ part /* [nblocks][3] */) {
  __shared__ double sm[RB], ss[RB], sq[RB];
  const long long b0 = (long long)blockIdx.x * chunk, b1 = b0 + chunk < n ? b0 + chunk : n;
  double mx = -INFINITY, su = 0.0, s2 = 0.0;
  for (long long i = b0 + threadIdx.x; i < b1; i += RB) {
    const T p = (T)(w[i] * (double)me[i]);
    me[i] = p;
    const double v = (double)p;
    mx = v > mx ? v : mx;
    su += v;
    s2 += v * v;
  }
  sm[threadIdx.x] = mx; ss[threadIdx.x] = su; sq[threadIdx.x] = s2;
  __syncthreads();
  for (int off = RB / 2; off > 0; off >>= 1) {
    if (threadIdx.x < off) {
      const double o = sm[threadIdx.x + off];
      if (o > sm[threadIdx.x]) sm[threadIdx.x] = o;
      ss[threadIdx.x] += ss[threadIdx.x + off];
      sq[threadIdx.x] += sq[threadIdx.x + off];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { part[3 * blockIdx.x] = sm[0]; part[3 * blockIdx.x + 1] = ss[0]; part[3 * blockIdx.x + 2] = sq[0]; }
}

// stage 2: one block; thread t adds partials t, t + RB, ... in index order, then the fixed tree
__global__ void __launch_bounds__(RB) weight_stage2(const double* __restrict__ part, int nblocks, double* __restrict__ out /* [3] */) {
  __shared__ double sm[RB], ss[RB], sq[RB];
  double mx = -INFINITY, su = 0.0, s2 = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += RB) {
    const double o = part[3 * b];
    mx = o > mx ? o : mx;
    su += part[3 * b + 1];
    s2 += part[3 * b + 2];
  }
  sm[threadIdx.x] = mx; ss[threadIdx.x] = su; sq[threadIdx.x] = s2;
  __syncthreads();
  for (int off = RB / 2; off > 0; off >>= 1) {
    if (threadIdx.x < off) {
      const double o = sm[threadIdx.x + off];
      if (o > sm[threadIdx.x]) sm[threadIdx.x] = o;
      ss[threadIdx.x] += ss[threadIdx.x + off];
      sq[threadIdx.x] += sq[threadIdx.x + off];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = sm[0]; out[1] = ss[0]; out[2] = sq[0]; }
}

}  // namespace

cudaError_t mg_launch_probe_stats(int prec, const void* perhel, long long nevt, int nhel, double* out, cudaStream_t st) {
  if (prec == 0) probe_stats_kernel<double><<<nhel, RB, 0, st>>>((const double*)perhel, nevt, nhel, out);
  else probe_stats_kernel<float><<<nhel, RB, 0, st>>>((const float*)perhel, nevt, nhel, out);
  return cudaGetLastError();
}

int mg_weight_blocks(long long n) {
  // 8192 elements per block (32 per thread): 64 blocks per 2^19 events; at most MG_WEIGHT_MAX_BLOCKS partials
  long long nb = (n + 8191) / 8192;
  if (nb < 1) nb = 1;
  if (nb > MG_WEIGHT_MAX_BLOCKS) nb = MG_WEIGHT_MAX_BLOCKS;
  return (int)nb;
}

cudaError_t mg_launch_weight_max(int prec, void* me, const double* w, long long n, double* part, double* out, cudaStream_t st) {
  const int nb = mg_weight_blocks(n);
  const long long chunk = ((n + nb - 1) / nb + RB - 1) / RB * RB;
  if (prec == 0) weight_stage1<double><<<nb, RB, 0, st>>>((double*)me, w, n, chunk, part);
  else weight_stage1<float><<<nb, RB, 0, st>>>((float*)me, w, n, chunk, part);
  weight_stage2<<<1, RB, 0, st>>>(part, nb, out);
  return cudaGetLastError();
}

// ---- mixed precision with precision tracking ("tracking the precision of the matrix
// elements showed that single-precision computations are not accurate enough") ----
// The fp32 kernels evaluate every helicity h and its helicity-flipped mirror hbar; in exact arithmetic |M_h|^2 =
// |M_hbar|^2 (A13), so  eps = sum_{h < hbar} | |M_h|^2 - |M_hbar|^2 | / sum_h |M_h|^2  is a per-event
// measurement of the fp32 arithmetic error of that event.  It does not see the rounding of the inputs both mirrors share
// (the helicity-independent operands are rounded to fp32 once), whose effect grows with the event's conditioning, so the
// tracker adds  kappa 2^-24 s / (2 min_ij |p_i.p_j|)  over pairs of massless legs (kappa = 1/4, calibrated on the full
// batches of configs 3-4: DESIGN.md §7).  Events with eps > tol (or a non-finite value) are flagged for re-evaluation
// in fp64.
namespace {
__global__ void __launch_bounds__(RB) mixed_flag_kernel(const float* __restrict__ perhel, const double* __restrict__ mom,
                                                        long long nevt, int nhel, int npar, unsigned massless_mask, double kappa,
                                                        double tol, double* __restrict__ me_out, float* __restrict__ eps_out,
                                                        int* __restrict__ flagged, int* __restrict__ nflagged) {
  const long long i = (long long)blockIdx.x * RB + threadIdx.x;
  if (i >= nevt) return;
  double s = 0.0, a = 0.0;
  for (int h = 0; h < nhel / 2; ++h) {
    const double x = (double)perhel[(long long)h * nevt + i], y = (double)perhel[(long long)(nhel - 1 - h) * nevt + i];
    s += x + y;
    a += fabs(x - y);
  }
  double eps = a / s;
  if (kappa > 0.0) {
    const double* pm = mom + ((i / 32) * npar * 32 + (i % 32)) * 4;      // particle ip at pm + ip * 128
    double dmin = INFINITY;
    for (int ia = 0; ia < npar; ++ia) {
      if (!((massless_mask >> ia) & 1)) continue;
      const double* pa = pm + ia * 128;
      for (int ib = ia + 1; ib < npar; ++ib) {
        if (!((massless_mask >> ib) & 1)) continue;
        const double* pb = pm + ib * 128;
        const double d = fabs(pa[0] * pb[0] - pa[1] * pb[1] - pa[2] * pb[2] - pa[3] * pb[3]);
        dmin = d < dmin ? d : dmin;
      }
    }
    const double shat = 2.0 * fabs(pm[0] * pm[128] - pm[1] * pm[129] - pm[2] * pm[130] - pm[3] * pm[131]);   // massless beams
    eps += kappa * 5.9604644775390625e-08 * shat / (2.0 * dmin);
  }
  me_out[i] = s;
  if (eps_out) eps_out[i] = (float)eps;
  if (!(eps <= tol) || !(s > 0.0) || isinf(s)) flagged[atomicAdd(nflagged, 1)] = (int)i;
}
// flagged events' momenta -> compact AoSoA pages (32 events per page, [page][ipar][32][4])
__global__ void __launch_bounds__(RB) mixed_gather_kernel(const double* __restrict__ mom, const int* __restrict__ flagged, int n,
                                                          int npar, double* __restrict__ out) {
  const int k = blockIdx.x * RB + threadIdx.x;
  const int npad = (n + 31) / 32 * 32;
  if (k >= npad) return;
  const long long i = flagged[k < n ? k : n - 1];            // pad the last page with copies of the last event
  for (int ip = 0; ip < npar; ++ip) {
    const double* src = mom + (((i / 32) * npar + ip) * 32 + (i % 32)) * 4;
    double* dst = out + ((((long long)k / 32) * npar + ip) * 32 + (k % 32)) * 4;
    dst[0] = src[0]; dst[1] = src[1]; dst[2] = src[2]; dst[3] = src[3];
  }
}
__global__ void __launch_bounds__(RB) mixed_scatter_kernel(const double* __restrict__ me64, const int* __restrict__ flagged, int n,
                                                           double* __restrict__ me_out) {
  const int k = blockIdx.x * RB + threadIdx.x;
  if (k < n) me_out[flagged[k]] = me64[k];
}
}  // namespace

cudaError_t mg_launch_mixed_flag(const float* perhel, const double* mom, long long nevt, int nhel, int npar, unsigned massless_mask,
                                 double kappa, double tol, double* me_out, float* eps_out, int* flagged, int* nflagged,
                                 cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(nflagged, 0, sizeof(int), st);
  if (e != cudaSuccess) return e;
  mixed_flag_kernel<<<(unsigned)((nevt + RB - 1) / RB), RB, 0, st>>>(perhel, mom, nevt, nhel, npar, massless_mask, kappa, tol, me_out,
                                                                    eps_out, flagged, nflagged);
  return cudaGetLastError();
}
cudaError_t mg_launch_mixed_gather(const double* mom, const int* flagged, int n, int npar, double* out, cudaStream_t st) {
  const int npad = (n + 31) / 32 * 32;
  mixed_gather_kernel<<<(unsigned)((npad + RB - 1) / RB), RB, 0, st>>>(mom, flagged, n, npar, out);
  return cudaGetLastError();
}
cudaError_t mg_launch_mixed_scatter(const double* me64, const int* flagged, int n, double* me_out, cudaStream_t st) {
  mixed_scatter_kernel<<<(unsigned)((n + RB - 1) / RB), RB, 0, st>>>(me64, flagged, n, me_out);
  return cudaGetLastError();
}
