// mg_noalloc.cu — mg_weight_max_noalloc: the batch-unweighting primitive (PAPER.md:99-:103; mg_weight_max, mg_reduce.cu)
// for callers that cannot allocate device memory: code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  mg_weight_max needs a handle (mg_process_create allocates) whose partial-result buffer came from cudaMalloc;
// this variant needs neither: the first reduction stage's partials live in a file-scope __device__ array of fixed size.
//
//   * Limit: MG_NOALLOC_MAX_EVENTS = 1024 blocks x 8192 events = 8 388 608 events per call (16x the largest batch of
//     BASELINE.json); larger batches are rejected with MG_ERR_TOO_LARGE.  The array is 24 KiB; every GPU on which the
//     library is loaded holds it until the process exits.
//   * The array's name is a host-side stand-in in host code, not a device address: its address is taken once per device
//     with cudaGetSymbolAddress (that device current) and handed to the kernels.
//   * No cudaMalloc / cudaFree / allocating library call anywhere on this path.
//   * Every call on a device shares the array.  It keeps the last call's contents; nothing in it has to start at zero:
//     stage 1 overwrites the partials [0, nblocks) of this call before stage 2 (same stream) reads exactly those.  Calls
//     that overlap on the GPU (different streams, or graphs replayed concurrently) race on it: the caller serialises them.
//   * Same reduction shape as mg_weight_max (8192-element chunks rounded up to whole 256-thread sweeps, fixed tree inside
//     a block, one final block adding the partials in index order), so both give bit-identical results.
#include <atomic>
#include <math.h>
#include <stdio.h>

#include "../../include/mg5b200.h"
#include "mg_internal.h"

constexpr int NA_MAX_BLOCKS = 1024;                   // partial slots
constexpr long long NA_CHUNK = 8192;                  // events per block at most
static_assert((long long)NA_MAX_BLOCKS * NA_CHUNK == MG_NOALLOC_MAX_EVENTS, "header and scratch size disagree");

// the scratch: [block][max, sum, sum of squares]; 24 KiB on every GPU that loads the library
static __device__ __align__(256) double na_partials[3 * NA_MAX_BLOCKS];

namespace {

constexpr int RB = 256;                               // threads per block

// stage 1: block b handles elements [b * chunk, (b + 1) * chunk): product in place, block-level (max, sum, sum sq)
template <class T>
__global__ void __launch_bounds__(RB) na_weight_stage1(T* __restrict__ me, const double* __restrict__ w, long long n, long long chunk,
                                                       double* __restrict__ part) {
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
__global__ void __launch_bounds__(RB) na_weight_stage2(const double* __restrict__ part, int nblocks, double* __restrict__ out) {
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

constexpr int NA_MAX_DEVICES = 64;
std::atomic<double*> na_addr[NA_MAX_DEVICES];         // device address of na_partials, per device ordinal (nullptr: not set up)

int na_fail(int status, const char* what) {
  mg_set_last_error(what);
  return status;
}

// Set-up, once per device, with that device current: the DEVICE address of the scratch array.
int na_scratch(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cudaGetLastError(); return na_fail(MG_ERR_NO_DEVICE, "mg_weight_max_noalloc: no current CUDA device"); }
  if (dev < 0 || dev >= NA_MAX_DEVICES) return na_fail(MG_ERR_NO_DEVICE, "mg_weight_max_noalloc: device ordinal beyond 63");
  double* p = na_addr[dev].load(std::memory_order_acquire);
  if (!p) {
    e = cudaGetSymbolAddress((void**)&p, na_partials);
    if (e != cudaSuccess || !p) {
      char msg[256];
      snprintf(msg, sizeof msg, "mg_weight_max_noalloc: cudaGetSymbolAddress(na_partials): %s", cudaGetErrorString(e));
      cudaGetLastError();
      return na_fail(MG_ERR_CUDA, msg);
    }
    na_addr[dev].store(p, std::memory_order_release);     // a second thread racing here stores the same address
  }
  *out = p;
  return MG_OK;
}

}  // namespace

extern "C" int mg_weight_max_noalloc(int precision, void* me_dev, const double* weights_dev, int64_t nevt, double* out_dev,
                                     void* stream) {
  if (!out_dev || ((!me_dev || !weights_dev) && nevt > 0)) return MG_ERR_NULL;
  if (precision != MG_FP64 && precision != MG_FP32) return MG_ERR_BAD_PARAM;
  if (nevt < 0) return MG_ERR_BAD_NEVT;
  if (nevt > MG_NOALLOC_MAX_EVENTS) {
    char msg[256];
    snprintf(msg, sizeof msg, "mg_weight_max_noalloc: nevt = %lld exceeds MG_NOALLOC_MAX_EVENTS = %lld (fixed scratch); "
                              "split the batch or use mg_weight_max", (long long)nevt, (long long)MG_NOALLOC_MAX_EVENTS);
    return na_fail(MG_ERR_TOO_LARGE, msg);
  }
  const uintptr_t emask = precision == MG_FP64 ? 7 : 3;
  if (((uintptr_t)me_dev & emask) || ((uintptr_t)weights_dev & 7) || ((uintptr_t)out_dev & 7)) return MG_ERR_ALIGN;
  double* part = nullptr;
  const int rc = na_scratch(&part);
  if (rc != MG_OK) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  long long nb = (nevt + NA_CHUNK - 1) / NA_CHUNK;      // as mg_weight_blocks (mg_reduce.cu) below its cap
  if (nb < 1) nb = 1;
  const long long chunk = ((nevt + nb - 1) / nb + RB - 1) / RB * RB;
  if (precision == MG_FP64) na_weight_stage1<double><<<(unsigned)nb, RB, 0, st>>>((double*)me_dev, weights_dev, nevt, chunk, part);
  else na_weight_stage1<float><<<(unsigned)nb, RB, 0, st>>>((float*)me_dev, weights_dev, nevt, chunk, part);
  na_weight_stage2<<<1, RB, 0, st>>>(part, (int)nb, out_dev);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    char msg[256];
    snprintf(msg, sizeof msg, "mg_weight_max_noalloc launch: %s", cudaGetErrorString(e));
    return na_fail(MG_ERR_CUDA, msg);
  }
  return MG_OK;
}
