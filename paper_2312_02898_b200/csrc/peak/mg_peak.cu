// mg_peak.cu — measurement helper, NOT part of the product library: builds into libmg5b200_peak.so, which only
// bench.py loads.  FMA-rate micro-benchmarks for the denominator of "% of FP64 (FP32) peak" ("DFMA
// micro-benchmark peak measured on the same box in the same run"): 16 independent FMA chains per thread, 512 threads x
// 4 CTAs per SM, no memory traffic in the loop; and the same for mma.sync.m8n8k4.f64 (DMMA.8x8x4).
#include <cuda_runtime.h>

namespace {
template <class T>
__global__ void __launch_bounds__(512) fma_peak_kernel(T* out, int iters, T a, T b) {
  T x[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) x[k] = T(threadIdx.x + k) * T(1e-3);
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int k = 0; k < 16; ++k) x[k] = x[k] * a + b;
    }
  }
  T s = T(0);
#pragma unroll
  for (int k = 0; k < 16; ++k) s += x[k];
  if (s == T(-1.2345)) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true; keeps the chain alive
}

template <class T> cudaError_t run(double* flops_per_s) {
  int dev = 0, nsm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  const int block = 512, grid = nsm * 4 * 4;
  const int iters = sizeof(T) == 8 ? 2000 : 8000;
  T* out = nullptr;
  cudaError_t e = cudaMalloc(&out, sizeof(T) * (size_t)block * grid);
  if (e != cudaSuccess) return e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    fma_peak_kernel<T><<<grid, block>>>(out, iters, T(0.999999), T(1e-7));
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * 16 * 8 * (double)iters * block * (double)grid;
    if (rep >= 1 && fl / (ms * 1e-3) > best) best = fl / (ms * 1e-3);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out);
  *flops_per_s = best;
  return e != cudaSuccess ? e : cudaGetLastError();
}
}  // namespace

namespace {
// FP64 tensor-core rate: mma.sync.m8n8k4.f64 (DMMA.8x8x4), 8 independent accumulator pairs per warp
__global__ void __launch_bounds__(256) dmma_peak_kernel(double* out, int iters, double a, double b) {
  double c0[8], c1[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) { c0[k] = threadIdx.x * 1e-3 + k; c1[k] = -c0[k]; }
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 4; ++r) {
#pragma unroll
      for (int k = 0; k < 8; ++k)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(c0[k]), "+d"(c1[k]) : "d"(a), "d"(b));
    }
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += c0[k] + c1[k];
  if (s == -1.2345) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace

static cudaError_t run_dmma(double* flops_per_s) {
  int dev = 0, nsm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  const int block = 256, grid = nsm * 8, iters = 2000;
  double* out = nullptr;
  cudaError_t e = cudaMalloc(&out, sizeof(double) * (size_t)block * grid);
  if (e != cudaSuccess) return e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0);
    dmma_peak_kernel<<<grid, block>>>(out, iters, 1e-3, 1e-3);
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fl = 2.0 * 8 * 8 * 4 * 8 * 4 * (double)iters * (block / 32) * (double)grid;   // 512 flop per mma per warp
    if (rep >= 1 && fl / (ms * 1e-3) > best) best = fl / (ms * 1e-3);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out);
  *flops_per_s = best;
  return e != cudaSuccess ? e : cudaGetLastError();
}

// C entry points (ctypes): return 0 and the rate in FLOP/s, or a cudaError_t code.
extern "C" int mgpeak_fma(int device, int prec, double* flops_per_s) {
  if (cudaSetDevice(device) != cudaSuccess) return (int)cudaGetLastError();
  return (int)(prec == 0 ? run<double>(flops_per_s) : run<float>(flops_per_s));
}
extern "C" int mgpeak_dmma(int device, double* flops_per_s) {
  if (cudaSetDevice(device) != cudaSuccess) return (int)cudaGetLastError();
  return (int)run_dmma(flops_per_s);
}
