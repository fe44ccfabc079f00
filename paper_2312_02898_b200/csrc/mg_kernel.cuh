// mg_kernel.cuh — pieces shared by every generated process kernel (not by the oracle).
//   * the AoSoA momentum layout of the C ABI (include/mg5b200.h):
//       mom[page][ipar][ievt_in_page][4] doubles, NEPP = 32 events per page, (E,px,py,pz);
//     a thread's 4-vector is 32 contiguous bytes (two 128-bit loads), a warp reads 1 KiB contiguous.
//   * helicity index convention: bit (npar-1-i) of h set <=> particle i has lambda = +1.
//   * mg_procdesc_t: what a generated translation unit registers with the C-ABI layer.
#pragma once
#ifdef __CUDACC__
#include <cuda_runtime.h>
#endif
#include <math.h>
#include "mg_wave.cuh"

constexpr int MGK_NEPP = 32;

template <class T, int NPAR>
MG_DEV void load_momentum(const double* __restrict__ mom, long long ievt, int ipar, mgw::P4<T>& p) {
  const long long page = ievt / MGK_NEPP;
  const int lane = (int)(ievt % MGK_NEPP);
  const double* src = mom + ((page * NPAR + ipar) * MGK_NEPP + lane) * 4;
#ifdef __CUDA_ARCH__
  const double2* q = reinterpret_cast<const double2*>(src);
  const double2 a = __ldg(q), b = __ldg(q + 1);
  p.c[0] = T(a.x); p.c[1] = T(a.y); p.c[2] = T(b.x); p.c[3] = T(b.y);
#else
  p.c[0] = T(src[0]); p.c[1] = T(src[1]); p.c[2] = T(src[2]); p.c[3] = T(src[3]);
#endif
}

// Ordered loads/stores of the per-event invariants buffer inv[item][event] (split kernel shape).  asm volatile:
// the compiler neither hoists these out of the helicity loop nor merges repeated loads, so helicity-independent
// operands are fetched (L1/L2) where they are used instead of living in registers or spill slots.
#if defined(__CUDA_ARCH__) && !defined(MG_LDV_PLAIN)
MG_DEV double ldv(const double* p) { double v; asm volatile("ld.global.ca.f64 %0, [%1];" : "=d"(v) : "l"(p)); return v; }
MG_DEV float ldv(const float* p) { float v; asm volatile("ld.global.ca.f32 %0, [%1];" : "=f"(v) : "l"(p)); return v; }
#else
template <class T> MG_DEV T ldv(const T* p) { return *p; }
#endif
// ordered shared-memory loads (invariants staged in shared memory by a diagram-group kernel's prologue)
#if defined(__CUDA_ARCH__)
MG_DEV double lds(const double* p) {
  double v; asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"((unsigned)__cvta_generic_to_shared(p))); return v;
}
MG_DEV float lds(const float* p) {
  float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"((unsigned)__cvta_generic_to_shared(p))); return v;
}
#else
template <class T> MG_DEV T lds(const T* p) { return *p; }
#endif
template <class T> MG_DEV mgw::P4<T> ldps(const T* p, int blk) {
  mgw::P4<T> o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.c[m] = lds(p + m * blk);
  return o;
}
template <class T> MG_DEV mgw::P4<T> ldp(const T* p, long long stride) {
  mgw::P4<T> o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.c[m] = ldv(p + m * stride);
  return o;
}
template <class T> MG_DEV void stp(T* p, long long stride, const mgw::P4<T>& v) {
#pragma unroll
  for (int m = 0; m < 4; ++m) p[m * stride] = v.c[m];
}

template <int NPAR> MG_DEV int hel_of(int h, int ipar) {
  return ((h >> (NPAR - 1 - ipar)) & 1) ? 1 : -1;
}

#ifdef __CUDACC__
typedef int (*mg_launch_fn)(int prec, const double* mom, void* me_out, long long nevt, const int* hel_list,
                             int nhel_run, void* perhel_out, const double* par, void* ws, size_t ws_bytes,
                             cudaStream_t st);
struct mg_procdesc_t {
  const char* proc;          // canonical process string
  int npar, ngluons, ndiagrams, nhel, ncol, denominator;
  long long flops_per_helicity;   // generator's static count (DFMA = 2)
  int massive[8];            // 1 where the particle has mass mt
  mg_launch_fn launch;
  int ws_bytes_per_event_hel[2];  // workspace bytes per (event, helicity) for fp64 / fp32 (0: fused kernel)
  int nkernels;              // kernel launches per event tile (diagram groups + colour + helicity sum)
  int has_fp32;              // fp32 kernels were generated
  int ws_bytes_per_event[2]; // workspace bytes per event (helicity-independent invariants) for fp64 / fp32
  long long flops_algorithmic;    // static count per helicity pass with every current computed once (no diagram-group
                                  // recomputation): the method's own FLOPs; flops_per_helicity is what the kernels execute
};
// mg_launch_fn returns the number of kernels it launched.
#endif  // __CUDACC__
