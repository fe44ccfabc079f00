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

template <class T> MG_DEV void stp(T* p, long long stride, const mgw::P4<T>& v) {
#pragma unroll
  for (int m = 0; m < 4; ++m) p[m * stride] = v.c[m];
}

template <int NPAR> MG_DEV int hel_of(int h, int ipar) {
  return ((h >> (NPAR - 1 - ipar)) & 1) ? 1 : -1;
}

#ifdef __CUDACC__
// fused shape (thread = event): loops over hel_list[0..nhel_run) and adds hel_w[ih] * |M_h|^2
typedef int (*mg_launch_fn)(int prec, const double* mom, void* me_out, long long nevt, const int* hel_list,
                             const double* hel_w, int nhel_run, void* perhel_out, const double* par, cudaStream_t st);
// event-CTA shape (thread = (event, helicity)): lane_w[tb * nlane + lane] = weight of that helicity (element type of the
// precision), ntb = number of top-quark helicities run (2: both; 1: only tb_first)
typedef int (*mg_launch_slots_fn)(int prec, const double* mom, void* me_out, long long nevt, const void* lane_w, int ntb,
                                  int tb_first, void* perhel_out, const double* par, void* ws, size_t ws_bytes,
                                  cudaStream_t st);
struct mg_procdesc_t {
  const char* proc;          // canonical process string
  int npar, ngluons, ndiagrams, nhel, ncol, denominator;
  long long flops_per_helicity;   // generator's static count of what the kernels execute per evaluated helicity (DFMA = 2)
  int massive[8];            // 1 where the particle has mass mt
  mg_launch_fn launch;             // fused shape, else nullptr
  mg_launch_slots_fn launch_slots; // event-CTA shape, else nullptr
  int reserved[2];
  int nkernels;              // kernel launches per event tile
  int has_fp32;              // fp32 kernels were generated
  int ws_bytes_per_event[2]; // workspace bytes per event of a tile (per-event invariants) for fp64 / fp32
  long long flops_algorithmic;    // static count per helicity with every current computed once (no diagram-group
                                  // recomputation): the method's own FLOPs
  long long flops_per_event;      // executed once per (event, top-quark helicity) slot, whatever the number of
                                  // helicities: the helicity tables (event-CTA shape)
  long long flops_algorithmic_per_event;   // same with every table built once per slot
  int ws_bytes_per_cta[2];   // JAMP scratch per resident CTA for fp64 / fp32
  int nlane;                 // event-CTA shape: helicity lanes per slot = 2^(npar-1)
  int ctas_per_sm;           // event-CTA shape: resident CTAs per SM the launcher uses at most (sizes the JAMP scratch)
};
// both launch functions return the number of kernels they launched (< 0: error).
#endif  // __CUDACC__
