// mg_colour.cuh — K6 (colour sum) and K7 (helicity sum + averaging) for the split kernel shape
// (north_star (4)).  Input: the JAMP workspace written by the diagram-group kernels,
//     jamp[ih][flow][re/im][stride]   (element type T, event index fastest => coalesced),
// output: me_out[evt] = norm * sum_ih  J^dagger CF J,  and optionally the per-helicity values.
//
// Register-blocked symmetric quadratic form: thread = one (event, helicity); for each block of 8 rows i the
// thread keeps 8 complex partial sums z_i = CF_ii J_i + 2 sum_{j>i} CF_ij J_j in registers while J_j streams
// in from L1/L2 (each J_j is re-read once per row block: ncol/16 times on average), then adds
// Re(J_i^* z_i).  The coefficients come from a blocked upper-triangular table
//     cf_table[block b][j >= 8b][8 rows]   (integers; the common denominator is folded into `norm`),
// read with warp-uniform loads.  Half the FLOPs of the full matrix-vector product.
#pragma once
#include <cuda_runtime.h>

// Colour-table access: `tab` is an offset into the blocked table.  If the including unit defines MG_CF_CONST (the
// name of a __constant__ copy of the table, <= 64 KB) the coefficients come through the constant cache with
// warp-uniform LDC loads; otherwise from the global table `cft` through L1.
#ifdef MG_CF_CONST
#define MG_CF_LOAD2(tab, k) make_double2(MG_CF_CONST[(tab) + (k)], MG_CF_CONST[(tab) + (k) + 1])
#else
#define MG_CF_LOAD2(tab, k) __ldg(reinterpret_cast<const double2*>(cft + (tab) + (k)))
#endif

namespace mgc {

template <class T, int NCOL>
__global__ void __launch_bounds__(128) colour_kernel(const double* __restrict__ cft, const T* __restrict__ jamp,
                                                     T* __restrict__ meh, long long stride, long long nevt, int nhel_run) {
  const long long ievt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int ih = blockIdx.y;
  if (ievt >= nevt) return;
  const T* __restrict__ jb = jamp + (long long)ih * (2 * NCOL) * stride + ievt;
  T me = T(0);
  int tab = 0;
#pragma unroll 1
  for (int i0 = 0; i0 < NCOL; i0 += 8) {
    T zr[8], zi[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) { zr[r] = T(0); zi[r] = T(0); }
#pragma unroll 2
    for (int j = i0; j < NCOL; ++j) {
      const T jr = jb[(2 * j) * stride], ji = jb[(2 * j + 1) * stride];
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const double2 c = MG_CF_LOAD2(tab, 2 * r);
        zr[2 * r] += T(c.x) * jr; zi[2 * r] += T(c.x) * ji;
        zr[2 * r + 1] += T(c.y) * jr; zi[2 * r + 1] += T(c.y) * ji;
      }
      tab += 8;
    }
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      if (i0 + r < NCOL) {
        const T jr = jb[(2 * (i0 + r)) * stride], ji = jb[(2 * (i0 + r) + 1) * stride];
        me += jr * zr[r] + ji * zi[r];
      }
    }
  }
  meh[(long long)ih * stride + ievt] = me;
}

// JAMP[f] = sum of the partial slots the diagram groups wrote for flow f (CSR table ptr/idx), per (event, helicity).
// Pure streaming: each partial is read once, each JAMP written once; thread = (event, helicity).
template <class T, int NCOL>
__global__ void __launch_bounds__(256) gather_kernel(const short* __restrict__ ptr, const short* __restrict__ idx, int npart,
                                                     const T* __restrict__ part, T* __restrict__ jsum, long long stride,
                                                     long long nevt) {
  const long long ievt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int ih = blockIdx.y;
  if (ievt >= nevt) return;
  const T* __restrict__ pb = part + (long long)ih * npart * 2 * stride + ievt;
  T* __restrict__ jb = jsum + (long long)ih * (2 * NCOL) * stride + ievt;
#pragma unroll 4
  for (int f = 0; f < NCOL; ++f) {
    T re = T(0), im = T(0);
    for (int q = ptr[f]; q < ptr[f + 1]; ++q) {
      const int s = idx[q];
      re += pb[(2 * s) * stride];
      im += pb[(2 * s + 1) * stride];
    }
    jb[(2 * f) * stride] = re;
    jb[(2 * f + 1) * stride] = im;
  }
}

// fixed-order helicity sum (deterministic), normalisation, optional per-helicity output; `first` = overwrite me_out,
// else accumulate (helicity chunks are processed one after the other on the same stream)
template <class T>
__global__ void helsum_kernel(const T* __restrict__ meh, long long stride, long long nevt, int nhel_run, T norm,
                              T* __restrict__ me_out, T* __restrict__ perhel_out, long long perhel_stride, bool first) {
  const long long ievt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (ievt >= nevt) return;
  T s = T(0);
  for (int ih = 0; ih < nhel_run; ++ih) {
    const T v = meh[(long long)ih * stride + ievt];
    if (perhel_out) perhel_out[(long long)ih * perhel_stride + ievt] = v * norm;
    s += v;
  }
  me_out[ievt] = first ? s * norm : me_out[ievt] + s * norm;
}

// Fused gather + colour sum: a CTA owns PAIRS consecutive events of one helicity; GROUPS thread groups (each PAIRS
// threads = whole warps, so table reads stay warp-uniform) first sum the partial slots of the flows f = g, g+GROUPS, ..
// into shared memory sJ[2f][pair], then split the 8-row blocks of the symmetric colour form among themselves
// (block b and its mirror, to balance the triangle), each streaming J from shared memory, and finally add their
// partial results in shared memory.  Every partial JAMP is read from DRAM exactly once and the summed JAMPs never
// leave the SM.
template <class T, int NCOL, int PAIRS, int GROUPS, bool DIRECT>
__global__ void __launch_bounds__(PAIRS * GROUPS) gather_colour_kernel(const double* __restrict__ cft, const short* __restrict__ ptr,
                                                                       const short* __restrict__ idx, int npart,
                                                                       const T* __restrict__ part, T* __restrict__ meh,
                                                                       long long stride, long long nevt) {
  extern __shared__ __align__(16) unsigned char smem_raw_c[];
  T* sJ = reinterpret_cast<T*>(smem_raw_c);                 // [2 * NCOL][PAIRS]
  T* red = sJ + 2 * NCOL * PAIRS;                           // [GROUPS][PAIRS]
  const int p = threadIdx.x % PAIRS, g = threadIdx.x / PAIRS;
  const long long ievt0 = (long long)blockIdx.x * PAIRS + p;
  const bool live = ievt0 < nevt;
  const long long ievt = live ? ievt0 : nevt - 1;
  const int ih = blockIdx.y;
  const T* __restrict__ pb = part + (long long)ih * npart * 2 * stride + ievt;
  if (DIRECT) {       // `part` already holds the summed JAMPs [NCOL][2][stride] (npart == NCOL): plain staged copy
#pragma unroll 8
    for (int f = g; f < NCOL; f += GROUPS) {
      sJ[(2 * f) * PAIRS + p] = pb[(2 * f) * stride];
      sJ[(2 * f + 1) * PAIRS + p] = pb[(2 * f + 1) * stride];
    }
  } else
  for (int f = g; f < NCOL; f += GROUPS) {
    T re = T(0), im = T(0);
    const int q1 = ptr[f + 1];
#pragma unroll 4
    for (int q = ptr[f]; q < q1; ++q) {
      const int s = idx[q];
      re += pb[(2 * s) * stride];
      im += pb[(2 * s + 1) * stride];
    }
    sJ[(2 * f) * PAIRS + p] = re;
    sJ[(2 * f + 1) * PAIRS + p] = im;
  }
  __syncthreads();
  constexpr int NB = (NCOL + 7) / 8;
  T me = T(0);
  // row blocks of this group: b = g, 2*GROUPS-1-g, 2*GROUPS+g, 4*GROUPS-1-g, ...  (boustrophedon over the triangle)
  for (int k = 0;; ++k) {
    const int b = (k & 1) ? (k + 1) * GROUPS - 1 - g : k * GROUPS + g;
    if (k * GROUPS >= NB) break;
    if (b >= NB) continue;
    const int i0 = 8 * b;
    // offset of block b in the blocked upper-triangular table: sum_{b' < b} (NCOL - 8 b') * 8
    int tab = 8 * (b * NCOL - 4 * b * (b - 1));
    T zr[8], zi[8];
#pragma unroll
    for (int r = 0; r < 8; ++r) { zr[r] = T(0); zi[r] = T(0); }
#pragma unroll 4
    for (int j = i0; j < NCOL; ++j) {
      const T jr = sJ[(2 * j) * PAIRS + p], ji = sJ[(2 * j + 1) * PAIRS + p];
#pragma unroll
      for (int r = 0; r < 4; ++r) {
        const double2 c = MG_CF_LOAD2(tab, 2 * r);
        zr[2 * r] += T(c.x) * jr; zi[2 * r] += T(c.x) * ji;
        zr[2 * r + 1] += T(c.y) * jr; zi[2 * r + 1] += T(c.y) * ji;
      }
      tab += 8;
    }
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      if (i0 + r < NCOL) me += sJ[(2 * (i0 + r)) * PAIRS + p] * zr[r] + sJ[(2 * (i0 + r) + 1) * PAIRS + p] * zi[r];
    }
  }
  if (GROUPS > 1) {
    red[g * PAIRS + p] = me;
    __syncthreads();
    if (g == 0) {
#pragma unroll
      for (int k = 1; k < GROUPS; ++k) me += red[k * PAIRS + p];    // fixed order: deterministic
    }
  }
  if (g == 0 && live) meh[(long long)ih * stride + ievt] = me;
}

// K6 on the FP64 tensor cores (north_star (4)): Z = CF . J as a batched dense contraction with
// mma.sync.m8n8k4.f64 (DMMA.8x8x4, the native FP64 MMA shape of sm_100a), then me = sum_i Re(J_i^* Z_i).
// CTA = 4 warps x 32 events of one helicity; the 2*NCOL x 32 JAMP tile is staged once in shared memory (B operand:
// k = flow j, n = (event, re/im)); warp w owns the row blocks w, w+4, ... of CF (A operand, dense [NCOL][NCOL]
// table in global memory, L1-resident) and reuses every A fragment for the 8 column tiles.  The dense product
// uses the symmetry of CF at the level of 8x8 blocks (upper block triangle only, off-diagonal blocks doubled).
template <int NCOL>
__global__ void __launch_bounds__(128) colour_dmma_kernel(const double* __restrict__ cfd, const double* __restrict__ jamp,
                                                          double* __restrict__ meh, long long stride, long long nevt) {
  constexpr int PAIRS = 32, RS = 34;     // row stride 34: the 8 rows x 2 events a half-warp reads fall into 16 distinct banks
  extern __shared__ __align__(16) unsigned char smem_raw_d[];
  double* sJ = reinterpret_cast<double*>(smem_raw_d);     // [2 * NCOL][RS]
  double* red = sJ + 2 * NCOL * RS;                    // [4][PAIRS]
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int ih = blockIdx.y;
  {
    const int p = lane;
    const long long ievt0 = (long long)blockIdx.x * PAIRS + p;
    const long long ievt = ievt0 < nevt ? ievt0 : nevt - 1;
    const double* __restrict__ jb = jamp + (long long)ih * (2 * NCOL) * stride + ievt;
#pragma unroll 8
    for (int q = w; q < 2 * NCOL; q += 4) sJ[q * RS + p] = jb[q * stride];
  }
  __syncthreads();
  const int ar = lane >> 2, ak = lane & 3;          // A: row ar, k ak ; B: k ak, column ar ; C: row ar, columns 2*ak, 2*ak+1
  const int bc = ar & 1, bp = ar >> 1;              // B column ar = (event bp within the tile of 4, component bc)
  double mep[8];
#pragma unroll
  for (int ct = 0; ct < 8; ++ct) mep[ct] = 0.0;
  // block-triangular: row block rb only meets column blocks kb >= rb (the table holds CF on the diagonal blocks and
  // 2 CF above them), which halves the MMAs; warps take row blocks boustrophedon to balance the triangle
  for (int t = 0;; ++t) {
    const int rb = (t & 1) ? (t + 1) * 4 - 1 - w : t * 4 + w;
    if (t * 4 >= NCOL / 8) break;
    if (rb >= NCOL / 8) continue;
    double c0[8], c1[8];
#pragma unroll
    for (int ct = 0; ct < 8; ++ct) { c0[ct] = 0.0; c1[ct] = 0.0; }
    const double* __restrict__ arow = cfd + (long long)(rb * 8 + ar) * NCOL + ak;
#pragma unroll 2
    for (int k0 = rb * 8; k0 < NCOL; k0 += 4) {
      const double a = __ldg(arow + k0);
      const double* __restrict__ brow = sJ + (2 * (k0 + ak) + bc) * RS + bp;
#pragma unroll
      for (int ct = 0; ct < 8; ++ct) {
        const double b = brow[ct * 4];
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(c0[ct]), "+d"(c1[ct]) : "d"(a), "d"(b));
      }
    }
    // C fragment: Z[rb*8 + ar][event ct*4 + ak] = (c0, c1) = (re, im)
    const int i = rb * 8 + ar;
#pragma unroll
    for (int ct = 0; ct < 8; ++ct) {
      const int p = ct * 4 + ak;
      mep[ct] += sJ[(2 * i) * RS + p] * c0[ct] + sJ[(2 * i + 1) * RS + p] * c1[ct];
    }
  }
  // sum over the 8 rows held by lanes with the same ak (fixed order: deterministic), then over the 4 warps
#pragma unroll
  for (int ct = 0; ct < 8; ++ct) {
    double v = mep[ct];
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    v += __shfl_xor_sync(0xffffffffu, v, 8);
    v += __shfl_xor_sync(0xffffffffu, v, 16);
    if (ar == 0) red[w * PAIRS + ct * 4 + ak] = v;
  }
  __syncthreads();
  if (w == 0) {
    const long long ievt = (long long)blockIdx.x * PAIRS + lane;
    if (ievt < nevt) meh[(long long)ih * stride + ievt] = (red[lane] + red[PAIRS + lane]) + (red[2 * PAIRS + lane] + red[3 * PAIRS + lane]);
  }
}

template <class T, int NCOL>
void gather_colour_sum(const double* cft, const short* ptr, const short* idx, int npart, const T* part, T* jsum, T* meh,
                       long long stride, long long nevt, int nhel_run, T norm, T* me_out, T* perhel_out,
                       long long perhel_stride, bool first, bool gather, cudaStream_t st, const double* cfd_dense = nullptr) {
  // NCOL <= 32: one thread per pair does everything (128 pairs per CTA); larger bases: 32 pairs x 5 groups
  constexpr int PAIRS = NCOL <= 32 ? 128 : 32, GROUPS = NCOL <= 32 ? 1 : 5;
  const size_t smem = (size_t)(2 * NCOL + GROUPS) * PAIRS * sizeof(T);
  const dim3 grid((unsigned)((nevt + PAIRS - 1) / PAIRS), (unsigned)nhel_run);
  static bool attr_set = false;
#ifdef MG_FUSED_COLOUR
  // measured on B200: 5.5M vs 6.1M ME/s (gg->tt~gg), 165k vs 168k (gg->tt~ggg) — the separate gather
  // kernel streams the partial slots at 84 % of the DRAM peak, the fused one cannot keep as many loads in flight
  auto kern = gather_colour_kernel<T, NCOL, PAIRS, GROUPS, false>;
  if (!attr_set) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr_set = true; }
  kern<<<grid, PAIRS * GROUPS, smem, st>>>(cft, ptr, idx, npart, part, meh, stride, nevt);
  (void)gather;
#else
  // gather == false: the diagram-group kernels accumulated the JAMPs in place (jsum == part, npart == NCOL)
  if (gather) {
    const dim3 g1((unsigned)((nevt + 255) / 256), (unsigned)nhel_run);
    gather_kernel<T, NCOL><<<g1, 256, 0, st>>>(ptr, idx, npart, part, jsum, stride, nevt);
  }
#ifndef MG_COLOUR_NO_DMMA
  // large colour basis in fp64: dense contraction on the FP64 tensor cores (measured 277k vs 273k ME/s for gg->tt~ggg
  // against the shared-memory staged scalar kernel below, which stays for fp32 and as the reference variant)
  if (sizeof(T) == 8 && NCOL > 32 && NCOL % 8 == 0 && cfd_dense != nullptr) {
    const size_t sm = ((size_t)2 * NCOL * 34 + 4 * 32) * sizeof(double);
    auto kd = colour_dmma_kernel<NCOL>;
    static bool dset = false;
    if (!dset) { cudaFuncSetAttribute(kd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); dset = true; }
    kd<<<dim3((unsigned)((nevt + 31) / 32), (unsigned)nhel_run), 128, sm, st>>>(cfd_dense, (const double*)jsum, (double*)meh, stride, nevt);
  } else
#endif
  if (NCOL > 32) {
    // large colour basis: JAMPs staged once in shared memory (the plain kernel re-reads them 7.7x from DRAM at
    // NCOL = 120); measured +3 % on gg->tt~ggg, -1 % on gg->tt~gg (NCOL = 24, where the plain kernel stays)
    auto kern = gather_colour_kernel<T, NCOL, PAIRS, GROUPS, true>;
    if (!attr_set) { cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr_set = true; }
    kern<<<grid, PAIRS * GROUPS, smem, st>>>(cft, ptr, idx, NCOL, jsum, meh, stride, nevt);
  } else {
    const dim3 grid2((unsigned)((nevt + 127) / 128), (unsigned)nhel_run);
    colour_kernel<T, NCOL><<<grid2, 128, 0, st>>>(cft, jsum, meh, stride, nevt, nhel_run);
  }
#endif
  helsum_kernel<T><<<(unsigned)((nevt + 255) / 256), 256, 0, st>>>(meh, stride, nevt, nhel_run, norm, me_out, perhel_out,
                                                                   perhel_stride, first);
}

}  // namespace mgc
