// mg_internal.h — declarations shared by the hand-written translation units of libmg5b200.so.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

constexpr int MG_NEPP_I = 32;   // events per AoSoA page (== MG_NEPP of include/mg5b200.h)
constexpr int MG_WEIGHT_MAX_BLOCKS = 4096;   // partial results of mg_weight_max's first reduction stage

// parameter vector handed to every generated launch function
enum { MG_PAR_GS2 = 0, MG_PAR_MT = 1, MG_PAR_E2 = 2, MG_PAR_GL = 3, MG_PAR_GR = 4, MG_PAR_MZ2 = 5, MG_PAR_MZGZ = 6,
       MG_NPAR_VEC = 8 };

cudaError_t mg_launch_rambo(int nfinal, const double* masses, double sqrt_s, uint64_t seed, long long first_event,
                            long long nevt, double* mom, double* wgt, cudaStream_t st);
cudaError_t mg_launch_philox_raw(uint64_t seed, long long first_event, long long nevt, int nfinal, uint32_t* out,
                                 cudaStream_t st);
// mg_reduce.cu
cudaError_t mg_launch_probe_stats(int prec, const void* perhel, long long nevt, int nhel, double* out, cudaStream_t st);
int mg_weight_blocks(long long n);
cudaError_t mg_launch_weight_max(int prec, void* me, const double* w, long long n, double* part, double* out, cudaStream_t st);
// mixed precision with precision tracking (mg_sigma_mixed)
cudaError_t mg_launch_mixed_flag(const float* perhel, const double* mom, long long nevt, int nhel, int npar, unsigned massless_mask,
                                 double kappa, double tol, double* me_out, float* eps_out, int* flagged, int* nflagged,
                                 cudaStream_t st);
cudaError_t mg_launch_mixed_gather(const double* mom, const int* flagged, int n, int npar, double* out, cudaStream_t st);
cudaError_t mg_launch_mixed_scatter(const double* me64, const int* flagged, int n, double* me_out, cudaStream_t st);
// mg_api.cu: sets the thread's mg_last_error() text (for translation units other than mg_api.cu)
void mg_set_last_error(const char* text);
