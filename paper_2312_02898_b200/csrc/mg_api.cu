// mg_api.cu — the C ABI of include/mg5b200.h: argument checking, handle management, helicity filter (K8),
// and dispatch to the generated per-process launchers.  No arithmetic of the method lives here.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <string>
#include <vector>

#include "../../include/mg5b200.h"
#include "mg_internal.h"
#include "mg_kernel.cuh"

// table of generated processes: csrc/generated/mg_registry.cu (written by the generator)
extern const mg_procdesc_t* const mg_registry[];
extern const int mg_registry_n;

static thread_local char g_err[512] = "";
static int cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_err, sizeof g_err, "%s: %s", where, cudaGetErrorString(e));
  return MG_ERR_CUDA;
}
#define MG_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)

struct mg_process {
  const mg_procdesc_t* desc;
  mg_params_t par;
  double pvec[MG_NPAR_VEC];
  double masses[8];
  int nfinal;
  int* hel_dev;            // good-helicity list on the device (nhel ints)
  int* hel_all_dev;        // 0..nhel-1
  std::vector<int> good;
  bool probed;
  long long launches;      // kernels launched by the last mg_sigma / mg_sigma_per_helicity call
  void* io_mom; size_t io_mom_bytes;   // device staging of mg_sigma_host (grow-only, library-owned)
  void* io_out; size_t io_out_bytes;
  void* ws;                // workspace of the split kernel shape (JAMPs + per-helicity values), library-owned
  size_t ws_bytes;
};

// Workspace for the split kernel shape: jamp[nhel_run][ncol][2][tile] + meh[nhel_run][tile]; the generated launcher
// tiles the batch so that it fits.  Capped at MG5B200_WS_GB GiB (default: min(64, 40 % of free memory)).  Grows on demand (synchronous
// cudaFree/cudaMalloc on the first call that needs more), never shrinks.
static int ensure_ws(mg_process* p, int64_t nevt, int nhel_run) {
  const int ip = p->par.precision == MG_FP64 ? 0 : 1;
  const size_t per_eh = (size_t)p->desc->ws_bytes_per_event_hel[ip], per_e = (size_t)p->desc->ws_bytes_per_event[ip];
  if (per_eh == 0) return MG_OK;
  // default cap: 64 GiB or 40 % of the free device memory, whichever is smaller (B200: 180 GB)
  double cap_gb = 64.0;
  size_t free_b = 0, total_b = 0;
  if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
    const double f = 0.4 * (double)(free_b + p->ws_bytes) / 1073741824.0;
    if (f < cap_gb) cap_gb = f;
  }
  if (const char* e = getenv("MG5B200_WS_GB")) { const double v = atof(e); if (v > 0) cap_gb = v; }
  const size_t cap = (size_t)(cap_gb * 1073741824.0);
  size_t E = (size_t)((nevt + 31) / 32 * 32);
  if (E > ((size_t)1 << 20)) E = (size_t)1 << 20;             // the launcher's largest event tile
  size_t need = E * (per_e + (size_t)nhel_run * per_eh);      // whole batch, whole helicity list resident
  if (need > cap) need = cap;
  const size_t floor_bytes = (E < 1024 ? E : 1024) * (per_e + 4 * per_eh);
  if (need < floor_bytes) need = floor_bytes;
  if (p->ws_bytes >= need) return MG_OK;
  if (p->ws) { cudaDeviceSynchronize(); cudaFree(p->ws); p->ws = nullptr; p->ws_bytes = 0; }
  MG_CUDA(cudaMalloc(&p->ws, need));
  p->ws_bytes = need;
  return MG_OK;
}

static std::string squeeze(const char* s) {
  std::string o;
  for (; *s; ++s) if (!isspace((unsigned char)*s)) o.push_back(*s);
  return o;
}

extern "C" {

int mg_params_default(mg_params_t* p) {
  if (!p) return MG_ERR_NULL;
  memset(p, 0, sizeof *p);
  p->struct_size = sizeof(mg_params_t);
  p->precision = MG_FP64; p->helicity_mode = MG_HEL_FILTER; p->device = 0;
  p->alpha_s = 0.118; p->alpha_ew_inv = 132.507; p->gf = 1.16639e-5; p->sw2 = 0.0;
  p->mz = 91.188; p->gamma_z = 2.4414; p->mt = 173.0; p->gamma_t = 0.0;
  return MG_OK;
}

int mg_process_create(const char* proc, const mg_params_t* params, mg_process_t** out) {
  if (!proc || !params || !out) return MG_ERR_NULL;
  *out = nullptr;
  if (params->struct_size != sizeof(mg_params_t)) return MG_ERR_BAD_PARAM;
  if (params->helicity_mode != MG_HEL_FILTER && params->helicity_mode != MG_HEL_ALL) return MG_ERR_BAD_PARAM;
  if (!(params->alpha_s > 0) || !(params->alpha_ew_inv > 0) || !(params->mz > 0) || !(params->mt >= 0) ||
      params->gamma_t != 0.0)
    return MG_ERR_BAD_PARAM;
  const std::string key = squeeze(proc);
  const mg_procdesc_t* d = nullptr;
  for (int i = 0; i < mg_registry_n; ++i) if (squeeze(mg_registry[i]->proc) == key) d = mg_registry[i];
  if (!d) return MG_ERR_BAD_PROC;
  if (params->precision != MG_FP64 && !(params->precision == MG_FP32 && d->has_fp32)) return MG_ERR_BAD_PARAM;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || params->device < 0 || params->device >= ndev) {
    cudaGetLastError();
    return MG_ERR_NO_DEVICE;
  }
  MG_CUDA(cudaSetDevice(params->device));
  mg_process* p = new mg_process();
  p->desc = d; p->par = *params; p->probed = false; p->ws = nullptr; p->ws_bytes = 0; p->launches = 0;
  p->io_mom = p->io_out = nullptr; p->io_mom_bytes = p->io_out_bytes = 0;
  p->nfinal = d->npar - 2;
  for (int i = 0; i < 8; ++i) p->masses[i] = (i < d->npar && d->massive[i]) ? params->mt : 0.0;
  // derived couplings (DESIGN.md §3 C2, reading A1)
  const double pi = 3.14159265358979323846;
  const double aew = 1.0 / params->alpha_ew_inv;
  double sw2 = params->sw2;
  if (!(sw2 > 0)) {
    const double mz2 = params->mz * params->mz;
    const double mw2 = mz2 / 2 + sqrt(mz2 * mz2 / 4 - pi * aew * mz2 / (sqrt(2.0) * params->gf));
    sw2 = 1.0 - mw2 / mz2;
  }
  const double e2 = 4 * pi * aew, e = sqrt(e2);
  const double gz = e / (2 * sqrt(sw2 * (1 - sw2))), gv = -0.5 + 2 * sw2, ga = -0.5;
  memset(p->pvec, 0, sizeof p->pvec);
  p->pvec[MG_PAR_GS2] = 4 * pi * params->alpha_s;
  p->pvec[MG_PAR_MT] = params->mt;
  p->pvec[MG_PAR_E2] = e2;
  p->pvec[MG_PAR_GL] = -gz * (gv + ga);
  p->pvec[MG_PAR_GR] = -gz * (gv - ga);
  p->pvec[MG_PAR_MZ2] = params->mz * params->mz;
  p->pvec[MG_PAR_MZGZ] = params->mz * params->gamma_z;
  std::vector<int> all(d->nhel);
  for (int h = 0; h < d->nhel; ++h) all[h] = h;
  p->good = all;
  cudaError_t e1 = cudaMalloc(&p->hel_dev, sizeof(int) * d->nhel);
  cudaError_t e2c = e1 == cudaSuccess ? cudaMalloc(&p->hel_all_dev, sizeof(int) * d->nhel) : e1;
  if (e2c != cudaSuccess) { delete p; return cuda_fail(e2c, "cudaMalloc(helicity list)"); }
  cudaMemcpy(p->hel_dev, all.data(), sizeof(int) * d->nhel, cudaMemcpyHostToDevice);
  cudaMemcpy(p->hel_all_dev, all.data(), sizeof(int) * d->nhel, cudaMemcpyHostToDevice);
  if (params->helicity_mode == MG_HEL_ALL) p->probed = true;
  *out = p;
  return MG_OK;
}

int mg_process_destroy(mg_process_t* p) {
  if (!p) return MG_ERR_NULL;
  cudaSetDevice(p->par.device);
  cudaFree(p->hel_dev);
  cudaFree(p->hel_all_dev);
  if (p->ws) cudaFree(p->ws);
  if (p->io_mom) cudaFree(p->io_mom);
  if (p->io_out) cudaFree(p->io_out);
  delete p;
  return MG_OK;
}

size_t mg_momenta_bytes(const mg_process_t* p, int64_t nevt) {
  if (!p || nevt < 0) return 0;
  const int64_t pages = (nevt + MG_NEPP - 1) / MG_NEPP;
  return (size_t)pages * p->desc->npar * MG_NEPP * 4 * sizeof(double);
}

int mg_rambo_ex(mg_process_t* p, uint64_t seed, double sqrt_s, int64_t first_event, int64_t nevt,
                void* momenta_dev, double* weights_dev, void* stream) {
  if (!p || (!momenta_dev && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0 || first_event < 0) return MG_ERR_BAD_NEVT;
  if (((uintptr_t)momenta_dev & 15) || ((uintptr_t)weights_dev & 7)) return MG_ERR_ALIGN;
  double sm = 0;
  for (int f = 0; f < p->nfinal; ++f) sm += p->masses[2 + f];
  if (!(sqrt_s > sm)) return MG_ERR_KINEMATICS;
  MG_CUDA(cudaSetDevice(p->par.device));
  MG_CUDA(mg_launch_rambo(p->nfinal, p->masses + 2, sqrt_s, seed, first_event, nevt, (double*)momenta_dev, weights_dev,
                          (cudaStream_t)stream));
  return MG_OK;
}
int mg_rambo(mg_process_t* p, uint64_t seed, double sqrt_s, int64_t nevt, void* momenta_dev, void* stream) {
  return mg_rambo_ex(p, seed, sqrt_s, 0, nevt, momenta_dev, nullptr, stream);
}

int mg_philox_raw(mg_process_t* p, uint64_t seed, int64_t first_event, int64_t nevt, uint32_t* out_dev, void* stream) {
  if (!p || (!out_dev && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0 || first_event < 0) return MG_ERR_BAD_NEVT;
  if ((uintptr_t)out_dev & 15) return MG_ERR_ALIGN;
  MG_CUDA(cudaSetDevice(p->par.device));
  MG_CUDA(mg_launch_philox_raw(seed, first_event, nevt, p->nfinal, out_dev, (cudaStream_t)stream));
  return MG_OK;
}

static size_t esize(const mg_process_t* p) { return p->par.precision == MG_FP64 ? 8 : 4; }

int mg_sigma_per_helicity(mg_process_t* p, const void* momenta_dev, int64_t nevt, void* perhel_out_dev, void* stream) {
  if (!p || ((!momenta_dev || !perhel_out_dev) && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0) return MG_ERR_BAD_NEVT;
  if (((uintptr_t)momenta_dev & 15) || ((uintptr_t)perhel_out_dev & 7)) return MG_ERR_ALIGN;
  if (nevt == 0) return MG_OK;
  MG_CUDA(cudaSetDevice(p->par.device));
  void* tmp = nullptr;
  { const int rc = ensure_ws(p, nevt, p->desc->nhel); if (rc != MG_OK) return rc; }
  MG_CUDA(cudaMalloc(&tmp, esize(p) * (size_t)nevt));
  p->launches = p->desc->launch(p->par.precision, (const double*)momenta_dev, tmp, nevt, p->hel_all_dev, p->desc->nhel,
                  perhel_out_dev, p->pvec, p->ws, p->ws_bytes, (cudaStream_t)stream);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
  cudaFree(tmp);
  if (e != cudaSuccess) return cuda_fail(e, "sigma_per_helicity");
  return MG_OK;
}

int mg_helicity_probe(mg_process_t* p, const void* momenta_dev, int64_t nprobe, void* stream) {
  if (!p || !momenta_dev) return MG_ERR_NULL;
  if (nprobe <= 0) return MG_ERR_BAD_NEVT;
  const int nhel = p->desc->nhel;
  void* ph = nullptr;
  MG_CUDA(cudaSetDevice(p->par.device));
  MG_CUDA(cudaMalloc(&ph, esize(p) * (size_t)nprobe * nhel));
  int rc = mg_sigma_per_helicity(p, momenta_dev, nprobe, ph, stream);
  if (rc != MG_OK) { cudaFree(ph); return rc; }
  std::vector<double> sum(nhel, 0.0);
  if (p->par.precision == MG_FP64) {
    std::vector<double> h((size_t)nprobe * nhel);
    cudaMemcpy(h.data(), ph, sizeof(double) * h.size(), cudaMemcpyDeviceToHost);
    for (int ih = 0; ih < nhel; ++ih) for (int64_t i = 0; i < nprobe; ++i) sum[ih] += h[(size_t)ih * nprobe + i];
  } else {
    std::vector<float> h((size_t)nprobe * nhel);
    cudaMemcpy(h.data(), ph, sizeof(float) * h.size(), cudaMemcpyDeviceToHost);
    for (int ih = 0; ih < nhel; ++ih) for (int64_t i = 0; i < nprobe; ++i) sum[ih] += h[(size_t)ih * nprobe + i];
  }
  cudaFree(ph);
  double tot = 0;
  for (double s : sum) tot += s;
  // reading A6: h is good iff sum_probe ME_h > eps * sum_probe sum_h ME_h
  const double eps = p->par.precision == MG_FP64 ? 1e-14 : 1e-6;
  p->good.clear();
  for (int ih = 0; ih < nhel; ++ih) if (sum[ih] > eps * tot) p->good.push_back(ih);
  if (p->good.empty()) for (int ih = 0; ih < nhel; ++ih) p->good.push_back(ih);
  MG_CUDA(cudaMemcpy(p->hel_dev, p->good.data(), sizeof(int) * p->good.size(), cudaMemcpyHostToDevice));
  p->probed = true;
  return MG_OK;
}

int mg_sigma(mg_process_t* p, const void* momenta_dev, int64_t nevt, void* me_out_dev, void* stream) {
  if (!p || ((!momenta_dev || !me_out_dev) && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0) return MG_ERR_BAD_NEVT;
  if (((uintptr_t)momenta_dev & 15) || ((uintptr_t)me_out_dev & (esize(p) - 1))) return MG_ERR_ALIGN;
  if (nevt == 0) return MG_OK;
  MG_CUDA(cudaSetDevice(p->par.device));
  if (!p->probed) {
    int rc = mg_helicity_probe(p, momenta_dev, nevt < 4096 ? nevt : 4096, stream);
    if (rc != MG_OK) return rc;
  }
  { const int rc = ensure_ws(p, nevt, (int)p->good.size()); if (rc != MG_OK) return rc; }
  p->launches = p->desc->launch(p->par.precision, (const double*)momenta_dev, me_out_dev, nevt, p->hel_dev, (int)p->good.size(),
                  nullptr, p->pvec, p->ws, p->ws_bytes, (cudaStream_t)stream);
  MG_CUDA(cudaGetLastError());
  return MG_OK;
}

int mg_sigma_host(mg_process_t* p, const void* momenta_host, int64_t nevt, void* me_out_host, void* stream) {
  if (!p || ((!momenta_host || !me_out_host) && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0) return MG_ERR_BAD_NEVT;
  if (nevt == 0) return MG_OK;
  MG_CUDA(cudaSetDevice(p->par.device));
  cudaStream_t st = (cudaStream_t)stream;
  // device staging buffers are kept in the handle and only ever grow (a stream-ordered allocation per call showed
  // occasional second-long stalls when the pool returned memory to the OS between calls)
  const size_t mb = mg_momenta_bytes(p, nevt), ob = esize(p) * (size_t)nevt;
  if (p->io_mom_bytes < mb) {
    if (p->io_mom) { cudaDeviceSynchronize(); cudaFree(p->io_mom); p->io_mom = nullptr; p->io_mom_bytes = 0; }
    MG_CUDA(cudaMalloc(&p->io_mom, mb));
    p->io_mom_bytes = mb;
  }
  if (p->io_out_bytes < ob) {
    if (p->io_out) { cudaDeviceSynchronize(); cudaFree(p->io_out); p->io_out = nullptr; p->io_out_bytes = 0; }
    MG_CUDA(cudaMalloc(&p->io_out, ob));
    p->io_out_bytes = ob;
  }
  void *dm = p->io_mom, *dout = p->io_out;
  int rc = MG_OK;
  cudaError_t e = cudaMemcpyAsync(dm, momenta_host, mb, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) rc = mg_sigma(p, dm, nevt, dout, stream);
  if (e == cudaSuccess && rc == MG_OK) e = cudaMemcpyAsync(me_out_host, dout, ob, cudaMemcpyDeviceToHost, st);
  cudaError_t es = cudaStreamSynchronize(st);
  if (rc != MG_OK) return rc;
  if (e != cudaSuccess) return cuda_fail(e, "mg_sigma_host copy");
  if (es != cudaSuccess) return cuda_fail(es, "mg_sigma_host sync");
  return MG_OK;
}

int mg_good_helicities(const mg_process_t* p, int32_t* out, int32_t capacity, int32_t* ngood) {
  if (!p || !ngood) return MG_ERR_NULL;
  *ngood = (int32_t)p->good.size();
  if (out) for (int i = 0; i < capacity && i < (int)p->good.size(); ++i) out[i] = p->good[i];
  return MG_OK;
}

int mg_process_info(const mg_process_t* p, mg_info_t* o) {
  if (!p || !o) return MG_ERR_NULL;
  const mg_procdesc_t* d = p->desc;
  o->npar = d->npar; o->nfinal = d->npar - 2; o->ndiagrams = d->ndiagrams; o->nhel = d->nhel;
  o->ngoodhel = (int)p->good.size(); o->ncolor = d->ncol; o->denominator = d->denominator; o->nepp = MG_NEPP;
  o->flops_per_event_allhel = d->flops_algorithmic * d->nhel;
  o->flops_per_event_goodhel = d->flops_algorithmic * (long long)p->good.size();
  o->flops_executed_per_event_goodhel = d->flops_per_helicity * (long long)p->good.size();
  for (int i = 0; i < 8; ++i) o->masses[i] = p->masses[i];
  o->nkernels_per_tile = d->nkernels;
  o->launches_last_sigma = (int32_t)p->launches;
  o->workspace_bytes = (int64_t)p->ws_bytes;
  return MG_OK;
}

int mg_fma_peak(int device, int prec, double* flops_per_s) {
  if (!flops_per_s) return MG_ERR_NULL;
  if (prec != MG_FP64 && prec != MG_FP32) return MG_ERR_BAD_PARAM;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return MG_ERR_NO_DEVICE; }
  MG_CUDA(cudaSetDevice(device));
  MG_CUDA(mg_run_fma_peak(prec, flops_per_s));
  return MG_OK;
}

int mg_dmma_peak(int device, double* flops_per_s) {
  if (!flops_per_s) return MG_ERR_NULL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { cudaGetLastError(); return MG_ERR_NO_DEVICE; }
  MG_CUDA(cudaSetDevice(device));
  MG_CUDA(mg_run_dmma_peak(flops_per_s));
  return MG_OK;
}

const char* mg_status_string(int s) {
  switch (s) {
    case MG_OK: return "ok";
    case MG_ERR_NULL: return "null pointer argument";
    case MG_ERR_BAD_PROC: return "unknown process string";
    case MG_ERR_BAD_PARAM: return "bad parameter struct";
    case MG_ERR_BAD_NEVT: return "bad event count";
    case MG_ERR_ALIGN: return "misaligned device pointer";
    case MG_ERR_KINEMATICS: return "sqrt_s not above the final-state mass threshold";
    case MG_ERR_CUDA: return "CUDA error";
    case MG_ERR_NO_DEVICE: return "no CUDA device";
    default: return "unknown status";
  }
}
const char* mg_last_error(void) { return g_err; }

}  // extern "C"
