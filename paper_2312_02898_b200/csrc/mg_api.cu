// mg_api.cu — the C ABI of include/mg5b200.h: argument checking, handle management, helicity filter (K8),
// workspace, and dispatch to the generated per-process launchers.  No arithmetic of the method lives here.
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
static int fail(int status, const char* what) {
  snprintf(g_err, sizeof g_err, "%s", what);
  return status;
}
void mg_set_last_error(const char* text) { snprintf(g_err, sizeof g_err, "%s", text); }
#define MG_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)

struct mg_process {
  const mg_procdesc_t* desc = nullptr;
  mg_params_t par;
  double pvec[MG_NPAR_VEC];
  double masses[8];
  int nfinal = 0, nsm = 0;
  // helicity state (K8).  good: helicities that contribute; run: the ones evaluated, with weights (2 = stands for its
  // helicity-flipped mirror as well, which is then not evaluated)
  std::vector<int> good, run;
  std::vector<double> run_w;
  bool probed = false;
  int* hel_dev = nullptr;        // fused shape: run list / all helicities
  int* hel_all_dev = nullptr;
  double* helw_dev = nullptr;    // fused shape: weights of the run list / ones
  double* ones_dev = nullptr;
  void* lanew_dev = nullptr;     // event-CTA shape: lane weights [2][nlane] (element type of the precision) / ones
  void* lanew_all_dev = nullptr;
  int ntb = 2, tb_first = 0;     // event-CTA shape: top-quark helicities run
  double* stats_dev = nullptr;   // probe statistics [2][nhel]; first 3 doubles double as mg_weight_max's default output
  double* wpart_dev = nullptr;   // mg_weight_max stage-1 partials
  long long launches = 0;        // kernels launched by the last mg_sigma / mg_sigma_per_helicity call
  void* io_mom = nullptr; size_t io_mom_bytes = 0;   // device staging of mg_sigma_host (grow-only, library-owned)
  void* io_out = nullptr; size_t io_out_bytes = 0;
  void* ws = nullptr; size_t ws_bytes = 0; bool ws_user = false;   // event-CTA shape: JAMP scratch + per-event invariants
  void* lanew_all32_dev = nullptr;   // ones as float: fp32 pass of mg_sigma_mixed on an fp64 handle
  void* mx = nullptr; size_t mx_bytes = 0;   // scratch of mg_sigma_mixed (grow-only, library-owned)
};

static size_t esize(const mg_process_t* p) { return p->par.precision == MG_FP64 ? 8 : 4; }

static void free_all(mg_process* p) {
  cudaFree(p->hel_dev); cudaFree(p->hel_all_dev); cudaFree(p->helw_dev); cudaFree(p->ones_dev);
  cudaFree(p->lanew_dev); cudaFree(p->lanew_all_dev); cudaFree(p->stats_dev); cudaFree(p->wpart_dev);
  if (p->ws && !p->ws_user) cudaFree(p->ws);
  cudaFree(p->lanew_all32_dev); cudaFree(p->mx);
  if (p->io_mom) cudaFree(p->io_mom);
  if (p->io_out) cudaFree(p->io_out);
  cudaGetLastError();
}

// Workspace of the event-CTA shape: JAMP scratch for every resident CTA (desc->ctas_per_sm per SM) + the per-event invariants
// of one event tile.  Library-owned by default: sized for the whole batch, capped at MG_WS_DEFAULT_CAP, grown on
// demand (synchronously), never shrunk; or caller-provided through mg_set_workspace.
static const size_t MG_WS_DEFAULT_CAP = (size_t)1 << 30;
static size_t ws_scratch_bytes(const mg_process* p) {
  return (size_t)p->desc->ctas_per_sm * p->nsm * (size_t)p->desc->ws_bytes_per_cta[p->par.precision == MG_FP64 ? 0 : 1];
}
static size_t ws_need(const mg_process* p, int64_t nevt) {
  const size_t per_e = (size_t)p->desc->ws_bytes_per_event[p->par.precision == MG_FP64 ? 0 : 1];
  return ws_scratch_bytes(p) + per_e * (size_t)((nevt + 31) / 32 * 32);
}
static int ensure_ws(mg_process* p, int64_t nevt) {
  if (!p->desc->launch_slots) return MG_OK;
  const size_t per_e = (size_t)p->desc->ws_bytes_per_event[p->par.precision == MG_FP64 ? 0 : 1];
  const size_t floor_bytes = ws_scratch_bytes(p) + per_e * 32;
  if (p->ws_user) return p->ws_bytes >= floor_bytes ? MG_OK : fail(MG_ERR_BAD_PARAM, "caller-provided workspace too small");
  size_t need = ws_need(p, nevt);
  if (need > MG_WS_DEFAULT_CAP) need = MG_WS_DEFAULT_CAP;
  if (need < floor_bytes + per_e * 4096) need = floor_bytes + per_e * 4096;
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

// lane index of helicity h in the event-CTA shape: the helicity bits of all particles but the top quark (bit tpos)
static int lane_of(int h, int tpos) { return ((h >> (tpos + 1)) << tpos) | (h & ((1 << tpos) - 1)); }

// uploads the run list / weights of the current helicity state
static int upload_helicities(mg_process* p) {
  const mg_procdesc_t* d = p->desc;
  if (d->launch) {
    MG_CUDA(cudaMemcpy(p->hel_dev, p->run.data(), sizeof(int) * p->run.size(), cudaMemcpyHostToDevice));
    MG_CUDA(cudaMemcpy(p->helw_dev, p->run_w.data(), sizeof(double) * p->run_w.size(), cudaMemcpyHostToDevice));
    return MG_OK;
  }
  const int tpos = d->npar - 3, nl = d->nlane;
  std::vector<double> w(2 * nl, 0.0);
  bool any[2] = {false, false};
  for (size_t i = 0; i < p->run.size(); ++i) {
    const int h = p->run[i], tb = (h >> tpos) & 1;
    w[tb * nl + lane_of(h, tpos)] = p->run_w[i];
    any[tb] = true;
  }
  p->ntb = (any[0] && any[1]) ? 2 : 1;
  p->tb_first = any[1] ? 1 : 0;
  if (p->par.precision == MG_FP64) {
    MG_CUDA(cudaMemcpy(p->lanew_dev, w.data(), sizeof(double) * w.size(), cudaMemcpyHostToDevice));
  } else {
    std::vector<float> wf(w.begin(), w.end());
    MG_CUDA(cudaMemcpy(p->lanew_dev, wf.data(), sizeof(float) * wf.size(), cudaMemcpyHostToDevice));
  }
  return MG_OK;
}

static int run_sigma(mg_process* p, const void* mom, int64_t nevt, void* me_out, void* perhel, bool all, cudaStream_t st) {
  const mg_procdesc_t* d = p->desc;
  long long n;
  if (d->launch) {
    n = all ? d->launch(p->par.precision, (const double*)mom, me_out, nevt, p->hel_all_dev, p->ones_dev, d->nhel, perhel, p->pvec, st)
            : d->launch(p->par.precision, (const double*)mom, me_out, nevt, p->hel_dev, p->helw_dev, (int)p->run.size(), perhel, p->pvec, st);
  } else {
    { const int rc = ensure_ws(p, nevt); if (rc != MG_OK) return rc; }
    n = all ? d->launch_slots(p->par.precision, (const double*)mom, me_out, nevt, p->lanew_all_dev, 2, 0, perhel, p->pvec, p->ws, p->ws_bytes, st)
            : d->launch_slots(p->par.precision, (const double*)mom, me_out, nevt, p->lanew_dev, p->ntb, p->tb_first, perhel, p->pvec, p->ws, p->ws_bytes, st);
  }
  if (n < 0) { cudaGetLastError(); return fail(MG_ERR_CUDA, n == -2 ? "workspace too small for the kernel's JAMP scratch" : "kernel launch set-up failed"); }
  p->launches = n;
  MG_CUDA(cudaGetLastError());
  return MG_OK;
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
      !(params->gamma_z >= 0) || params->gamma_t != 0.0)
    return MG_ERR_BAD_PARAM;
  // derived couplings (DESIGN.md §3 C2, reading A1)
  const double pi = 3.14159265358979323846;
  const double aew = 1.0 / params->alpha_ew_inv;
  double sw2 = params->sw2;
  if (!(sw2 > 0)) {
    if (!(params->gf > 0)) return MG_ERR_BAD_PARAM;
    const double mz2 = params->mz * params->mz;
    const double rad = mz2 * mz2 / 4 - pi * aew * mz2 / (sqrt(2.0) * params->gf);
    if (!(rad >= 0)) return MG_ERR_BAD_PARAM;
    sw2 = 1.0 - (mz2 / 2 + sqrt(rad)) / mz2;
  }
  if (!(sw2 > 0 && sw2 < 1)) return MG_ERR_BAD_PARAM;
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
  p->desc = d; p->par = *params;
  p->nfinal = d->npar - 2;
  if (cudaDeviceGetAttribute(&p->nsm, cudaDevAttrMultiProcessorCount, params->device) != cudaSuccess) p->nsm = 148;
  for (int i = 0; i < 8; ++i) p->masses[i] = (i < d->npar && d->massive[i]) ? params->mt : 0.0;
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
  const int nhel = d->nhel;
  std::vector<int> all(nhel);
  for (int h = 0; h < nhel; ++h) all[h] = h;
  p->good = all; p->run = all; p->run_w.assign(nhel, 1.0);
  const size_t es = esize(p);
  std::vector<double> ones(nhel > 2 * d->nlane ? nhel : 2 * d->nlane + 1, 1.0);
  std::vector<float> onesf(ones.begin(), ones.end());
  cudaError_t ce = cudaMalloc(&p->stats_dev, sizeof(double) * 2 * nhel);
  if (ce == cudaSuccess) ce = cudaMalloc(&p->wpart_dev, sizeof(double) * 3 * MG_WEIGHT_MAX_BLOCKS);
  if (d->launch) {
    if (ce == cudaSuccess) ce = cudaMalloc(&p->hel_dev, sizeof(int) * nhel);
    if (ce == cudaSuccess) ce = cudaMalloc(&p->hel_all_dev, sizeof(int) * nhel);
    if (ce == cudaSuccess) ce = cudaMalloc(&p->helw_dev, sizeof(double) * nhel);
    if (ce == cudaSuccess) ce = cudaMalloc(&p->ones_dev, sizeof(double) * nhel);
    if (ce == cudaSuccess) ce = cudaMemcpy(p->hel_all_dev, all.data(), sizeof(int) * nhel, cudaMemcpyHostToDevice);
    if (ce == cudaSuccess) ce = cudaMemcpy(p->ones_dev, ones.data(), sizeof(double) * nhel, cudaMemcpyHostToDevice);
  } else {
    if (ce == cudaSuccess) ce = cudaMalloc(&p->lanew_dev, es * 2 * d->nlane);
    if (ce == cudaSuccess) ce = cudaMalloc(&p->lanew_all_dev, es * 2 * d->nlane);
    if (ce == cudaSuccess) ce = cudaMemcpy(p->lanew_all_dev, es == 8 ? (const void*)ones.data() : (const void*)onesf.data(),
                                           es * 2 * d->nlane, cudaMemcpyHostToDevice);
    if (ce == cudaSuccess && d->has_fp32) ce = cudaMalloc(&p->lanew_all32_dev, 4 * 2 * d->nlane);
    if (ce == cudaSuccess && d->has_fp32) ce = cudaMemcpy(p->lanew_all32_dev, onesf.data(), 4 * 2 * d->nlane, cudaMemcpyHostToDevice);
  }
  if (ce != cudaSuccess) { free_all(p); delete p; return cuda_fail(ce, "mg_process_create: device set-up"); }
  { const int rc = upload_helicities(p); if (rc != MG_OK) { free_all(p); delete p; return rc; } }
  if (params->helicity_mode == MG_HEL_ALL) p->probed = true;
  *out = p;
  return MG_OK;
}

int mg_process_destroy(mg_process_t* p) {
  if (!p) return MG_ERR_NULL;
  cudaSetDevice(p->par.device);
  free_all(p);
  if (cudaCtxResetPersistingL2Cache() != cudaSuccess) (void)cudaGetLastError();   // lines of mg_sigma's L2 window (gg -> t t~ g g g)
  delete p;
  return MG_OK;
}

size_t mg_momenta_bytes(const mg_process_t* p, int64_t nevt) {
  if (!p || nevt < 0) return 0;
  const int64_t pages = (nevt + MG_NEPP - 1) / MG_NEPP;
  return (size_t)pages * p->desc->npar * MG_NEPP * 4 * sizeof(double);
}

size_t mg_workspace_bytes(const mg_process_t* p, int64_t nevt) {
  if (!p || nevt < 0 || !p->desc->launch_slots) return 0;
  return ws_need(p, nevt);
}

int mg_set_workspace(mg_process_t* p, void* workspace_dev, size_t bytes) {
  if (!p) return MG_ERR_NULL;
  if ((uintptr_t)workspace_dev & 255) return MG_ERR_ALIGN;
  MG_CUDA(cudaSetDevice(p->par.device));
  if (p->ws && !p->ws_user) { cudaDeviceSynchronize(); cudaFree(p->ws); }
  p->ws = workspace_dev; p->ws_bytes = workspace_dev ? bytes : 0; p->ws_user = workspace_dev != nullptr;
  if (p->ws_user && p->desc->launch_slots && bytes < mg_workspace_bytes(p, 32))
    return fail(MG_ERR_BAD_PARAM, "workspace smaller than mg_workspace_bytes(p, 32)");
  return MG_OK;
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

int mg_sigma_per_helicity(mg_process_t* p, const void* momenta_dev, int64_t nevt, void* perhel_out_dev, void* stream) {
  if (!p || ((!momenta_dev || !perhel_out_dev) && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0) return MG_ERR_BAD_NEVT;
  if (((uintptr_t)momenta_dev & 15) || ((uintptr_t)perhel_out_dev & 7)) return MG_ERR_ALIGN;
  if (nevt == 0) return MG_OK;
  MG_CUDA(cudaSetDevice(p->par.device));
  void* tmp = nullptr;
  MG_CUDA(cudaMalloc(&tmp, esize(p) * (size_t)nevt));
  const int rc = run_sigma(p, momenta_dev, nevt, tmp, perhel_out_dev, true, (cudaStream_t)stream);
  const cudaError_t e = cudaStreamSynchronize((cudaStream_t)stream);
  cudaFree(tmp);
  if (rc != MG_OK) return rc;
  if (e != cudaSuccess) return cuda_fail(e, "sigma_per_helicity");
  return MG_OK;
}

int mg_helicity_probe(mg_process_t* p, const void* momenta_dev, int64_t nprobe, void* stream) {
  if (!p || !momenta_dev) return MG_ERR_NULL;
  if (nprobe <= 0) return MG_ERR_BAD_NEVT;
  if (p->par.helicity_mode == MG_HEL_ALL) return MG_OK;       // MG_HEL_ALL handles always sum every helicity
  const int nhel = p->desc->nhel;
  void* ph = nullptr;
  MG_CUDA(cudaSetDevice(p->par.device));
  MG_CUDA(cudaMalloc(&ph, esize(p) * (size_t)nprobe * nhel));
  int rc = mg_sigma_per_helicity(p, momenta_dev, nprobe, ph, stream);
  std::vector<double> st(2 * nhel, 0.0);
  if (rc == MG_OK) {
    cudaError_t e = mg_launch_probe_stats(p->par.precision, ph, nprobe, nhel, p->stats_dev, (cudaStream_t)stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(st.data(), p->stats_dev, sizeof(double) * 2 * nhel, cudaMemcpyDeviceToHost, (cudaStream_t)stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
    if (e != cudaSuccess) rc = cuda_fail(e, "helicity probe statistics");
  }
  cudaFree(ph);
  if (rc != MG_OK) return rc;
  double tot = 0;
  for (int h = 0; h < nhel; ++h) tot += st[h];
  // reading A6: h is good iff sum_probe ME_h > eps * sum_probe sum_h ME_h
  const double eps = p->par.precision == MG_FP64 ? 1e-14 : 1e-6;
  std::vector<char> isgood(nhel, 0);
  p->good.clear();
  for (int h = 0; h < nhel; ++h) if (st[h] > eps * tot) { isgood[h] = 1; p->good.push_back(h); }
  if (p->good.empty()) for (int h = 0; h < nhel; ++h) { isgood[h] = 1; p->good.push_back(h); }
  // helicity-flip symmetry (parity invariance of QCD: |M(-h)|^2 = |M(h)|^2 event by event): where the probe batch
  // shows it, the mirror hbar = nhel-1-h of a helicity whose top quark has lambda = +1 is not evaluated and h counts
  // twice.  Data driven: e+ e- -> mu+ mu- (Z exchange) does not have it and keeps every good helicity.
  const double sym = p->par.precision == MG_FP64 ? 1e-10 : 1e-4;
  const int tpos = p->desc->npar - 3;
  p->run.clear(); p->run_w.clear();
  for (int h = 0; h < nhel; ++h) {
    if (!isgood[h]) continue;
    const int hb = nhel - 1 - h;
    const bool paired = isgood[hb] && st[nhel + h] <= sym * (st[h] + st[hb]);
    if (paired && !((h >> tpos) & 1)) continue;               // represented by its mirror
    p->run.push_back(h);
    p->run_w.push_back(paired ? 2.0 : 1.0);
  }
  rc = upload_helicities(p);
  if (rc != MG_OK) return rc;
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
  return run_sigma(p, momenta_dev, nevt, me_out_dev, nullptr, false, (cudaStream_t)stream);
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

int mg_sigma_mixed(mg_process_t* p, const void* momenta_dev, int64_t nevt, double* me_out_dev, double tol,
                   float* eps_out_dev, int64_t* nflagged_out, void* stream) {
  if (!p || ((!momenta_dev || !me_out_dev) && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0 || nevt > 0x7fffffff) return MG_ERR_BAD_NEVT;
  if (((uintptr_t)momenta_dev & 15) || ((uintptr_t)me_out_dev & 7) || ((uintptr_t)eps_out_dev & 3)) return MG_ERR_ALIGN;
  if (p->par.precision != MG_FP64 || !p->desc->has_fp32 || !(tol >= 0)) return MG_ERR_BAD_PARAM;
  if (nflagged_out) *nflagged_out = 0;
  if (nevt == 0) return MG_OK;
  const mg_procdesc_t* d = p->desc;
  cudaStream_t st = (cudaStream_t)stream;
  MG_CUDA(cudaSetDevice(p->par.device));
  if (!p->probed) {                        // the fp64 re-evaluation uses the handle's helicity state
    const int rc = mg_helicity_probe(p, momenta_dev, nevt < 4096 ? nevt : 4096, stream);
    if (rc != MG_OK) return rc;
  }
  // scratch: perhel32 [nhel][nevt] | me32 [nevt] | flagged [nevt] + counter | compact momenta | compact |M|^2
  const size_t npad = (size_t)(nevt + 31) / 32 * 32;
  const size_t o_me32 = (size_t)d->nhel * nevt * 4, o_flag = o_me32 + npad * 4, o_cnt = o_flag + npad * 4;
  const size_t o_mom = (o_cnt + 256) / 256 * 256, o_me64 = o_mom + npad * d->npar * 32, need = o_me64 + npad * 8;
  if (p->mx_bytes < need) {
    if (p->mx) { cudaDeviceSynchronize(); cudaFree(p->mx); p->mx = nullptr; p->mx_bytes = 0; }
    MG_CUDA(cudaMalloc(&p->mx, need));
    p->mx_bytes = need;
  }
  char* base = (char*)p->mx;
  float* perhel = (float*)base;
  int* flagged = (int*)(base + o_flag);
  int* cnt = (int*)(base + o_cnt);
  // 1. fp32 pass, every helicity, per-helicity output
  long long n;
  if (d->launch) n = d->launch(MG_FP32, (const double*)momenta_dev, base + o_me32, nevt, p->hel_all_dev, p->ones_dev, d->nhel, perhel, p->pvec, st);
  else {
    { const int rc = ensure_ws(p, nevt); if (rc != MG_OK) return rc; }
    n = d->launch_slots(MG_FP32, (const double*)momenta_dev, base + o_me32, nevt, p->lanew_all32_dev, 2, 0, perhel, p->pvec, p->ws, p->ws_bytes, st);
  }
  if (n < 0) { cudaGetLastError(); return fail(MG_ERR_CUDA, "mg_sigma_mixed: fp32 launch set-up failed"); }
  long long launches = n;
  // 2. per-event precision estimate, fp32 sums, flags
  unsigned massless = 0;
  for (int i = 0; i < d->npar; ++i) if (!d->massive[i]) massless |= 1u << i;
  const double kappa = d->ngluons > 0 ? 0.25 : 0.0;          // the conditioning term is about soft / collinear gluons
  MG_CUDA(mg_launch_mixed_flag(perhel, (const double*)momenta_dev, nevt, d->nhel, d->npar, massless, kappa, tol, me_out_dev,
                               eps_out_dev, flagged, cnt, st));
  int nf = 0;
  MG_CUDA(cudaMemcpyAsync(&nf, cnt, sizeof(int), cudaMemcpyDeviceToHost, st));
  MG_CUDA(cudaStreamSynchronize(st));
  launches += 1;
  // 3. fp64 re-evaluation of the flagged events
  if (nf > 0) {
    double* cmom = (double*)(base + o_mom);
    double* cme = (double*)(base + o_me64);
    MG_CUDA(mg_launch_mixed_gather((const double*)momenta_dev, flagged, nf, d->npar, cmom, st));
    const int rc = run_sigma(p, cmom, nf, cme, nullptr, false, st);
    if (rc != MG_OK) return rc;
    launches += p->launches + 2;
    MG_CUDA(mg_launch_mixed_scatter(cme, flagged, nf, me_out_dev, st));
  }
  p->launches = launches;
  if (nflagged_out) *nflagged_out = nf;
  return MG_OK;
}

int mg_weight_max(mg_process_t* p, void* me_dev, const double* weights_dev, int64_t nevt, double* out_dev, void* stream) {
  if (!p || !out_dev || ((!me_dev || !weights_dev) && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0) return MG_ERR_BAD_NEVT;
  if (((uintptr_t)me_dev & (esize(p) - 1)) || ((uintptr_t)weights_dev & 7) || ((uintptr_t)out_dev & 7)) return MG_ERR_ALIGN;
  MG_CUDA(cudaSetDevice(p->par.device));
  MG_CUDA(mg_launch_weight_max(p->par.precision, me_dev, weights_dev, nevt, p->wpart_dev, out_dev, (cudaStream_t)stream));
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
  memset(o, 0, sizeof *o);
  o->npar = d->npar; o->nfinal = d->npar - 2; o->ndiagrams = d->ndiagrams; o->nhel = d->nhel;
  o->ngoodhel = (int)p->good.size(); o->ncolor = d->ncol; o->denominator = d->denominator; o->nepp = MG_NEPP;
  o->nhel_evaluated = (int)p->run.size();
  // per-slot work (helicity tables) is done once per (event, top helicity) that is run
  const long long nslot = d->launch_slots ? p->ntb : 0;
  o->flops_per_event_allhel = d->flops_algorithmic * d->nhel + d->flops_algorithmic_per_event * (d->launch_slots ? 2 : 0);
  o->flops_per_event_goodhel = d->flops_algorithmic * (long long)p->run.size() + d->flops_algorithmic_per_event * nslot;
  o->flops_executed_per_event_goodhel = d->flops_per_helicity * (long long)p->run.size() + d->flops_per_event * nslot;
  for (int i = 0; i < 8; ++i) o->masses[i] = p->masses[i];
  o->nkernels_per_tile = d->nkernels;
  o->launches_last_sigma = (int32_t)p->launches;
  o->workspace_bytes = (int64_t)p->ws_bytes;
  return MG_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// Several subprocesses behind one handle ("processes with multiple subprocesses, such as p p -> t t~ 0-2 j").
// `p` (beams) and `j` (jets) stand for {g, q, q~, r, r~}; the string is expanded to every combination, jets as a multiset, and
// the combinations for which a subprocess was generated are kept (quark number is conserved by construction: the others
// do not exist).  All subprocesses share npar, hence one momenta buffer.
// ---------------------------------------------------------------------------------------------------------------
struct mg_multi {
  std::vector<mg_process*> sub;
  std::vector<std::string> names;
};

static const mg_procdesc_t* find_desc(const std::string& key) {
  for (int i = 0; i < mg_registry_n; ++i) if (squeeze(mg_registry[i]->proc) == key) return mg_registry[i];
  return nullptr;
}

int mg_multi_create(const char* proc, const mg_params_t* params, mg_multi_t** out) {
  if (!proc || !params || !out) return MG_ERR_NULL;
  std::vector<std::string> ini, fin;
  {
    std::vector<std::string>* cur = &ini;
    std::string tok;
    for (const char* c = proc;; ++c) {
      if (*c == 0 || isspace((unsigned char)*c) || *c == '>') {
        if (!tok.empty()) { cur->push_back(tok); tok.clear(); }
        if (*c == '>') { if (cur == &fin) return MG_ERR_BAD_PROC; cur = &fin; }
        if (*c == 0) break;
      } else tok.push_back(*c);
    }
  }
  if (ini.size() != 2 || fin.size() < 2 || fin.size() > 6) return MG_ERR_BAD_PROC;
  static const char* const parton[5] = {"g", "q", "q~", "r", "r~"};     // q, r: two distinct massless flavours
  constexpr int NP = 5;
  std::vector<int> jets;                           // positions of the j's in the final state
  for (size_t i = 0; i < fin.size(); ++i) if (fin[i] == "j") jets.push_back((int)i);
  const int nj = (int)jets.size();
  int ncomb = 1;
  for (int i = 0; i < nj; ++i) ncomb *= NP;
  mg_multi* m = new mg_multi();
  int rc = MG_OK;
  for (int a = 0; a < NP && rc == MG_OK; ++a) {
    if (ini[0] != "p" && a > 0) break;
    for (int b = 0; b < NP && rc == MG_OK; ++b) {
      if (ini[1] != "p" && b > 0) break;
      for (int c = 0; c < ncomb && rc == MG_OK; ++c) {
        std::vector<std::string> f = fin;
        int r = c;
        for (int i = 0; i < nj; ++i) { f[jets[i]] = parton[r % NP]; r /= NP; }
        std::string name = std::string(ini[0] == "p" ? parton[a] : ini[0].c_str()) + " " +
                           (ini[1] == "p" ? parton[b] : ini[1].c_str()) + " >";
        for (const std::string& t : f) name += " " + t;
        const mg_procdesc_t* d = find_desc(squeeze(name.c_str()));
        if (!d) continue;                          // jets in another order, or no such subprocess
        bool dup = false;
        for (const mg_process* q : m->sub) if (q->desc == d) dup = true;
        if (dup) continue;
        mg_process* h = nullptr;
        rc = mg_process_create(d->proc, params, &h);
        if (rc == MG_OK) { m->sub.push_back(h); m->names.push_back(d->proc); }
      }
    }
  }
  if (rc == MG_OK && m->sub.empty()) rc = MG_ERR_BAD_PROC;
  if (rc != MG_OK) { mg_multi_destroy(m); return rc; }
  *out = m;
  return MG_OK;
}

int mg_multi_destroy(mg_multi_t* m) {
  if (!m) return MG_ERR_NULL;
  for (mg_process* h : m->sub) mg_process_destroy(h);
  delete m;
  return MG_OK;
}

int mg_multi_count(const mg_multi_t* m) { return m ? (int)m->sub.size() : 0; }
const char* mg_multi_name(const mg_multi_t* m, int i) { return (m && i >= 0 && i < (int)m->sub.size()) ? m->names[i].c_str() : nullptr; }
mg_process_t* mg_multi_process(mg_multi_t* m, int i) { return (m && i >= 0 && i < (int)m->sub.size()) ? m->sub[i] : nullptr; }

int mg_multi_sigma(mg_multi_t* m, const void* momenta_dev, int64_t nevt, void* me_out_dev, void* stream) {
  if (!m || ((!momenta_dev || !me_out_dev) && nevt > 0)) return MG_ERR_NULL;
  if (nevt < 0) return MG_ERR_BAD_NEVT;
  for (size_t i = 0; i < m->sub.size(); ++i) {
    char* out = (char*)me_out_dev + i * (size_t)nevt * esize(m->sub[i]);
    const int rc = mg_sigma(m->sub[i], momenta_dev, nevt, out, stream);
    if (rc != MG_OK) return rc;
  }
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
    case MG_ERR_TOO_LARGE: return "size beyond the fixed maximum of a no-allocation entry point";
    default: return "unknown status";
  }
}
const char* mg_last_error(void) { return g_err; }

}  // extern "C"
