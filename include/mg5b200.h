/* mg5b200.h — C ABI of the B200-native matrix-element library (libmg5b200.so).
 *
 * The hot path of arXiv:2312.02898 ("Madgraph5_aMC@NLO on GPUs and vector CPUs"), standalone-program shape
 * (Fig. 1b): a batch of random numbers -> RAMBO phase-space points -> per-event
 * tree-level |M|^2 summed over helicities and colours, evaluated event-parallel on the GPU (PAPER.md:13,
 * :41, :45).  The caller owns batches; the library is a pure function momenta -> |M|^2 (the shape of the
 * Fortran<->CUDA bridge of PAPER.md:67-:89, Fig. 1c).  Processes: the set validated in PAPER.md:139 —
 *     "e+ e- > mu+ mu-", "g g > t t~", "g g > t t~ g", "g g > t t~ g g", "g g > t t~ g g g"
 * (leading order, fixed couplings: PAPER.md:141), and the quark channels of p p > t t~ + 0..2 jets that have one
 * light-quark line ("p p -> t t~ 0-2 j"; q = one massless flavour other than the top):
 *     "q q~ > t t~ [g [g]]", "q~ q > t t~ [g [g]]", "q g > t t~ q [g]", "g q > t t~ q [g]", "q~ g > t t~ q~ [g]",
 *     "g q~ > t t~ q~ [g]", "g g > t t~ q q~";
 * and those with two light-quark lines (r: a second massless flavour; same flavour twice includes the Fermi interference):
 *     "q q~ > t t~ r r~", "q r > t t~ q r", "q r~ > t t~ q r~", "q~ r > t t~ q~ r", "q~ r~ > t t~ q~ r~", "q q~ > t t~ q q~",
 *     "q q > t t~ q q", "q~ q~ > t t~ q~ q~" (+ "q~ q > ...");   several subprocesses behind one handle: mg_multi_* below.
 *
 * Plain C: opaque handle, plain pointers and sizes.  Every `*_dev` pointer is DEVICE memory owned by the
 * caller (the library never frees or reallocates it); `stream` is a cudaStream_t passed as void* (NULL =
 * default stream).  All calls return mg_status_t (0 = OK); none throws, exits or prints.  There is no CPU
 * fallback: without a CUDA device mg_process_create returns MG_ERR_NO_DEVICE.
 *
 * Momenta layout (fixed by this ABI; element type double for both precisions): AoSoA pages of
 * MG_NEPP = 32 events,
 *       mom[page][ipar][ievt_in_page][4],   4-vector order (E, px, py, pz), GeV, metric (+,-,-,-),
 * particles in the order of the process string (initial state first).  nevt need not be a multiple of 32
 * but the buffer must be mg_momenta_bytes(p, nevt) long (whole pages) and 16-byte aligned.
 * Output: me_out[nevt], double (MG_FP64) or float (MG_FP32): spin- and colour-averaged |M|^2 including the
 * 1/k! for k identical final-state gluons (denominators 4, 256, 256, 512, 1536 for the five processes of PAPER.md:139;
 * 36 / 96 / 256 x k! for q q~ / q g / g g beams in the quark channels), in GeV^(-2(npar-4)).
 */
#ifndef MG5B200_H
#define MG5B200_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define MG_NEPP 32

typedef struct mg_process mg_process_t; /* opaque, library-owned */

typedef enum {
  MG_OK = 0,
  MG_ERR_NULL = -1,       /* a required pointer argument is NULL                       */
  MG_ERR_BAD_PROC = -2,   /* process string not one of the generated processes         */
  MG_ERR_BAD_PARAM = -3,  /* struct_size mismatch, unknown precision / helicity mode   */
  MG_ERR_BAD_NEVT = -4,   /* nevt < 0                                                  */
  MG_ERR_ALIGN = -5,      /* a device pointer is not 16-byte aligned                   */
  MG_ERR_KINEMATICS = -6, /* sqrt_s <= sum of final-state masses                       */
  MG_ERR_CUDA = -7,       /* a CUDA call failed; text in mg_last_error()               */
  MG_ERR_NO_DEVICE = -8,  /* no CUDA device / bad ordinal                              */
  MG_ERR_TOO_LARGE = -9   /* beyond the fixed maximum of a no-allocation entry point; text in mg_last_error() */
} mg_status_t;

typedef enum { MG_FP64 = 0, MG_FP32 = 1 } mg_precision_t;
typedef enum {
  MG_HEL_FILTER = 0, /* find the non-vanishing helicities on a probe batch (first mg_sigma call) */
  MG_HEL_ALL = 1     /* always sum all 2^npar helicities                                        */
} mg_helmode_t;

typedef struct {          /* caller-owned, copied by mg_process_create                              */
  uint32_t struct_size;   /* = sizeof(mg_params_t)                                                  */
  int32_t precision;      /* mg_precision_t of the matrix-element kernels (RAMBO is always fp64)    */
  int32_t helicity_mode;  /* mg_helmode_t                                                           */
  int32_t device;         /* CUDA ordinal                                                           */
  double alpha_s;         /* 0.118, fixed                                            */
  double alpha_ew_inv;    /* 132.507                                                                */
  double gf;              /* 1.16639e-5 GeV^-2; only used to derive sw2 when sw2 <= 0               */
  double sw2;             /* > 0 overrides the derived sin^2(theta_W)                               */
  double mz, gamma_z;     /* 91.188, 2.4414                                                         */
  double mt, gamma_t;     /* 173.0; gamma_t must be 0 (external on-shell tops; reading A2)*/
} mg_params_t;

typedef struct {
  int32_t npar, nfinal, ndiagrams, nhel, ngoodhel, ncolor, denominator, nepp;
  int64_t flops_per_event_allhel;  /* generator's static FLOP count (FMA = 2) with all 2^npar helicities evaluated: */
                                   /* the method's own (algorithmic) count — every current computed once per        */
                                   /* helicity, the tabled low-multiplicity currents once per event                 */
  int64_t flops_per_event_goodhel; /* same for the helicities evaluated now (nhel_evaluated)                        */
  double masses[8];                /* per particle, process order                                                   */
  int32_t nkernels_per_tile;       /* kernel launches mg_sigma makes per event tile (1 = fused kernel)              */
  int32_t launches_last_sigma;     /* kernels launched by the last mg_sigma call on this handle                     */
  int64_t workspace_bytes;         /* workspace currently attached (library-owned or caller-provided)               */
  int64_t flops_executed_per_event_goodhel; /* FLOPs the kernels execute, including the currents that diagram      */
                                   /* groups recompute (>= flops_per_event_goodhel)                                 */
  int32_t nhel_evaluated;          /* helicities evaluated per event: a good helicity whose helicity-flipped mirror */
                                   /* has the same |M_h|^2 on the probe batch is evaluated once and counted twice   */
  int32_t reserved;
} mg_info_t;

/* Fills *params with the defaults of BASELINE.json's configs (fp64, helicity filter, device 0). */
int mg_params_default(mg_params_t* params);

/* Creates the process object: parses `proc` (MG5 syntax, whitespace-insensitive), copies `params`,
 * selects the generated kernel set, uploads constants.  PAPER.md:45 (per-process generated code). */
int mg_process_create(const char* proc, const mg_params_t* params, mg_process_t** out);
int mg_process_destroy(mg_process_t* p);

/* K1+K2: device Philox4x32-10 + RAMBO (PAPER.md:39 Fig. 1b, :47).  Writes nevt phase-space points for the
 * process (beams along +-z with energy sqrt_s/2, final state flat in n-body phase space, massive tops put
 * on shell by the RAMBO rescaling) into momenta_dev (layout above).  Random stream: Philox key = seed,
 * counter = (global event index, final-particle index), so event i is the same for any batch split.
 * Asynchronous on `stream`. */
int mg_rambo(mg_process_t* p, uint64_t seed, double sqrt_s, int64_t nevt, void* momenta_dev, void* stream);
/* Same, for events [first_event, first_event + nevt) of the stream, optionally with RAMBO weights
 * (weights_dev may be NULL; double[nevt]; phase-space weight without the (2 pi)^(4-3n) factor). */
int mg_rambo_ex(mg_process_t* p, uint64_t seed, double sqrt_s, int64_t first_event, int64_t nevt,
                void* momenta_dev, double* weights_dev, void* stream);

/* K1 alone (diagnostic / bit-exact test entry): the raw Philox4x32-10 words RAMBO consumes,
 * out_dev[(ievt * nfinal + ifinal) * 4 + m], uint32, 16-byte aligned.  Asynchronous on `stream`. */
int mg_philox_raw(mg_process_t* p, uint64_t seed, int64_t first_event, int64_t nevt, uint32_t* out_dev, void* stream);

/* K3..K7: |M|^2 for nevt events.  momenta_dev: layout above; me_out_dev: nevt doubles (MG_FP64) or floats
 * (MG_FP32).  Asynchronous on `stream`, except that in MG_HEL_FILTER mode the first call runs the
 * helicity probe (K8) on the first min(nevt, 4096) events and synchronises the stream once, and that the
 * processes with >= 24 colour flows use a workspace (per-event invariants of one event tile + the L2-resident JAMP
 * scratch of the resident CTAs): library-owned by default — at most 1 GiB, larger batches are processed in event
 * tiles; (re)allocated, synchronously, by the first call that needs a bigger one — or caller-provided
 * (mg_set_workspace).  One handle serves one stream at a time: the workspace and the helicity lists belong to the
 * handle, so calls on the same handle must be ordered by the caller (distinct handles are independent).
 * Device-state side effect (g g > t t~ g g g only, scratch 108 MB): for the duration of its launches the call puts an
 * L2 access-policy window (the JAMP part of the scratch persisting) on `stream` and raises the device limit
 * cudaLimitPersistingL2CacheSize to min(73 MB, device maximum); the window is removed from the stream before the call
 * returns, the limit stays, mg_process_destroy resets the persisting lines. */
int mg_sigma(mg_process_t* p, const void* momenta_dev, int64_t nevt, void* me_out_dev, void* stream);

/* Caller-provided workspace: `workspace_dev` (256-byte aligned device memory, `bytes` long) replaces
 * the library-owned one; the library never frees it; NULL returns to the library-owned workspace.
 * mg_workspace_bytes(p, nevt) is the size with which a batch of nevt events runs as one tile (0 for the processes
 * that need none); anything >= mg_workspace_bytes(p, 32) works (smaller tiles).  MG_ERR_BAD_PARAM if too small. */
int mg_set_workspace(mg_process_t* p, void* workspace_dev, size_t bytes);
size_t mg_workspace_bytes(const mg_process_t* p, int64_t nevt);

/* Batch-unweighting primitive (PAPER.md:99-:103, Table 2 :119-:127: "weights from Jacobian terms and PDFs are
 * transferred to the GPU, and multiplied with the matrix elements that are already in GPU memory ... The maximum of
 * these weights is computed in parallel"): me_dev[i] <- weights_dev[i] * me_dev[i] in place (me_dev: the output of
 * mg_sigma, element type of the handle's precision; weights_dev: nevt doubles) and
 *     out_dev[0] = max_i, out_dev[1] = sum_i, out_dev[2] = sum_i of squares        of the products (doubles).
 * Fixed reduction tree: results are bit-reproducible.  nevt = 0 gives (-inf, 0, 0).  Asynchronous on `stream`. */
int mg_weight_max(mg_process_t* p, void* me_dev, const double* weights_dev, int64_t nevt, double* out_dev, void* stream);

/* The same primitive for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): no handle (mg_process_create allocates), no cudaMalloc / cudaFree / allocating
 * library call.  The first reduction stage's partial results live in a fixed 24 KiB __device__ array inside the library
 * (every GPU that loads the library holds it until the process exits), hence the limit
 *     nevt <= MG_NOALLOC_MAX_EVENTS = 8 388 608;   beyond it: MG_ERR_TOO_LARGE, nothing is launched.
 * precision: mg_precision_t of me_dev's elements; runs on the CURRENT device (the first call on a device looks up the
 * array's device address, nothing else is set up); arguments, results and reduction tree as mg_weight_max — both give
 * bit-identical results.  All calls on one device share the scratch array: calls that overlap on the GPU (different
 * streams, concurrently replayed graphs) race on it and must be serialised by the caller; calls on one stream are safe.
 * Asynchronous on `stream`. */
#define MG_NOALLOC_MAX_EVENTS 8388608LL
int mg_weight_max_noalloc(int precision, void* me_dev, const double* weights_dev, int64_t nevt, double* out_dev,
                          void* stream);

/* Same from HOST buffers (momenta_host: layout above, me_out_host: nevt elements; pinned memory recommended): copies
 * in, runs, copies out and synchronises.  The device staging buffers belong to the handle, grow on demand and are
 * freed by mg_process_destroy.  This is the end-to-end entry point bench.py times as `e2e`. */
int mg_sigma_host(mg_process_t* p, const void* momenta_host, int64_t nevt, void* me_out_host, void* stream);

/* K8: explicit helicity probe on nprobe events; sets the good-helicity list (h is good iff its share of the summed
 * |M|^2 of the probe batch exceeds 1e-14, 1e-6 in fp32) and finds the helicities whose helicity-flipped mirror has
 * the same |M_h|^2 on every probe event (parity invariance of QCD; not e+ e- -> mu+ mu-): those are evaluated once
 * and counted twice.  The statistics are reduced on the device; synchronises.  A no-op on MG_HEL_ALL handles. */
int mg_helicity_probe(mg_process_t* p, const void* momenta_dev, int64_t nprobe, void* stream);
/* Per-helicity |M_h|^2 (already divided by the denominator), all 2^npar helicities:
 * perhel_out_dev[h * nevt + ievt].  Diagnostic / test entry point. */
int mg_sigma_per_helicity(mg_process_t* p, const void* momenta_dev, int64_t nevt, void* perhel_out_dev,
                          void* stream);
/* Mixed precision with precision tracking ("tracking the precision of the matrix elements
 * showed that single-precision computations are not accurate enough"): on an MG_FP64 handle of a process that has fp32
 * kernels (all but g g > t t~ g g g), evaluates every helicity in fp32, measures per event
 *     eps = sum over mirror pairs | |M_h|^2 - |M_hbar|^2 | / sum_h |M_h|^2  +  2^-26 s / (2 min_ij |p_i.p_j|)
 * (hbar = all helicities flipped: the first term is zero in exact arithmetic, i.e. it measures the event's fp32
 * arithmetic error; the second, over pairs of massless legs of the gluon processes, covers the rounding of the inputs
 * the two mirrors share, which grows with the event's conditioning), and re-evaluates in fp64 the events with
 * eps > tol (or a non-finite value).  me_out_dev: nevt doubles (fp32 sums for the
 * events kept, fp64 values for the re-evaluated ones); eps_out_dev: NULL or nevt floats; *nflagged_out (host, may be
 * NULL): number of re-evaluated events.  Synchronises the stream once (the count).  MG_ERR_BAD_PARAM on an MG_FP32
 * handle, a process without fp32 kernels, or tol < 0. */
int mg_sigma_mixed(mg_process_t* p, const void* momenta_dev, int64_t nevt, double* me_out_dev, double tol,
                   float* eps_out_dev, int64_t* nflagged_out, void* stream);

/* Copies the current good-helicity list (indices; bit (npar-1-i) set <=> particle i has lambda=+1). */
int mg_good_helicities(const mg_process_t* p, int32_t* out, int32_t capacity, int32_t* ngood);

/* Several subprocesses behind one handle ("Processes with multiple subprocesses, such as
 * proton-proton collisions p p -> t t~ 0-2 j ... are being tested").  `proc` may use the multi-particle labels p (beams)
 * and j (jets) = {g, q, q~, r, r~} (q, r: two distinct massless quark flavours other than the top), e.g. "p p > t t~ j":
 * it is expanded to every combination and the combinations for which a subprocess was generated are kept — the gluon
 * channels g g > t t~ (g (g)), the 15 subprocesses with one light-quark line (q q~ > t t~ g, q g > t t~ q, ...,
 * g g > t t~ q q~) and the 10 two-jet subprocesses with two light-quark lines (q q~ > t t~ r r~, q r > t t~ q r,
 * q r~ > t t~ q r~, q~ r > t t~ q~ r, q~ r~ > t t~ q~ r~, q q~ > t t~ q q~, q q > t t~ q q, q~ q~ > t t~ q~ q~, and the two
 * with q~ q beams).  Matrix elements do not depend on which flavours q and r are; one generated function per distinct
 * particle order (e.g. "r q > t t~ r q" is "q r > t t~ q r" with the momenta of the beams and of the jets exchanged and is
 * not generated separately).  mg_multi_name lists what the handle holds.  MG_ERR_BAD_PROC if nothing matches.
 * mg_multi_sigma: |M|^2 of every subprocess on the SAME nevt momenta (all share npar and the momenta layout);
 * me_out_dev[isub * nevt + ievt], element type of the precision.  PDFs and the sum over subprocesses stay with the caller
 * (host side).  mg_multi_process returns the borrowed single-subprocess handle (owned by the multi handle)
 * for mg_rambo, mg_process_info, mg_helicity_probe etc.  Same stream / ordering rules as mg_sigma. */
typedef struct mg_multi mg_multi_t;
int mg_multi_create(const char* proc, const mg_params_t* params, mg_multi_t** out);
int mg_multi_destroy(mg_multi_t* m);
int mg_multi_count(const mg_multi_t* m);
const char* mg_multi_name(const mg_multi_t* m, int isub);
mg_process_t* mg_multi_process(mg_multi_t* m, int isub);
int mg_multi_sigma(mg_multi_t* m, const void* momenta_dev, int64_t nevt, void* me_out_dev, void* stream);

int mg_process_info(const mg_process_t* p, mg_info_t* out);
size_t mg_momenta_bytes(const mg_process_t* p, int64_t nevt);

const char* mg_status_string(int status);
const char* mg_last_error(void); /* thread-local detail of the last MG_ERR_CUDA */

#ifdef __cplusplus
}
#endif
#endif
