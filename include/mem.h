/* include/mem.h -- C ABI of the B200-native matrix-element-method integrator.
 *
 * One call estimates, for every measured event, the MEM likelihood of
 * arXiv 1407.7595 (PAPER.md:45 Eq. 1, :49 Eq. 2, :56 Eq. 3)
 *
 *     p = int sum_flav |M|^2(Y) f1(x1) f2(x2) / (|q1||q2|) T(X;Y) dPhi_n
 *
 * by Monte Carlo (PAPER.md:76 Eq. 5, :80 Eq. 6): sampling, variable maps,
 * matrix element, toy PDFs, jet transfer functions, phase-space Jacobian, the
 * reduction to (mean, standard error) and the optional per-event VEGAS grid
 * refinement all run in sm_100a CUDA kernels.  There is no
 * CPU fallback: every entry point that needs the device fails with
 * MEM_ERR_CUDA when no CUDA device is usable.
 *
 * Conventions: natural units, GeV, metric (+,-,-,-).  "device" pointers are
 * CUDA device pointers valid on the current device, 8-byte aligned; "host"
 * pointers are ordinary process memory.  The library never frees, reallocates
 * or retains caller buffers.  All functions return a mem_status and never
 * throw or abort; mem_last_error() gives a thread-local message for the last
 * failure on the calling thread.  A handle must not be used from two threads
 * at once; distinct handles are independent.  One handle may be used from
 * several CUDA streams in turn: its workspace is shared by consecutive calls,
 * so every call first makes its stream wait (on the device, without blocking
 * the host) for the previous call on that handle, and a workspace growth step
 * waits for it on the host before freeing anything.  The exception is a call
 * made while its stream is being captured into a CUDA graph: no cross-stream
 * ordering is recorded then, and the caller owns the handle exclusively for
 * as long as the graph is replayed.
 */
#ifndef MEM_B200_H
#define MEM_B200_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mem_handle mem_handle; /* opaque; owned by the library */

typedef enum {
  MEM_OK = 0,
  MEM_ERR_INVALID_ARG = 1, /* null / negative / misaligned / out-of-range argument */
  MEM_ERR_UNSUPPORTED = 2, /* valid request this build does not implement */
  MEM_ERR_CUDA = 3,        /* CUDA runtime error (message in mem_last_error) */
  MEM_ERR_NOMEM = 4        /* workspace allocation failed */
} mem_status;

/* Process hypotheses = BASELINE.json:configs[0..3]. */
typedef enum {
  MEM_PROC_W_ENU = 1,    /* u dbar -> W+ -> e+ nu,            D = 1,  5 record fields */
  MEM_PROC_Z_BB = 2,     /* q qbar -> Z -> b bbar,            D = 2,  6 record fields */
  MEM_PROC_TT_LJETS = 3, /* t tbar -> b l nu bbar q qbar',    D = 6, 17 record fields */
  MEM_PROC_TT_DILEP = 4, /* t tbar -> b l+ nu bbar l- nubar,  D = 8, 14 record fields */
  /* NEXT-4, the paper's own benchmark integral (PAPER.md:101-109 Eq. 7, :111-118 Eq. 8, :120-137 Eq. 9, :178-180
   * Eq. 11): t tbar H(-> b bbar), both tops leptonic, four b jets.  Record = (pT, eta, phi) of l+ and l-, then
   * (E, eta, phi) of the jets taken as b (pairs with l+), bbar (pairs with l-), b1, b2 (Higgs candidates); no MET
   * field: Eq. 11 defines the neutrinos' total transverse momentum from the partons of each point.  Dimensions:
   * E_b, E_bbar, the Breit-Wigner mapped s_W+, s_t, s_W-, s_tbar, and Eq. 9's (m_H^2, f = E1 + E2) with both
   * orderings of its inverse summed.  mem_params.tth_hyp selects the hypothesis of Eq. 10. */
  MEM_PROC_TTH_DILEP = 5 /* t tbar H -> b l+ nu bbar l- nubar b bbar, D = 8, 18 record fields */
} mem_process;

/* All physics constants, integration windows and VEGAS options (DESIGN.md
 * "Readings" O4-O8, A13, A14).  Size-prefixed POD: set struct_size =
 * sizeof(mem_params); mem_params_default() fills every field. */
typedef struct mem_params {
  uint32_t struct_size;
  uint32_t precision;   /* 64, or 32 (fp32 integrand core; MEM_PROC_TT_LJETS only, reading A15) */
  double sqrt_s;        /* pp centre-of-mass energy */
  double G_F, m_W, Gam_W, m_Z, Gam_Z, sin2_thw, m_t, Gam_t, alpha_s, V_ud, V_tb;
  double pdf_A_q, pdf_A_g, pdf_pow_x, pdf_pow_1mx; /* toy PDF f(x) = A x^pow_x (1-x)^pow_1mx */
  double tf_w_tail, tf_mu1, tf_sig1, tf_mu2, tf_sig2; /* double-Gaussian jet TF, fractions of parton E; the core must not be
                                                       * so much narrower than the tail that exp(z1^2 - z2^2) overflows inside
                                                       * the energy window (sigma1 >~ 0.03 for the defaults): INVALID_ARG */
  double jetE_rlo, jetE_rhi; /* parton-energy window, fractions of the measured jet energy */
  double bw_nwidths;         /* Breit-Wigner windows m +- n Gamma */
  double nu_pz_max;          /* config 1: |nu_z| <= nu_pz_max */
  double nu_eta_max;         /* config 3: |eta_nu| <= nu_eta_max */
  double met_sigma, met_nsigma; /* config 4: Gaussian MET TF, flat +-n sigma sampling */
  double vegas_alpha;        /* grid damping exponent */
  int64_t vegas_points;      /* points per adaptation pass */
  int32_t vegas_iters;       /* adaptation passes; 0 = plain Monte Carlo */
  int32_t vegas_bins;        /* bins per dimension, 1..64 */
  int32_t n_flav;            /* light flavours summed in the initial state */
  int32_t n_perm;            /* jet-parton assignments summed per point (Eq. 7 "sum over all
                              * permutations of assigning measured jets to partons"): 0 or 1 = record order only;
                              * MEM_PROC_TT_LJETS: 4 = b-tags known (b jets swapped x light jets swapped), 24 = all;
                              * MEM_PROC_TT_DILEP: 2 = both b assignments; MEM_PROC_TTH_DILEP: 12 = the 4!/2
                              * distinct assignments of four b jets to (b, bbar, {b1, b2}).
                              * Anything else: MEM_ERR_INVALID_ARG. */
  /* NEXT-4 (MEM_PROC_TTH_DILEP only; readings A20, A21) */
  double m_H, Gam_H;         /* Higgs mass and width: Breit-Wigner map of Eq. 9's m_H^2, window m +- n Gamma */
  double yuk_t, yuk_b;       /* Yukawa couplings of the factorised t tbar H matrix element */
  int32_t tth_hyp;           /* hypothesis of Eq. 10: 0 = t tbar H(-> b bbar), 1 = non-resonant t tbar b bbar stand-in */
  int32_t reserved0;         /* must be 0 */
} mem_params;

/* Fill *params with the defaults of `process` (precision 64, plain MC). */
mem_status mem_params_default(mem_process process, mem_params* params /* host, out */);

/* Record fields per event (5 / 6 / 17 / 14 / 18) and integration dimensions (1 / 2 / 6 / 8 / 8);
 * -1 for an unknown process. */
int32_t mem_event_fields(mem_process process);
int32_t mem_n_dims(mem_process process);

/* Create an integrator for one process hypothesis on the current CUDA device.
 * params (host) is copied; NULL = defaults.  *out receives the handle. */
mem_status mem_create(mem_process process, const mem_params* params, mem_handle** out);

/* Free the handle and its workspace (synchronises the handle's device, whichever device is current). NULL is a no-op. */
mem_status mem_destroy(mem_handle* h);

/* Multi-GPU sharding: the event index that enters the
 * Philox counter is first_event + local index, so a contiguous shard of a
 * larger list reproduces the unsharded result bit for bit.  Default 0. */
mem_status mem_set_event_offset(mem_handle* h, uint64_t first_event);

/* The hot path.  For each event e in [0, n_events):
 *   w_i = integrand at the point drawn from Philox4x32-10 with key = seed and
 *         counter = (point i, first_event + e, pass, word block),  i in [0, n_points)
 *   out_p[e]   = (1/N) sum w_i
 *   out_err[e] = sqrt(max(0, (sum w_i^2)/N - out_p[e]^2) / (N - 1))
 * With params.vegas_iters > 0 each event first runs vegas_iters adaptation
 * passes of vegas_points points that refine its own importance-sampling grid;
 * the outputs then come from the final pass of n_points only.
 *
 * events : device, float64, SoA field-major [mem_event_fields][n_events]; read-only
 * out_p, out_err : device, float64 [n_events]; overwritten
 * cuda_stream : a cudaStream_t (NULL = legacy default stream).  All work is
 *   enqueued on it and the call returns without synchronising.  The handle's
 *   workspace grows on demand (a growth step synchronises that stream and waits for
 *   the handle's previous call); once a call of the same size has run, further calls
 *   allocate nothing and may be captured into a CUDA graph on a capturing stream and
 *   replayed (mem_last_pass_ms does not see captured calls).
 * n_events == 0 is MEM_OK with no launch; n_points < 2 is MEM_ERR_INVALID_ARG; so is a call made while
 * another CUDA device than the handle's is current.
 * A call that fails after it has started launching (MEM_ERR_NOMEM or MEM_ERR_CUDA between two passes) leaves
 * out_p / out_err undefined but the handle usable: the next call on it first resets the workspace's block arrival
 * counters on its stream.  After a sticky CUDA error (every later CUDA call fails too) destroy the handle.
 * Kinematically forbidden or non-finite points contribute w = 0 and still count in N. */
mem_status mem_integrate(mem_handle* h, const double* events, int64_t n_events,
                         int64_t n_points, uint64_t seed,
                         double* out_p, double* out_err, void* cuda_stream);

/* Same computation through host buffers: copies `events` host->device, runs
 * mem_integrate, copies the two result arrays device->host, all on cuda_stream,
 * and synchronises that stream before returning (other streams keep running).
 * Pinned host buffers make the copies asynchronous with respect to other streams.
 * This is the end-to-end entry the benchmark's "e2e" figure times. */
mem_status mem_integrate_host(mem_handle* h, const double* events_host, int64_t n_events,
                              int64_t n_points, uint64_t seed,
                              double* out_p_host, double* out_err_host, void* cuda_stream);

/* mem_integrate for callers that must not allocate device memory.
 *
 * mem_integrate keeps its intermediate arrays (per-event constants, per-block partial sums, block arrival counters)
 * in a workspace it obtains with cudaMalloc and regrows with cudaFree + cudaMalloc whenever a call is larger than
 * any before it.  Some hosts cannot live with that: an online event filter or another real-time loop whose device
 * memory was divided up once at start-up and where a later driver allocation may fail or stall; a host application
 * whose own memory pool has already claimed the whole GPU; any loop in which the device-wide synchronisation that
 * cudaFree / cudaMalloc imply would stall work queued on other streams.  For them this entry point computes the same
 * plain Monte Carlo estimate (Eq. 5-6; same kernels, same launch geometry, same Philox counters, hence
 * the same bits in out_p and out_err as mem_integrate) with the intermediate arrays laid out in ONE array of
 * MEM_NOALLOC_SCRATCH_BYTES bytes that is part of the library image: every GPU on which the library gets loaded
 * holds those bytes from then until the process exits, whether or not this function is ever called.  The call makes
 * no cudaMalloc, cudaFree or other allocating call; the caller passes inputs and outputs exactly as to mem_integrate.
 *
 * Limits and rules:
 *  - plain Monte Carlo only: a handle created with vegas_iters > 0 gets MEM_ERR_UNSUPPORTED (the VEGAS grids and
 *    histograms are not part of the fixed array);
 *  - the call needs  r256(4 n_events) + r256(8 K n_perm n_events) + 16 n_events n_chunks  bytes, r256 = rounded up
 *    to 256, K = 16 / 12 / 44 / 64 / 80 constants per event for processes 1..5, n_perm = max(1, params.n_perm),
 *    n_chunks = blocks per event (64 at 2^20 points, 16 to 32 below 2^18).  More than MEM_NOALLOC_SCRATCH_BYTES is
 *    MEM_ERR_INVALID_ARG, with both numbers in mem_last_error(), before anything is launched: split the event list
 *    (with mem_set_event_offset the pieces reproduce the whole list bit for bit).  The headline workload, 4096
 *    t tbar l+jets events x 2^20 points, needs 5.4 MiB;
 *  - the first call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *    current) and keeps it for the life of the process.  Make that first call during set-up, outside any CUDA
 *    stream capture;
 *  - every call on a device, from every handle, stream and host thread, uses the same array, which still holds what
 *    the previous call left there: each call zeroes the arrival counters on `cuda_stream` before its kernels and
 *    overwrites the rest before reading it.  Two such calls that overlap on the GPU (different streams with no
 *    dependency between them) corrupt each other's results; keeping them ordered is up to the caller.  Calls of
 *    mem_integrate are not affected: they never touch this array;
 *  - mem_last_pass_ms does not see these calls.
 * Arguments, error codes, asynchrony on cuda_stream and the n_events == 0 case are those of mem_integrate. */
#define MEM_NOALLOC_SCRATCH_BYTES (8u << 20)
mem_status mem_integrate_noalloc(mem_handle* h, const double* events, int64_t n_events,
                                 int64_t n_points, uint64_t seed,
                                 double* out_p, double* out_err, void* cuda_stream);

/* Diagnostic for the parity tests: the individual weights w_i of one event,
 * i in [first_point, first_point + n), for Philox pass `iteration`.
 * grid (device, may be NULL): VEGAS edges [D][vegas_bins + 1] of THIS event;
 * when given, the unit-cube point is warped through it and w includes the
 * grid Jacobian.  out_w: device, float64 [n]. */
mem_status mem_eval_points(mem_handle* h, const double* events, int64_t n_events, int64_t event,
                           int64_t first_point, int64_t n, uint64_t seed, int32_t iteration,
                           const double* grid, double* out_w, void* cuda_stream);

/* Grid PDFs (NEXT-3; "stored in (x, Q^2) grids for each parton flavor ... bilinear interpolation
 * within the kernel", listing PAPER.md:274-306 Fig. A.5).  Replaces the toy PDF of this handle by tables:
 * table : host, float64 [6][nq][nx]: species 0 = gluon, 1..5 = d, u, s, c, b (antiquark = quark); sample
 *         (iq, ix) at ln Q = lqmin + iq (lqmax - lqmin)/nq, ln x = lxmin + ix (lxmax - lxmin)/nx (the listing's
 *         step); copied, the caller keeps ownership.  NULL switches back to the toy PDF.
 * Q     : the fixed factorisation scale (BASELINE: "at fixed Q"); the ln Q direction of the bilinear formula is
 *         folded into one row per species here, the kernels interpolate in ln x; cell indices are clamped to
 *         [0, n - 2] as in the listing, so points outside the grid extrapolate the edge cell.
 * The flavour sum of t tbar production becomes f_g f_g |M_gg|^2 + sum over the first n_flav quark species of
 * 2 f_q f_q |M_qq|^2.  MEM_PROC_TT_LJETS / MEM_PROC_TT_DILEP with precision 64 only (MEM_ERR_UNSUPPORTED
 * otherwise).  Synchronises the whole device first (work in flight on any stream may still read the
 * table being replaced), then copies synchronously. */
mem_status mem_set_pdf_grid(mem_handle* h, const double* table, int32_t nx, int32_t nq, double lxmin, double lxmax,
                            double lqmin, double lqmax, double Q);

/* Parton-level mode (NEXT-2; Table 2): the transfer functions are delta
 * functions and nothing is integrated.  For each fully specified partonic configuration
 *   out_w[e] = sum over the handle's n_perm jet-parton assignments and the initial-state flavours of
 *              f(x1) f(x2) / (|q1||q2|) * |M|^2(l, nu, b_had, b_lep, q, qbar')
 * i.e. the integrand of PAPER.md:45 Eq. 1 without dPhi (transverse boost O7 applied, propagators
 * from the momenta; kinematically forbidden configurations give 0).
 * momenta : device, float64, SoA field-major [24][n_events] = (E, px, py, pz) of l, nu, b_had, b_lep,
 *           q, qbar' (t = b_lep + l + nu, tbar = b_had + q + qbar'); read-only
 * out_w   : device, float64 [n_events]; overwritten.  Asynchronous on cuda_stream.
 * MEM_PROC_TT_LJETS handles with precision 64 only (MEM_ERR_UNSUPPORTED otherwise). */
mem_status mem_eval_parton(mem_handle* h, const double* momenta, int64_t n_events, double* out_w,
                           void* cuda_stream);

/* Post-processing of the likelihoods (PAPER.md:45 Eq. 1 "sigma is the overall normalization", :143 Eq. 10
 * "D = log10(p_ttH / p_ttbb)"; reading A22).
 * mem_normalisation: sigma = (1/n) sum_e p[e] / g[e], the importance-sampled acceptance integral of the
 *   likelihood over events drawn from the density g (one fixed-order reduction, result reproducible).
 *   p, g : device, float64 [n], read-only;  out_sigma : device, float64 [1].
 * mem_discriminant: out_D[e] = log10((p_sig[e] / sigma_sig[0]) / (p_bkg[e] / sigma_bkg[0])).
 *   p_sig, p_bkg : device, float64 [n];  sigma_sig, sigma_bkg : device, float64 [1];  out_D : device [n].
 * Both are asynchronous on cuda_stream, need no handle and never synchronise.  n < 1 (normalisation) or
 * n < 0 (discriminant), NULL or misaligned pointers: MEM_ERR_INVALID_ARG. */
mem_status mem_normalisation(const double* p, const double* g, int64_t n, double* out_sigma, void* cuda_stream);
mem_status mem_discriminant(const double* p_sig, const double* p_bkg, int64_t n, const double* sigma_sig,
                            const double* sigma_bkg, double* out_D, void* cuda_stream);

/* Diagnostic: copy the VEGAS grids left by the last mem_integrate with
 * vegas_iters > 0 into out_grid (device, float64 [n_events][D][vegas_bins+1]). */
mem_status mem_get_grid(mem_handle* h, int64_t n_events, double* out_grid, void* cuda_stream);

/* Kernels launched by this handle since creation (for the benchmark's launch count). */
int64_t mem_launch_count(const mem_handle* h);

/* Measurement support.  Every mem_integrate records CUDA events on
 * its stream around the dominant kernel, i.e. the integrate pass that produces the outputs.
 * mem_last_pass_ms waits for that pass and returns its duration in *ms (host, out) and the
 * number of integrand evaluations it made in *evals (host, out; may be NULL).  A call captured into a CUDA
 * graph records no events: after it mem_last_pass_ms returns MEM_ERR_INVALID_ARG until an eager call has run. */
mem_status mem_last_pass_ms(mem_handle* h, double* ms, int64_t* evals);

/* FP64 FMA peak of the current device, measured with independent DFMA chains on all SMs:
 * *tflops (host, out) = 2 * fused multiply-adds / second / 1e12, best of `repeats` launches.
 * The denominator of the "alu" roofline (MEASURED_PEAKS.json has no FP64 figure). */
mem_status mem_measure_fp64_peak(int32_t repeats, double* tflops, void* cuda_stream);

/* Thread-local description of the last error on this thread ("" if none). */
const char* mem_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MEM_B200_H */
