// mem_api.cu -- the C ABI of include/mem.h: argument checks, workspace, kernel launches.
// No arithmetic of the method lives here beyond turning mem_params into DevConst.
#include "../../include/mem.h"
#include "../../include/mem_bench.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <type_traits>

#include "mem_kernels.cuh"
#include "mem_parton.cuh"

using namespace memb200;

namespace {

thread_local char g_err[512] = "";

mem_status fail(mem_status s, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return s;
}

#define CUDA_TRY(expr)                                                                      \
  do {                                                                                      \
    cudaError_t _e = (expr);                                                                \
    if (_e != cudaSuccess)                                                                  \
      return fail(_e == cudaErrorMemoryAllocation ? MEM_ERR_NOMEM : MEM_ERR_CUDA, "%s: %s", \
                  #expr, cudaGetErrorString(_e));                                           \
  } while (0)

int n_fields_of(int process) {
  switch (process) {
    case MEM_PROC_W_ENU: return 5;
    case MEM_PROC_Z_BB: return 6;
    case MEM_PROC_TT_LJETS: return 17;
    case MEM_PROC_TT_DILEP: return 14;
    case MEM_PROC_TTH_DILEP: return 18;
  }
  return -1;
}
int n_dims_of(int process) {
  switch (process) {
    case MEM_PROC_W_ENU: return 1;
    case MEM_PROC_Z_BB: return 2;
    case MEM_PROC_TT_LJETS: return 6;
    case MEM_PROC_TT_DILEP: return 8;
    case MEM_PROC_TTH_DILEP: return 8;
  }
  return -1;
}
int n_consts_of(int process) {
  switch (process) {
    case MEM_PROC_W_ENU: return ProcWenu::NC;
    case MEM_PROC_Z_BB: return ProcZbb::NC;
    case MEM_PROC_TT_LJETS: return ProcTTljets::NC;
    case MEM_PROC_TT_DILEP: return ProcTTdilep::NC;
    case MEM_PROC_TTH_DILEP: return ProcTTHdilep::NC;
  }
  return -1;
}

struct Buffer {
  void* p = nullptr;
  size_t cap = 0;
};

}  // namespace

struct mem_handle {
  int process;
  int device;
  mem_params params;
  DevConst dc;
  DevConstF dcf;            // fp32 mirror of dc for precision = 32 (reading A15)
  uint64_t event_offset;
  int64_t launches;
  int64_t grid_events;      // events covered by the grids of the last VEGAS call
  Buffer ecs, partials, grids, hist, stage_in, stage_out, pdf_tab, tickets;
  cudaEvent_t ev_begin, ev_end;  // around the dominant kernel of the last mem_integrate
  cudaEvent_t ev_done;           // recorded after the last launch of every call that uses the workspace
  bool has_done;                 // ev_done has been recorded at least once
  bool tickets_dirty;            // a mem_integrate on this handle returned an error after it had started launching
  int64_t last_evals;            // integrand evaluations of that kernel; 0 = none yet
};

namespace {

// Grow-only workspace.  A growth step frees the old allocation, so it first waits for every kernel that may still
// read it: the last call on this handle (whatever stream it ran on) and the current stream.
mem_status ensure(mem_handle* h, Buffer& b, size_t bytes, cudaStream_t st) {
  if (bytes <= b.cap) return MEM_OK;
  if (b.p) {
    if (h->has_done) CUDA_TRY(cudaEventSynchronize(h->ev_done));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaFree(b.p));
    b.p = nullptr; b.cap = 0;
  }
  size_t want = bytes + bytes / 4;
  cudaError_t e = cudaMalloc(&b.p, want);
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    want = bytes;
    e = cudaMalloc(&b.p, want);
  }
  if (e != cudaSuccess) {
    (void)cudaGetLastError();
    b.p = nullptr;
    return fail(MEM_ERR_NOMEM, "cudaMalloc(%zu bytes): %s", want, cudaGetErrorString(e));
  }
  b.cap = want;
  return MEM_OK;
}

// Every entry point that launches on a handle: the current device must be the handle's.
mem_status check_device(const mem_handle* h) {
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev != h->device)
    return fail(MEM_ERR_INVALID_ARG, "handle was created on device %d, the current device is %d", h->device, dev);
  return MEM_OK;
}
// ... and the event index must fit the 32-bit Philox counter word
mem_status check_counter(const mem_handle* h, int64_t n_events) {
  if (h->event_offset + (uint64_t)n_events > 0x100000000ULL)
    return fail(MEM_ERR_INVALID_ARG, "event index exceeds the 32-bit Philox counter word");
  return MEM_OK;
}

// One handle, several streams: the workspace (per-event constants, partial sums, grids, histograms) is shared by
// consecutive calls, so a call first makes its stream wait for the previous call on this handle (a no-op when that
// ran on the same stream) and leaves an event behind for the next one.  While the stream is being captured into a
// CUDA graph neither is done (events recorded outside a capture cannot be waited on inside it): the caller then owns
// the handle exclusively for the lifetime of the graph.
mem_status begin_call(mem_handle* h, cudaStream_t st, bool* capturing) {
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  CUDA_TRY(cudaStreamIsCapturing(st, &cs));
  *capturing = cs != cudaStreamCaptureStatusNone;
  if (!*capturing && h->has_done) CUDA_TRY(cudaStreamWaitEvent(st, h->ev_done, 0));
  return MEM_OK;
}
mem_status end_call(mem_handle* h, cudaStream_t st, bool capturing) {
  if (capturing) return MEM_OK;
  CUDA_TRY(cudaEventRecord(h->ev_done, st));
  h->has_done = true;
  return MEM_OK;
}

// flavours in the paper's order (d, u, s, c, b); L = T3 - Q sin^2, R = -Q sin^2 (O8)
void z_coupling_sums(const mem_params& p, double* cu, double* ct) {
  const double Lb = -0.5 + p.sin2_thw / 3.0, Rb = p.sin2_thw / 3.0;
  double su = 0.0, st = 0.0;
  for (int f = 0; f < p.n_flav; ++f) {
    const bool up = (f == 1 || f == 3);
    const double T3 = up ? 0.5 : -0.5, Q = up ? 2.0 / 3.0 : -1.0 / 3.0;
    const double L = T3 - Q * p.sin2_thw, R = -Q * p.sin2_thw;
    su += L * L * Lb * Lb + R * R * Rb * Rb;
    st += L * L * Rb * Rb + R * R * Lb * Lb;
  }
  *cu = su; *ct = st;
}

void bw_window(double m, double G, double n, double* t_lo, double* dt) {
  const double lo = std::atan(((m - n * G) * (m - n * G) - m * m) / (m * G));
  const double hi = std::atan(((m + n * G) * (m + n * G) - m * m) / (m * G));
  *t_lo = lo; *dt = hi - lo;
}

DevConst make_dev_const(const mem_params& p) {
  DevConst c;
  std::memset(&c, 0, sizeof(c));
  c.sqrt_s = p.sqrt_s; c.inv_sqrt_s = 1.0 / p.sqrt_s; c.S = p.sqrt_s * p.sqrt_s; c.inv_S = 1.0 / c.S;
  c.pdf_pow_x = p.pdf_pow_x; c.pdf_pow_1mx = p.pdf_pow_1mx;
  c.pdf_fast = (p.pdf_pow_x == -0.5 && p.pdf_pow_1mx == 3.0) ? 1 : 0;
  c.n_flav = p.n_flav;
  c.A_q2 = p.pdf_A_q * p.pdf_A_q; c.A_g2 = p.pdf_A_g * p.pdf_A_g;
  c.rlo = p.jetE_rlo; c.dr = p.jetE_rhi - p.jetE_rlo;
  const double r2 = std::sqrt(2.0), r2pi = std::sqrt(2.0 * kPi);
  c.tf_a1 = 1.0 / (p.tf_sig1 * r2); c.tf_b1 = -(1.0 + p.tf_mu1) / (p.tf_sig1 * r2);
  c.tf_a2 = 1.0 / (p.tf_sig2 * r2); c.tf_b2 = -(1.0 + p.tf_mu2) / (p.tf_sig2 * r2);
  c.tf_c1 = (1.0 - p.tf_w_tail) / (p.tf_sig1 * r2pi); c.tf_c2 = p.tf_w_tail / (p.tf_sig2 * r2pi);
  c.tf_q2 = (c.tf_a1 - c.tf_a2) * (c.tf_a1 + c.tf_a2); c.tf_q1 = 2.0 * (c.tf_a1 * c.tf_b1 - c.tf_a2 * c.tf_b2);
  c.tf_q0 = (c.tf_b1 - c.tf_b2) * (c.tf_b1 + c.tf_b2);
  c.mW = p.m_W; c.GW = p.Gam_W; c.mW2 = p.m_W * p.m_W; c.mWGW = p.m_W * p.Gam_W; c.mWGW2 = c.mWGW * c.mWGW;
  bw_window(p.m_W, p.Gam_W, p.bw_nwidths, &c.tW_lo, &c.tW_dt);
  c.mt2 = p.m_t * p.m_t; c.mtGt = p.m_t * p.Gam_t; c.mtGt2 = c.mtGt * c.mtGt;
  bw_window(p.m_t, p.Gam_t, p.bw_nwidths, &c.tT_lo, &c.tT_dt);
  c.mZ2 = p.m_Z * p.m_Z; c.mZGZ2 = p.m_Z * p.m_Z * p.Gam_Z * p.Gam_Z;
  const double g2 = 4.0 * r2 * p.G_F * p.m_W * p.m_W, gz2 = 4.0 * r2 * p.G_F * p.m_Z * p.m_Z;
  const double gs2 = 4.0 * kPi * p.alpha_s;
  c.g4w = g2 * g2; c.gz4 = gz2 * gz2; c.gs4 = gs2 * gs2;
  c.V_ud2 = p.V_ud * p.V_ud; c.V_tb2 = p.V_tb * p.V_tb;
  z_coupling_sums(p, &c.z_cu, &c.z_ct);
  c.nu_pz_max = p.nu_pz_max; c.nu_eta_max = p.nu_eta_max;
  c.met_sigma = p.met_sigma; c.met_nsigma = p.met_nsigma;
  c.vegas_bins = p.vegas_bins; c.vegas_alpha = p.vegas_alpha;
  c.n_perm = p.n_perm > 1 ? p.n_perm : 1;
  // NEXT-4 (mem_tth.cuh; readings A20, A21)
  c.rhi = p.jetE_rhi; c.lnr = 2.0 * std::log(p.jetE_rhi / p.jetE_rlo);
  c.mH2 = p.m_H * p.m_H; c.mHGH = p.m_H * p.Gam_H;
  bw_window(p.m_H, p.Gam_H, p.bw_nwidths, &c.tH_lo, &c.tH_dt);
  c.tth_hyp = p.tth_hyp;
  // hypothesis 0: dt_H (ds/dt D_H = 1/(m_H Gam_H)) y_t^2 4 m_t^2 (eikonal scalar emission) 3 y_b^2 2 (H -> b bbar; k^2 stays);
  // hypothesis 1: ln(s_hi/s_lo) (ds/du = s ln) g_s^2 (eikonal vector emission) (1/k^4) g_s^2 k^2 (splitting) -> constant
  c.tth_c = p.tth_hyp ? c.lnr * gs2 * gs2
                      : c.tH_dt / c.mHGH * (p.yuk_t * p.yuk_t * 4.0 * p.m_t * p.m_t) * (3.0 * p.yuk_b * p.yuk_b * 2.0);
  c.pdf_tab = nullptr; c.pdf_nx = 0; c.pdf_lxmin = c.pdf_dx = c.pdf_inv_dx = 0.0;
  return c;
}

DevConstF to_float(const DevConst& d) {
  DevConstF f;
#define CP(x) f.x = (float)d.x
  CP(sqrt_s); CP(inv_sqrt_s); CP(S); CP(inv_S); CP(pdf_pow_x); CP(pdf_pow_1mx); CP(A_q2); CP(A_g2); CP(rlo); CP(dr);
  CP(tf_a1); CP(tf_b1); CP(tf_c1); CP(tf_a2); CP(tf_b2); CP(tf_c2); CP(tf_q2); CP(tf_q1); CP(tf_q0); CP(mW); CP(GW); CP(mW2); CP(mWGW); CP(mWGW2);
  CP(tW_lo); CP(tW_dt); CP(mt2); CP(mtGt); CP(mtGt2); CP(tT_lo); CP(tT_dt); CP(mZ2); CP(mZGZ2); CP(g4w); CP(gz4);
  CP(gs4); CP(V_ud2); CP(V_tb2); CP(z_cu); CP(z_ct); CP(nu_pz_max); CP(nu_eta_max); CP(met_sigma); CP(met_nsigma);
  CP(vegas_alpha); CP(rhi); CP(mH2); CP(mHGH); CP(tH_lo); CP(tH_dt); CP(lnr); CP(tth_c);
#undef CP
  f.tth_hyp = d.tth_hyp;
  f.pdf_fast = d.pdf_fast; f.n_flav = d.n_flav; f.vegas_bins = d.vegas_bins; f.n_perm = d.n_perm;
  f.pdf_tab = nullptr; f.pdf_nx = 0; f.pdf_lxmin = f.pdf_dx = f.pdf_inv_dx = 0.0;      // grid PDFs are fp64 only
  return f;
}

template <typename T> const DevConstR<T>& dc_of(const mem_handle* h);
template <> const DevConstR<double>& dc_of<double>(const mem_handle* h) { return h->dc; }
template <> const DevConstR<float>& dc_of<float>(const mem_handle* h) { return h->dcf; }

mem_status check_params(int process, const mem_params& p) {
  if (p.struct_size != sizeof(mem_params))
    return fail(MEM_ERR_INVALID_ARG, "mem_params.struct_size = %u, expected %zu", p.struct_size, sizeof(mem_params));
  if (p.precision != 64 && p.precision != 32) return fail(MEM_ERR_INVALID_ARG, "precision must be 64 or 32");
  if (p.reserved0 != 0) return fail(MEM_ERR_INVALID_ARG, "mem_params.reserved0 must be 0");
  if (p.precision == 32 && process != MEM_PROC_TT_LJETS)
    return fail(MEM_ERR_UNSUPPORTED, "precision 32 is implemented for MEM_PROC_TT_LJETS only (reading A15)");
  const bool pos = p.sqrt_s > 0 && p.G_F > 0 && p.m_W > 0 && p.Gam_W > 0 && p.m_Z > 0 && p.Gam_Z > 0 && p.m_t > 0 &&
                   p.Gam_t > 0 && p.alpha_s > 0 && p.tf_sig1 > 0 && p.tf_sig2 > 0 && p.jetE_rlo > 0 &&
                   p.jetE_rhi > p.jetE_rlo && p.bw_nwidths > 0 && p.nu_pz_max > 0 && p.nu_eta_max > 0 &&
                   p.met_sigma > 0 && p.met_nsigma > 0;
  if (!pos) return fail(MEM_ERR_INVALID_ARG, "mem_params: a constant that must be positive is not");
  if (!(p.tf_w_tail >= 0.0 && p.tf_w_tail <= 1.0)) return fail(MEM_ERR_INVALID_ARG, "tf_w_tail outside [0,1]");
  if (p.nu_eta_max > 50.0) return fail(MEM_ERR_INVALID_ARG, "nu_eta_max above 50");
  if (p.precision == 32 && p.nu_eta_max > 20.0)
    return fail(MEM_ERR_INVALID_ARG, "nu_eta_max above 20 with precision 32 (e^(2 eta) leaves the fp32 range)");
  if (process != MEM_PROC_W_ENU) {
    // The kernels write E T = exp(-z1^2) (c1 + c2 exp(z1^2 - z2^2)) (mem_common.cuh: tf_accum); z1^2 - z2^2 must
    // stay inside the range of exp over the parton-energy window, i.e. the core Gaussian must not be
    // absurdly narrower than the tail one (sigma1 >~ 0.03 for the default window).
    const double r2 = std::sqrt(2.0);
    const double a1 = 1.0 / (p.tf_sig1 * r2), b1 = -(1.0 + p.tf_mu1) * a1, a2 = 1.0 / (p.tf_sig2 * r2), b2 = -(1.0 + p.tf_mu2) * a2;
    auto g = [&](double v) { return (a1 * v + b1) * (a1 * v + b1) - (a2 * v + b2) * (a2 * v + b2); };
    const double v_lo = 1.0 / p.jetE_rhi, v_hi = 1.0 / p.jetE_rlo;
    double gmax = std::fmax(g(v_lo), g(v_hi));
    if (a1 * a1 != a2 * a2) {
      const double v = -(a1 * b1 - a2 * b2) / (a1 * a1 - a2 * a2);
      if (v > v_lo && v < v_hi) gmax = std::fmax(gmax, g(v));
    }
    if (!(gmax < 600.0))
      return fail(MEM_ERR_INVALID_ARG, "jet TF: core Gaussian too narrow for the parton-energy window (z1^2 - z2^2 reaches %.0f)", gmax);
    // the kernels' inner exponentials (exp_tab<false>, no range check) see z1^2 - z2^2: bounded above by gmax and
    // below by -max z2^2; the outer exponential exp(-sum z1^2 ...) is range checked (it may legitimately underflow)
    const double z2max = std::fmax(std::fabs(a2 * v_lo + b2), std::fabs(a2 * v_hi + b2));
    if (!(z2max * z2max < 600.0))
      return fail(MEM_ERR_INVALID_ARG, "jet TF: tail Gaussian too narrow for the parton-energy window (z2^2 reaches %.0f)", z2max * z2max);
  }
  if (p.n_flav < 1 || p.n_flav > 5) return fail(MEM_ERR_INVALID_ARG, "n_flav outside 1..5");
  if (p.bw_nwidths * p.Gam_W >= p.m_W || p.bw_nwidths * p.Gam_t >= p.m_t)
    return fail(MEM_ERR_INVALID_ARG, "bw_nwidths * Gamma must stay below the mass");
  if (process == MEM_PROC_TTH_DILEP) {
    if (!(p.m_H > 0 && p.Gam_H > 0 && p.yuk_t > 0 && p.yuk_b > 0)) return fail(MEM_ERR_INVALID_ARG, "m_H, Gam_H, yuk_t, yuk_b must be positive");
    if (p.bw_nwidths * p.Gam_H >= p.m_H) return fail(MEM_ERR_INVALID_ARG, "bw_nwidths * Gam_H must stay below m_H");
    if (p.tth_hyp != 0 && p.tth_hyp != 1) return fail(MEM_ERR_INVALID_ARG, "tth_hyp must be 0 or 1");
  }
  if (p.vegas_iters < 0 || p.vegas_iters > 255) return fail(MEM_ERR_INVALID_ARG, "vegas_iters outside 0..255");
  if (p.vegas_iters > 0) {
    if (p.vegas_bins < 1 || p.vegas_bins > kMaxBins) return fail(MEM_ERR_INVALID_ARG, "vegas_bins outside 1..%d", kMaxBins);
    if (p.vegas_points < 2) return fail(MEM_ERR_INVALID_ARG, "vegas_points < 2");
    if (!(p.vegas_alpha >= 0.0)) return fail(MEM_ERR_INVALID_ARG, "vegas_alpha < 0");
  }
  const bool perm_ok = p.n_perm == 0 || p.n_perm == 1 ||
                       (process == MEM_PROC_TT_LJETS && (p.n_perm == 4 || p.n_perm == 24)) ||
                       (process == MEM_PROC_TT_DILEP && p.n_perm == 2) ||
                       (process == MEM_PROC_TTH_DILEP && p.n_perm == 12);
  if (!perm_ok) return fail(MEM_ERR_INVALID_ARG, "n_perm = %d is not defined for process %d", p.n_perm, process);
  return MEM_OK;
}

bool aligned8(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 7u) == 0; }

size_t integrate_smem(int NC, int D, int B, int mode) {   // NC = constants per event (all assignments)
  size_t n = (size_t)NC + 2 * kWarps;
  if (mode != MODE_PLAIN) n += (size_t)D * (B + 1);
  if (mode == MODE_ADAPT) {
    const size_t wh = (size_t)kWarps * D * B, scratch = (size_t)D * (3 * kMaxBins + 2);   // the refinement reuses the histograms' space
    n += wh > scratch ? wh : scratch;
  }
  return n * sizeof(double);
}

template <class P>
mem_status launch_prepare(mem_handle* h, const double* events, int64_t n_events, cudaStream_t st) {
  const int64_t n_rec = n_events * h->dc.n_perm;            // one block of NC constants per (event, assignment)
  mem_status s = ensure(h, h->ecs, (size_t)n_rec * P::NC * sizeof(double), st);
  if (s != MEM_OK) return s;
  const int threads = 128;
  prepare_kernel<P><<<(unsigned)((n_rec + threads - 1) / threads), threads, 0, st>>>(
      h->dc, events, n_events, (double*)h->ecs.p);
  ++h->launches;
  CUDA_TRY(cudaGetLastError());
  return MEM_OK;
}

template <class P, int MODE>
mem_status launch_pass(mem_handle* h, int64_t n_events, int64_t n_points, int64_t chunk, int n_chunks,
                       uint64_t seed, uint32_t pass, cudaStream_t st, double* out_p = nullptr, double* out_err = nullptr) {
  const int64_t blocks = n_events * n_chunks;
  if (blocks > 0x7fffffffLL) return fail(MEM_ERR_INVALID_ARG, "n_events * chunks = %lld exceeds the grid limit", (long long)blocks);
  // lane-compacting kernels keep (classes + 1) queues of 64 32-bit point offsets per warp, plus their counters
  size_t smem = integrate_smem(P::NC * h->dc.n_perm, P::D, h->dc.vegas_bins, MODE);
  if constexpr (P::kCompact) {
    if (MODE == MODE_PLAIN) smem += (size_t)kWarps * (P::kClasses + P::kPreStages) * 64 * sizeof(uint32_t);
  }
  auto launch = [&](auto perm, auto grid) {
    integrate_kernel<P, MODE, decltype(perm)::value, decltype(grid)::value><<<(unsigned)blocks, kThreads, smem, st>>>(
        dc_of<typename P::real>(h), (const double*)h->ecs.p, (double*)h->grids.p, (double*)h->partials.p,
        (double*)h->hist.p, n_points, chunk, n_chunks, make_philox(seed), h->event_offset, pass,
        (unsigned*)h->tickets.p, out_p, out_err);
  };
  const bool perm = h->dc.n_perm > 1, grid = h->dc.pdf_tab != nullptr;
  if (perm && grid) launch(std::true_type{}, std::true_type{});
  else if (perm) launch(std::true_type{}, std::false_type{});
  else if (grid) launch(std::false_type{}, std::true_type{});
  else launch(std::false_type{}, std::false_type{});
  ++h->launches;
  CUDA_TRY(cudaGetLastError());
  return MEM_OK;
}

// Points per (event, chunk) block of the pass that produces the outputs: kChunk, or less for short
// integrations so that a few events still fill the GPU (config 1: 64 events x 2^16 points -> 2048 blocks of 2^11).  A
// function of n_points alone -- never of the number of events -- so that the reduction order, and
// with it every bit of the result, is the same however the event list is sharded.
// (Measured and dropped: persistent blocks walking the items round-robin -- 7 to 15 % slower on every config, the
// hardware block scheduler balances better; 32 chunks for every size -- config 4 loses 1.7 %.)
// compact = the staged lane-compacting loop of the conic-solver processes: every queue ends a chunk with a partial
// batch, so a warp should see many points (2^16 per block, at least 4 chunks per event).
int64_t chunk_for(int64_t n_points, bool compact = false) {
  if (compact) {
    int64_t c = 4 * kChunk;
    while (c > 1024 && c * 4 > n_points) c >>= 1;
    return c;
  }
  int64_t c = kChunk;
  const int64_t min_chunks = n_points < (1 << 18) ? 32 : 16;
  while (c > 1024 && c * min_chunks > n_points) c >>= 1;
  return c;
}

// the pass that produces the outputs, bracketed by the handle's events
template <class P, int MODE>
mem_status launch_timed_pass(mem_handle* h, int64_t n_events, int64_t n_points, int n_chunks, uint64_t seed,
                             uint32_t pass, cudaStream_t st, bool capturing, double* out_p, double* out_err) {
  // no event records inside a stream capture: they would belong to the graph and mem_last_pass_ms could not read them
  if (!capturing) CUDA_TRY(cudaEventRecord(h->ev_begin, st));
  mem_status s = launch_pass<P, MODE>(h, n_events, n_points, chunk_for(n_points, P::kCompact && MODE == MODE_PLAIN && h->dc.n_perm <= 1), n_chunks, seed, pass, st, out_p, out_err);
  if (s != MEM_OK) return s;
  if (!capturing) CUDA_TRY(cudaEventRecord(h->ev_end, st));
  h->last_evals = capturing ? 0 : n_events * n_points;
  return MEM_OK;
}

// the launches of one mem_integrate, between begin_call and end_call
template <class P>
mem_status integrate_launches(mem_handle* h, const double* events, int64_t n_events, int64_t n_points, uint64_t seed,
                              double* out_p, double* out_err, cudaStream_t st, bool capturing) {
  mem_status s = launch_prepare<P>(h, events, n_events, st);
  if (s != MEM_OK) return s;
  const int64_t chunk = chunk_for(n_points, P::kCompact && h->params.vegas_iters == 0 && h->dc.n_perm <= 1);
  const int n_chunks = (int)((n_points + chunk - 1) / chunk);
  s = ensure(h, h->partials, (size_t)n_events * n_chunks * 2 * sizeof(double), st);
  if (s != MEM_OK) return s;
  // arrival counters of the "last block of an event finishes it" step: zero when allocated, reset by the last block
  if ((size_t)n_events * sizeof(unsigned) > h->tickets.cap) {
    s = ensure(h, h->tickets, (size_t)n_events * sizeof(unsigned), st);
    if (s != MEM_OK) return s;
    CUDA_TRY(cudaMemsetAsync(h->tickets.p, 0, h->tickets.cap, st));
  }
  const mem_params& p = h->params;
  if (p.vegas_iters > 0) {
    const int D = P::D, B = p.vegas_bins;
    // adaptation passes: at most kMaxAdaptChunks blocks per event, chunk a multiple of kThreads
    int64_t a_chunk = (p.vegas_points + kMaxAdaptChunks - 1) / kMaxAdaptChunks;
    if (a_chunk < chunk_for(p.vegas_points)) a_chunk = chunk_for(p.vegas_points);
    a_chunk = (a_chunk + kThreads - 1) / kThreads * kThreads;
    const int a_chunks = (int)((p.vegas_points + a_chunk - 1) / a_chunk);
    s = ensure(h, h->grids, (size_t)n_events * D * (B + 1) * sizeof(double), st);
    if (s != MEM_OK) return s;
    s = ensure(h, h->hist, (size_t)n_events * a_chunks * D * B * sizeof(double), st);
    if (s != MEM_OK) return s;
    if (a_chunks > n_chunks) {
      s = ensure(h, h->partials, (size_t)n_events * a_chunks * 2 * sizeof(double), st);
      if (s != MEM_OK) return s;
    }
    // each adaptation pass refines the grids itself (last block per event); the first starts from the uniform grid
    for (int it = 0; it < p.vegas_iters; ++it) {
      s = launch_pass<P, MODE_ADAPT>(h, n_events, p.vegas_points, a_chunk, a_chunks, seed, (uint32_t)it, st);
      if (s != MEM_OK) return s;
    }
    h->grid_events = n_events;
    s = launch_timed_pass<P, MODE_GRID>(h, n_events, n_points, n_chunks, seed, (uint32_t)p.vegas_iters, st, capturing, out_p, out_err);
  } else {
    s = launch_timed_pass<P, MODE_PLAIN>(h, n_events, n_points, n_chunks, seed, 0u, st, capturing, out_p, out_err);
  }
  return s;
}

// The arrival counters are zero between calls only because every pass runs to its end (the last block of an event
// resets its counter).  A call that returns an error part-way (an allocation or a launch refused between two VEGAS
// passes, a launch failure) may leave some of them counting, and a later pass would then finish events early from
// partial sums not yet written, or never.  So a failed call marks the handle; the next call zeroes the counters on its
// stream before it launches anything.  A failed call also leaves its event behind, so that the next call is still
// ordered after whatever did get launched.  (After a sticky CUDA error nothing helps: destroy the handle.)
template <class P>
mem_status integrate_impl(mem_handle* h, const double* events, int64_t n_events, int64_t n_points, uint64_t seed,
                          double* out_p, double* out_err, cudaStream_t st) {
  bool capturing = false;
  mem_status s = begin_call(h, st, &capturing);
  if (s != MEM_OK) return s;
  if (h->tickets_dirty && h->tickets.p) CUDA_TRY(cudaMemsetAsync(h->tickets.p, 0, h->tickets.cap, st));
  h->tickets_dirty = true;
  s = integrate_launches<P>(h, events, n_events, n_points, seed, out_p, out_err, st, capturing);
  if (s != MEM_OK) {
    char keep[sizeof(g_err)];
    std::memcpy(keep, g_err, sizeof(keep));            // end_call may overwrite the message of the real failure
    (void)end_call(h, st, capturing);
    std::memcpy(g_err, keep, sizeof(keep));
    return s;
  }
  h->tickets_dirty = false;
  return end_call(h, st, capturing);
}

template <class P>
mem_status eval_impl(mem_handle* h, const double* events, int64_t n_events, int64_t event, int64_t first,
                     int64_t n, uint64_t seed, int32_t iteration, const double* grid, double* out_w,
                     cudaStream_t st) {
  bool capturing = false;
  mem_status s = begin_call(h, st, &capturing);
  if (s != MEM_OK) return s;
  s = launch_prepare<P>(h, events, n_events, st);
  if (s != MEM_OK) return s;
  const int threads = 128;
  const size_t smem = ((size_t)P::NC * h->dc.n_perm + (size_t)P::D * (kMaxBins + 1)) * sizeof(double);
  eval_points_kernel<P><<<(unsigned)((n + threads - 1) / threads), threads, smem, st>>>(
      dc_of<typename P::real>(h), (const double*)h->ecs.p, event, grid, first, n, make_philox(seed), h->event_offset, (uint32_t)iteration, out_w);
  ++h->launches;
  CUDA_TRY(cudaGetLastError());
  return end_call(h, st, capturing);
}

}  // namespace

// ---- mem_integrate_noalloc (include/mem.h): the plain Monte Carlo path with its intermediate arrays in a fixed array ----
//
// For hosts that cannot let a library allocate device memory after start-up (a real-time event filter with a fixed
// memory plan, an application whose own pool owns the GPU, a loop that cannot afford the device-wide stall of
// cudaFree / cudaMalloc).  The array below is part of the library's device image: each GPU that loads the library
// holds MEM_NOALLOC_SCRATCH_BYTES for it until the process ends.
//
// In host code the name `g_noalloc_scratch` is only a host-side handle for the symbol -- not an address a kernel can
// use -- so the device address is asked for once per device (cudaGetSymbolAddress with that device current) and it
// is that address, never the name, that is handed to the kernels.
static __device__ __align__(256) unsigned char g_noalloc_scratch[MEM_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
unsigned char* g_noalloc_addr[kNoallocMaxDevices] = {};

// Device address of the array on device `dev`, which must be the current device (the callers have run check_device).
mem_status noalloc_scratch(int dev, unsigned char** out) {
  if (dev < 0 || dev >= kNoallocMaxDevices)
    return fail(MEM_ERR_UNSUPPORTED, "mem_integrate_noalloc: device %d is outside the %d devices it keeps an address for", dev, kNoallocMaxDevices);
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_addr[dev]) {
    void* p = nullptr;
    CUDA_TRY(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255u) != 0)
      return fail(MEM_ERR_CUDA, "cudaGetSymbolAddress(g_noalloc_scratch) returned %p", p);
    g_noalloc_addr[dev] = static_cast<unsigned char*>(p);
  }
  *out = g_noalloc_addr[dev];
  return MEM_OK;
}

size_t round256(size_t b) { return (b + 255u) & ~(size_t)255u; }

// prepare_kernel + the plain-MC integrate_kernel of mem_integrate, same geometry, workspace = slices of the fixed array:
//   [ tickets: n_events x u32 | ecs: n_events x n_perm x NC f64 | partials: n_events x n_chunks x 2 f64 ]
template <class P>
mem_status integrate_noalloc_impl(mem_handle* h, const double* events, int64_t n_events, int64_t n_points,
                                  uint64_t seed, double* out_p, double* out_err, cudaStream_t st) {
  const int n_perm = h->dc.n_perm;
  const int64_t chunk = chunk_for(n_points, P::kCompact && n_perm <= 1);
  const int64_t n_chunks = (n_points + chunk - 1) / chunk;
  // sizes first, in floating point so that no product can wrap, then the exact integers
  if ((double)n_events * (double)n_chunks > (double)0x7fffffffLL)
    return fail(MEM_ERR_INVALID_ARG, "n_events * chunks exceeds the grid limit");
  const int64_t blocks = n_events * n_chunks;
  const size_t b_tickets = round256((size_t)n_events * sizeof(unsigned));
  const size_t b_ecs = round256((size_t)n_events * (size_t)n_perm * P::NC * sizeof(double));
  const size_t b_partials = (size_t)blocks * 2 * sizeof(double);
  const size_t need = b_tickets + b_ecs + b_partials;
  if (need > (size_t)MEM_NOALLOC_SCRATCH_BYTES)
    return fail(MEM_ERR_INVALID_ARG,
                "mem_integrate_noalloc: %lld events x %lld points need %zu bytes of scratch, the fixed array has %zu; "
                "split the event list (mem_set_event_offset keeps the pieces bit-identical to the whole)",
                (long long)n_events, (long long)n_points, need, (size_t)MEM_NOALLOC_SCRATCH_BYTES);
  unsigned char* base = nullptr;
  mem_status s = noalloc_scratch(h->device, &base);
  if (s != MEM_OK) return s;
  unsigned* tickets = reinterpret_cast<unsigned*>(base);
  double* ecs = reinterpret_cast<double*>(base + b_tickets);
  double* partials = reinterpret_cast<double*>(base + b_tickets + b_ecs);
  // the array keeps whatever the last call (or a failed one) left: the arrival counters must start at zero; the
  // constants and partial sums are written by this call's kernels before they are read
  CUDA_TRY(cudaMemsetAsync(tickets, 0, b_tickets, st));
  const int64_t n_rec = n_events * n_perm;
  prepare_kernel<P><<<(unsigned)((n_rec + 127) / 128), 128, 0, st>>>(h->dc, events, n_events, ecs);
  ++h->launches;
  CUDA_TRY(cudaGetLastError());
  size_t smem = integrate_smem(P::NC * n_perm, P::D, h->dc.vegas_bins, MODE_PLAIN);
  if constexpr (P::kCompact) smem += (size_t)kWarps * (P::kClasses + P::kPreStages) * 64 * sizeof(uint32_t);
  auto launch = [&](auto perm, auto grid) {
    integrate_kernel<P, MODE_PLAIN, decltype(perm)::value, decltype(grid)::value><<<(unsigned)blocks, kThreads, smem, st>>>(
        dc_of<typename P::real>(h), ecs, nullptr, partials, nullptr, n_points, chunk, (int)n_chunks,
        make_philox(seed), h->event_offset, 0u, tickets, out_p, out_err);
  };
  const bool perm = n_perm > 1, grid = h->dc.pdf_tab != nullptr;
  if (perm && grid) launch(std::true_type{}, std::true_type{});
  else if (perm) launch(std::true_type{}, std::false_type{});
  else if (grid) launch(std::false_type{}, std::true_type{});
  else launch(std::false_type{}, std::false_type{});
  ++h->launches;
  CUDA_TRY(cudaGetLastError());
  return MEM_OK;
}

}  // namespace

extern "C" {

const char* mem_last_error(void) { return g_err; }

int32_t mem_event_fields(mem_process process) { return n_fields_of((int)process); }
int32_t mem_n_dims(mem_process process) { return n_dims_of((int)process); }

mem_status mem_params_default(mem_process process, mem_params* p) {
  if (!p) return fail(MEM_ERR_INVALID_ARG, "params is NULL");
  if (n_fields_of((int)process) < 0) return fail(MEM_ERR_INVALID_ARG, "unknown process %d", (int)process);
  std::memset(p, 0, sizeof(*p));
  p->struct_size = (uint32_t)sizeof(mem_params);
  p->precision = 64;
  p->sqrt_s = 14000.0;                                       // BASELINE.json:configs[0]
  p->G_F = 1.16637e-5; p->m_W = 80.4; p->Gam_W = 2.09;       // configs[0]
  p->m_Z = 91.1876; p->Gam_Z = 2.4952; p->sin2_thw = 0.2312;
  p->m_t = 173.0; p->Gam_t = 1.4;                            // configs[2]
  p->alpha_s = 0.118; p->V_ud = 1.0; p->V_tb = 1.0;
  p->pdf_A_q = 1.0; p->pdf_A_g = 1.0; p->pdf_pow_x = -0.5; p->pdf_pow_1mx = 3.0;   // configs[0]
  p->tf_w_tail = 0.3; p->tf_mu1 = 0.0; p->tf_sig1 = 0.15; p->tf_mu2 = -0.1; p->tf_sig2 = 0.35;  // configs[1]
  p->jetE_rlo = 0.5; p->jetE_rhi = 2.0; p->bw_nwidths = 15.0;
  p->nu_pz_max = 500.0;                                      // configs[0]
  p->nu_eta_max = 5.0; p->met_sigma = 10.0; p->met_nsigma = 4.0;
  p->vegas_alpha = 0.5; p->vegas_points = 1 << 17; p->vegas_iters = 0; p->vegas_bins = 50;      // configs[4]
  p->n_flav = (process == MEM_PROC_Z_BB) ? 3 : 5;            // configs[1]
  // NEXT-4 (reading A21; the paper gives none): m_H = 125, Gamma_H = 4.07 MeV, y_f = m_f sqrt(2 sqrt2 G_F), m_b = 4.18
  p->m_H = 125.0; p->Gam_H = 0.00407;
  p->yuk_t = p->m_t * std::sqrt(2.0 * std::sqrt(2.0) * p->G_F);
  p->yuk_b = 4.18 * std::sqrt(2.0 * std::sqrt(2.0) * p->G_F);
  p->tth_hyp = 0;
  return MEM_OK;
}

mem_status mem_create(mem_process process, const mem_params* params, mem_handle** out) {
  if (!out) return fail(MEM_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (n_fields_of((int)process) < 0) return fail(MEM_ERR_INVALID_ARG, "unknown process %d", (int)process);
  mem_params p;
  if (params) p = *params;
  else mem_params_default(process, &p);
  mem_status s = check_params((int)process, p);
  if (s != MEM_OK) return s;
  if (n_consts_of((int)process) < 0)
    return fail(MEM_ERR_UNSUPPORTED, "process %d is not implemented in this build", (int)process);
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (prop.major < 10)
    return fail(MEM_ERR_CUDA, "device %d is sm_%d%d; this library is built for sm_100a only", dev, prop.major, prop.minor);
  mem_handle* h = new (std::nothrow) mem_handle();
  if (!h) return fail(MEM_ERR_NOMEM, "out of host memory");
  h->process = (int)process; h->device = dev; h->params = p; h->dc = make_dev_const(p); h->dcf = to_float(h->dc);
  h->event_offset = 0; h->launches = 0; h->grid_events = 0; h->last_evals = 0; h->has_done = false; h->tickets_dirty = false;
  cudaError_t ce = cudaEventCreate(&h->ev_begin);
  if (ce == cudaSuccess) ce = cudaEventCreate(&h->ev_end);
  if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&h->ev_done, cudaEventDisableTiming);
  if (ce != cudaSuccess) {
    delete h;
    return fail(MEM_ERR_CUDA, "cudaEventCreate: %s", cudaGetErrorString(ce));
  }
  *out = h;
  return MEM_OK;
}

mem_status mem_destroy(mem_handle* h) {
  if (!h) return MEM_OK;
  // synchronise and free on the handle's own device, whatever device is current, and restore the caller's
  int cur = -1;
  const bool have_cur = cudaGetDevice(&cur) == cudaSuccess;
  if (have_cur && cur != h->device) cudaSetDevice(h->device);
  cudaDeviceSynchronize();
  Buffer* bs[] = {&h->ecs, &h->partials, &h->grids, &h->hist, &h->stage_in, &h->stage_out, &h->pdf_tab, &h->tickets};
  for (Buffer* b : bs)
    if (b->p) cudaFree(b->p);
  cudaEventDestroy(h->ev_begin);
  cudaEventDestroy(h->ev_end);
  cudaEventDestroy(h->ev_done);
  if (have_cur && cur != h->device) cudaSetDevice(cur);
  delete h;
  return MEM_OK;
}

mem_status mem_set_event_offset(mem_handle* h, uint64_t first_event) {
  if (!h) return fail(MEM_ERR_INVALID_ARG, "handle is NULL");
  h->event_offset = first_event;
  return MEM_OK;
}

int64_t mem_launch_count(const mem_handle* h) { return h ? h->launches : -1; }

mem_status mem_last_pass_ms(mem_handle* h, double* ms, int64_t* evals) {
  if (!h || !ms) return fail(MEM_ERR_INVALID_ARG, "handle / ms is NULL");
  if (h->last_evals == 0) return fail(MEM_ERR_INVALID_ARG, "no mem_integrate has run on this handle");
  CUDA_TRY(cudaEventSynchronize(h->ev_end));
  float f = 0.f;
  CUDA_TRY(cudaEventElapsedTime(&f, h->ev_begin, h->ev_end));
  *ms = (double)f;
  if (evals) *evals = h->last_evals;
  return MEM_OK;
}

static mem_status measure_fp64(int kind, int32_t repeats, double* tflops, void* cuda_stream) {
  if (!tflops || repeats < 1 || kind < 0 || kind > 6) return fail(MEM_ERR_INVALID_ARG, "tflops is NULL, repeats < 1 or kind outside 0..6");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  double* sink = nullptr;
  CUDA_TRY(cudaMalloc(&sink, sizeof(double)));
  cudaEvent_t a = nullptr, b = nullptr;
  cudaError_t ce = cudaEventCreate(&a);
  if (ce == cudaSuccess) ce = cudaEventCreate(&b);
  if (ce != cudaSuccess) {
    cudaFree(sink);
    if (a) cudaEventDestroy(a);
    return fail(MEM_ERR_CUDA, "cudaEventCreate: %s", cudaGetErrorString(ce));
  }
  const int blocks = sms * 8 * 4, threads = 256;           // 4 waves of 8 resident blocks per SM
  double best = 0.0;
  for (int r = 0; r < repeats + 1; ++r) {                  // first launch is the warm-up
    cudaEventRecord(a, st);
    switch (kind) {
      case 0: fp64_peak_kernel<0><<<blocks, threads, 0, st>>>(sink, 0.999999, 1e-9, 0x9e3779b9u); break;
      case 1: fp64_peak_kernel<1><<<blocks, threads, 0, st>>>(sink, 0.999999, 1e-9, 0x9e3779b9u); break;
      case 2: fp64_peak_kernel<2><<<blocks, threads, 0, st>>>(sink, 0.999999, 1e-9, 0x9e3779b9u); break;
      case 3: fp64_peak_kernel<3><<<blocks, threads, 0, st>>>(sink, 0.999999, 1e-9, 0x9e3779b9u); break;
      case 4: fp64_peak_kernel<4><<<blocks, threads, 0, st>>>(sink, 0.999999, 1e-9, 0x9e3779b9u); break;
      case 5: fp64_peak_kernel<5><<<blocks, threads, 0, st>>>(sink, 0.999999, 1e-9, 0x9e3779b9u); break;
      default: fp64_peak_kernel<6><<<blocks, threads, 0, st>>>(sink, 0.999999, 1e-9, 0x9e3779b9u); break;
    }
    cudaEventRecord(b, st);
    cudaError_t e = cudaEventSynchronize(b);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    if (e != cudaSuccess) {
      cudaFree(sink); cudaEventDestroy(a); cudaEventDestroy(b);
      return fail(MEM_ERR_CUDA, "fp64 peak kernel: %s", cudaGetErrorString(e));
    }
    const double flops = 2.0 * 8.0 * kPeakIters * (double)threads * (double)blocks;
    if (r > 0 && flops / (ms * 1e-3) / 1e12 > best) best = flops / (ms * 1e-3) / 1e12;
  }
  cudaFree(sink); cudaEventDestroy(a); cudaEventDestroy(b);
  *tflops = best;
  return MEM_OK;
}

mem_status mem_measure_fp64_peak(int32_t repeats, double* tflops, void* cuda_stream) {
  return measure_fp64(0, repeats, tflops, cuda_stream);
}

mem_status mem_measure_fp64_peak_rrr(int32_t repeats, double* tflops, void* cuda_stream) {
  return measure_fp64(1, repeats, tflops, cuda_stream);
}

mem_status mem_measure_fp64_rate(int32_t kind, int32_t repeats, double* tflops, void* cuda_stream) {
  return measure_fp64(kind, repeats, tflops, cuda_stream);
}

mem_status mem_integrate(mem_handle* h, const double* events, int64_t n_events, int64_t n_points, uint64_t seed,
                         double* out_p, double* out_err, void* cuda_stream) {
  if (!h) return fail(MEM_ERR_INVALID_ARG, "handle is NULL");
  if (n_events < 0) return fail(MEM_ERR_INVALID_ARG, "n_events < 0");
  if (n_points < 2) return fail(MEM_ERR_INVALID_ARG, "n_points < 2");
  if (n_events == 0) return MEM_OK;
  if (!events || !out_p || !out_err) return fail(MEM_ERR_INVALID_ARG, "events / out_p / out_err is NULL");
  if (!aligned8(events) || !aligned8(out_p) || !aligned8(out_err))
    return fail(MEM_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
  mem_status cs = check_device(h);
  if (cs == MEM_OK) cs = check_counter(h, n_events);
  if (cs != MEM_OK) return cs;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  switch (h->process) {
    case MEM_PROC_W_ENU: return integrate_impl<ProcWenu>(h, events, n_events, n_points, seed, out_p, out_err, st);
    case MEM_PROC_Z_BB: return integrate_impl<ProcZbb>(h, events, n_events, n_points, seed, out_p, out_err, st);
    case MEM_PROC_TT_LJETS:
      if (h->params.precision == 32)
        return integrate_impl<ProcTTljetsF>(h, events, n_events, n_points, seed, out_p, out_err, st);
      return integrate_impl<ProcTTljets>(h, events, n_events, n_points, seed, out_p, out_err, st);
    case MEM_PROC_TT_DILEP: return integrate_impl<ProcTTdilep>(h, events, n_events, n_points, seed, out_p, out_err, st);
    case MEM_PROC_TTH_DILEP: return integrate_impl<ProcTTHdilep>(h, events, n_events, n_points, seed, out_p, out_err, st);
  }
  return fail(MEM_ERR_UNSUPPORTED, "process %d is not implemented", h->process);
}

mem_status mem_integrate_noalloc(mem_handle* h, const double* events, int64_t n_events, int64_t n_points, uint64_t seed,
                                 double* out_p, double* out_err, void* cuda_stream) {
  if (!h) return fail(MEM_ERR_INVALID_ARG, "handle is NULL");
  if (n_events < 0) return fail(MEM_ERR_INVALID_ARG, "n_events < 0");
  if (n_points < 2) return fail(MEM_ERR_INVALID_ARG, "n_points < 2");
  if (h->params.vegas_iters > 0)
    return fail(MEM_ERR_UNSUPPORTED, "mem_integrate_noalloc is plain Monte Carlo only (this handle has vegas_iters = %d)", h->params.vegas_iters);
  if (n_events == 0) return MEM_OK;
  if (!events || !out_p || !out_err) return fail(MEM_ERR_INVALID_ARG, "events / out_p / out_err is NULL");
  if (!aligned8(events) || !aligned8(out_p) || !aligned8(out_err))
    return fail(MEM_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
  mem_status cs = check_device(h);
  if (cs == MEM_OK) cs = check_counter(h, n_events);
  if (cs != MEM_OK) return cs;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  switch (h->process) {
    case MEM_PROC_W_ENU: return integrate_noalloc_impl<ProcWenu>(h, events, n_events, n_points, seed, out_p, out_err, st);
    case MEM_PROC_Z_BB: return integrate_noalloc_impl<ProcZbb>(h, events, n_events, n_points, seed, out_p, out_err, st);
    case MEM_PROC_TT_LJETS:
      if (h->params.precision == 32)
        return integrate_noalloc_impl<ProcTTljetsF>(h, events, n_events, n_points, seed, out_p, out_err, st);
      return integrate_noalloc_impl<ProcTTljets>(h, events, n_events, n_points, seed, out_p, out_err, st);
    case MEM_PROC_TT_DILEP: return integrate_noalloc_impl<ProcTTdilep>(h, events, n_events, n_points, seed, out_p, out_err, st);
    case MEM_PROC_TTH_DILEP: return integrate_noalloc_impl<ProcTTHdilep>(h, events, n_events, n_points, seed, out_p, out_err, st);
  }
  return fail(MEM_ERR_UNSUPPORTED, "process %d is not implemented", h->process);
}

mem_status mem_integrate_host(mem_handle* h, const double* events_host, int64_t n_events, int64_t n_points,
                              uint64_t seed, double* out_p_host, double* out_err_host, void* cuda_stream) {
  if (!h) return fail(MEM_ERR_INVALID_ARG, "handle is NULL");
  if (n_events < 0) return fail(MEM_ERR_INVALID_ARG, "n_events < 0");
  if (n_points < 2) return fail(MEM_ERR_INVALID_ARG, "n_points < 2");
  if (n_events == 0) return MEM_OK;
  if (!events_host || !out_p_host || !out_err_host) return fail(MEM_ERR_INVALID_ARG, "a host buffer is NULL");
  mem_status s = check_device(h);
  if (s != MEM_OK) return s;
  const size_t in_bytes = (size_t)n_events * n_fields_of(h->process) * sizeof(double);
  const size_t out_bytes = (size_t)n_events * sizeof(double);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // the staging buffers belong to the workspace: order this call after the previous one before touching them
  if (h->has_done) CUDA_TRY(cudaStreamWaitEvent(st, h->ev_done, 0));
  s = ensure(h, h->stage_in, in_bytes, st);
  if (s != MEM_OK) return s;
  s = ensure(h, h->stage_out, 2 * out_bytes, st);
  if (s != MEM_OK) return s;
  double* d_out = (double*)h->stage_out.p;
  CUDA_TRY(cudaMemcpyAsync(h->stage_in.p, events_host, in_bytes, cudaMemcpyHostToDevice, st));
  s = mem_integrate(h, (const double*)h->stage_in.p, n_events, n_points, seed, d_out, d_out + n_events, st);
  if (s != MEM_OK) return s;
  CUDA_TRY(cudaMemcpyAsync(out_p_host, d_out, out_bytes, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpyAsync(out_err_host, d_out + n_events, out_bytes, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaEventRecord(h->ev_done, st));          // the copies out read the staging buffer too
  CUDA_TRY(cudaStreamSynchronize(st));
  return MEM_OK;
}

mem_status mem_eval_points(mem_handle* h, const double* events, int64_t n_events, int64_t event, int64_t first_point,
                           int64_t n, uint64_t seed, int32_t iteration, const double* grid, double* out_w,
                           void* cuda_stream) {
  if (!h) return fail(MEM_ERR_INVALID_ARG, "handle is NULL");
  if (n_events <= 0 || event < 0 || event >= n_events) return fail(MEM_ERR_INVALID_ARG, "event outside [0, n_events)");
  if (n < 0 || first_point < 0) return fail(MEM_ERR_INVALID_ARG, "n < 0 or first_point < 0");
  if (iteration < 0 || iteration > 255) return fail(MEM_ERR_INVALID_ARG, "iteration outside 0..255");
  if (n == 0) return MEM_OK;
  if (!events || !out_w) return fail(MEM_ERR_INVALID_ARG, "events / out_w is NULL");
  if (!aligned8(events) || !aligned8(out_w) || !aligned8(grid))
    return fail(MEM_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
  if (grid && (h->params.vegas_bins < 1 || h->params.vegas_bins > kMaxBins))
    return fail(MEM_ERR_INVALID_ARG, "vegas_bins outside 1..%d", kMaxBins);
  mem_status cs = check_device(h);
  if (cs == MEM_OK) cs = check_counter(h, n_events);
  if (cs != MEM_OK) return cs;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  switch (h->process) {
    case MEM_PROC_W_ENU: return eval_impl<ProcWenu>(h, events, n_events, event, first_point, n, seed, iteration, grid, out_w, st);
    case MEM_PROC_Z_BB: return eval_impl<ProcZbb>(h, events, n_events, event, first_point, n, seed, iteration, grid, out_w, st);
    case MEM_PROC_TT_LJETS:
      if (h->params.precision == 32)
        return eval_impl<ProcTTljetsF>(h, events, n_events, event, first_point, n, seed, iteration, grid, out_w, st);
      return eval_impl<ProcTTljets>(h, events, n_events, event, first_point, n, seed, iteration, grid, out_w, st);
    case MEM_PROC_TT_DILEP: return eval_impl<ProcTTdilep>(h, events, n_events, event, first_point, n, seed, iteration, grid, out_w, st);
    case MEM_PROC_TTH_DILEP: return eval_impl<ProcTTHdilep>(h, events, n_events, event, first_point, n, seed, iteration, grid, out_w, st);
  }
  return fail(MEM_ERR_UNSUPPORTED, "process %d is not implemented", h->process);
}

mem_status mem_set_pdf_grid(mem_handle* h, const double* table, int32_t nx, int32_t nq, double lxmin, double lxmax,
                            double lqmin, double lqmax, double Q) {
  if (!h) return fail(MEM_ERR_INVALID_ARG, "handle is NULL");
  mem_status cs = check_device(h);
  if (cs != MEM_OK) return cs;
  // kernels in flight on any stream (torch side streams do not synchronise with the legacy stream) may still read
  // the table that is about to be replaced or dropped
  CUDA_TRY(cudaDeviceSynchronize());
  if (!table) {                                             // back to the toy PDF
    h->dc.pdf_tab = nullptr;
    return MEM_OK;
  }
  if ((h->process != MEM_PROC_TT_LJETS && h->process != MEM_PROC_TT_DILEP && h->process != MEM_PROC_TTH_DILEP) ||
      h->params.precision != 64)
    return fail(MEM_ERR_UNSUPPORTED, "grid PDFs are implemented for the t tbar processes in fp64");
  if (nx < 2 || nq < 2 || nx > 65536 || nq > 65536) return fail(MEM_ERR_INVALID_ARG, "nx, nq outside 2..65536");
  if (!(lxmax > lxmin) || !(lqmax > lqmin) || !(Q > 0.0)) return fail(MEM_ERR_INVALID_ARG, "empty grid range or Q <= 0");
  // fold the ln Q direction of the bilinear interpolation (listing PAPER.md:274-306) into one row per species
  const double lq = std::log(Q), dq = (lqmax - lqmin) / nq;
  int iq = 0;
  if (lqmin < lq) iq = (int)((lq - lqmin) / dq);
  iq = iq < nq - 1 ? iq : nq - 2;
  const double c11q = lqmin + dq * iq, c22q = lqmin + dq * (iq + 1);
  double* row = new (std::nothrow) double[(size_t)6 * nx];
  if (!row) return fail(MEM_ERR_NOMEM, "out of host memory");
  for (int s = 0; s < 6; ++s)
    for (int ix = 0; ix < nx; ++ix) {
      const double d0 = table[((size_t)s * nq + iq) * nx + ix], d1 = table[((size_t)s * nq + iq + 1) * nx + ix];
      row[(size_t)s * nx + ix] = (d0 * (c22q - lq) + d1 * (lq - c11q)) / dq;
    }
  cudaStream_t st = 0;
  mem_status r = ensure(h, h->pdf_tab, (size_t)6 * nx * sizeof(double), st);
  cudaError_t e = cudaSuccess;
  if (r == MEM_OK) {
    e = cudaMemcpy(h->pdf_tab.p, row, (size_t)6 * nx * sizeof(double), cudaMemcpyHostToDevice);   // synchronous
  }
  delete[] row;
  if (r != MEM_OK) return r;
  if (e != cudaSuccess) return fail(MEM_ERR_CUDA, "cudaMemcpy(pdf table): %s", cudaGetErrorString(e));
  h->dc.pdf_tab = (const double*)h->pdf_tab.p;
  h->dc.pdf_nx = nx;
  h->dc.pdf_lxmin = lxmin;
  h->dc.pdf_dx = (lxmax - lxmin) / nx;
  h->dc.pdf_inv_dx = 1.0 / h->dc.pdf_dx;
  return MEM_OK;
}

mem_status mem_eval_parton(mem_handle* h, const double* momenta, int64_t n_events, double* out_w, void* cuda_stream) {
  if (!h) return fail(MEM_ERR_INVALID_ARG, "handle is NULL");
  if (h->process != MEM_PROC_TT_LJETS || h->params.precision != 64)
    return fail(MEM_ERR_UNSUPPORTED, "parton-level mode is implemented for MEM_PROC_TT_LJETS in fp64");
  if (n_events < 0) return fail(MEM_ERR_INVALID_ARG, "n_events < 0");
  if (n_events == 0) return MEM_OK;
  if (!momenta || !out_w) return fail(MEM_ERR_INVALID_ARG, "momenta / out_w is NULL");
  if (!aligned8(momenta) || !aligned8(out_w)) return fail(MEM_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
  mem_status cs = check_device(h);
  if (cs != MEM_OK) return cs;
  const int threads = h->dc.n_perm > 1 ? 128 : 256;
  const int64_t blocks = (n_events + threads - 1) / threads;
  if (blocks > 0x7fffffffLL) return fail(MEM_ERR_INVALID_ARG, "n_events exceeds the grid limit");
  if (h->dc.n_perm > 1)
    parton_ttljets_kernel<false><<<(unsigned)blocks, threads, 0, (cudaStream_t)cuda_stream>>>(h->dc, momenta, n_events, out_w);
  else
    parton_ttljets_kernel<true><<<(unsigned)blocks, threads, 0, (cudaStream_t)cuda_stream>>>(h->dc, momenta, n_events, out_w);
  ++h->launches;
  CUDA_TRY(cudaGetLastError());
  return MEM_OK;
}

mem_status mem_normalisation(const double* p, const double* g, int64_t n, double* out_sigma, void* cuda_stream) {
  if (n < 1) return fail(MEM_ERR_INVALID_ARG, "n < 1");
  if (!p || !g || !out_sigma) return fail(MEM_ERR_INVALID_ARG, "p / g / out_sigma is NULL");
  if (!aligned8(p) || !aligned8(g) || !aligned8(out_sigma)) return fail(MEM_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
  normalisation_kernel<<<1, kThreads, 0, (cudaStream_t)cuda_stream>>>(p, g, n, out_sigma);
  CUDA_TRY(cudaGetLastError());
  return MEM_OK;
}

mem_status mem_discriminant(const double* p_sig, const double* p_bkg, int64_t n, const double* sigma_sig,
                            const double* sigma_bkg, double* out_D, void* cuda_stream) {
  if (n < 0) return fail(MEM_ERR_INVALID_ARG, "n < 0");
  if (n == 0) return MEM_OK;
  if (!p_sig || !p_bkg || !sigma_sig || !sigma_bkg || !out_D) return fail(MEM_ERR_INVALID_ARG, "a pointer is NULL");
  if (!aligned8(p_sig) || !aligned8(p_bkg) || !aligned8(sigma_sig) || !aligned8(sigma_bkg) || !aligned8(out_D))
    return fail(MEM_ERR_INVALID_ARG, "device pointers must be 8-byte aligned");
  const int64_t blocks = (n + 255) / 256;
  if (blocks > 0x7fffffffLL) return fail(MEM_ERR_INVALID_ARG, "n exceeds the grid limit");
  discriminant_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)cuda_stream>>>(p_sig, p_bkg, n, sigma_sig, sigma_bkg, out_D);
  CUDA_TRY(cudaGetLastError());
  return MEM_OK;
}

mem_status mem_get_grid(mem_handle* h, int64_t n_events, double* out_grid, void* cuda_stream) {
  if (!h || !out_grid) return fail(MEM_ERR_INVALID_ARG, "handle / out_grid is NULL");
  if (h->params.vegas_iters <= 0 || !h->grids.p || n_events != h->grid_events)
    return fail(MEM_ERR_INVALID_ARG, "no VEGAS grids for %lld events on this handle", (long long)n_events);
  mem_status cs = check_device(h);
  if (cs != MEM_OK) return cs;
  const size_t bytes = (size_t)n_events * n_dims_of(h->process) * (h->params.vegas_bins + 1) * sizeof(double);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  bool capturing = false;
  cs = begin_call(h, st, &capturing);
  if (cs != MEM_OK) return cs;
  CUDA_TRY(cudaMemcpyAsync(out_grid, h->grids.p, bytes, cudaMemcpyDeviceToDevice, st));
  return end_call(h, st, capturing);
}

}  // extern "C"
