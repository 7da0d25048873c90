// mem_parton.cuh -- NEXT-2, parton-level mode (Table 2): transfer functions
// are delta functions, nothing is integrated; one thread evaluates the integrand of Eq. 1 (without
// dPhi) at one fully specified partonic configuration, summed over the jet-parton assignments and
// the initial-state flavours.  Shares nothing with oracle/.
#pragma once
#include "mem_processes.cuh"

namespace memb200 {

struct P4 { double E, x, y, z; };
__device__ __forceinline__ P4 operator+(const P4& a, const P4& b) { return {a.E + b.E, a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ double mdot(const P4& a, const P4& b) {
  return fma(a.E, b.E, -fma(a.x, b.x, fma(a.y, b.y, a.z * b.z)));
}

// mom: SoA field-major [24][n_events] = (E, px, py, pz) of l, nu, b_had, b_lep, q, qbar'
// ONE = the record's own assignment only (n_perm = 1): no assignment loop, no role selection.  With one assignment
// the kernel moves 200 B per event and is bound by HBM, so everything that costs issue slots next to the loads --
// IEEE divisions, the generic assignment machinery, a second store -- was removed (profiles/r02_parton.md).
template <bool ONE>
__global__ void __launch_bounds__(ONE ? 256 : 128, 3)
parton_ttljets_kernel(const DevConst c, const double* __restrict__ mom, int64_t n_events, double* __restrict__ out_w) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n_events) return;
  P4 p[6];
#pragma unroll
  for (int i = 0; i < 6; ++i)
    p[i] = {__ldg(mom + (4 * i) * n_events + e), __ldg(mom + (4 * i + 1) * n_events + e),
            __ldg(mom + (4 * i + 2) * n_events + e), __ldg(mom + (4 * i + 3) * n_events + e)};
  double w = 0.0;
  do {
  // ---- O7: pure transverse boost that removes P_T (the same for every assignment)
  const P4 P = ((p[0] + p[1]) + (p[2] + p[3])) + (p[4] + p[5]);
  const double PT2 = fma(P.x, P.x, P.y * P.y);
  if (!(PT2 < P.E * P.E)) break;
  const double iPE = rcp_fast(P.E);
  const double bx = P.x * iPE, by = P.y * iPE;
  const double gam = rsqrt_fast(1.0 - fma(bx, bx, by * by));
  const double k2 = gam * gam * rcp_fast(gam + 1.0);               // (gamma - 1) / beta^2, finite at beta = 0
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    const double bp = fma(bx, p[i].x, by * p[i].y);
    const double k = fma(k2, bp, -gam * p[i].E);
    p[i].E = gam * (p[i].E - bp);
    p[i].x = fma(k, bx, p[i].x);
    p[i].y = fma(k, by, p[i].y);
  }
  double PE = 0.0;
#pragma unroll
  for (int i = 0; i < 6; ++i) PE += p[i].E;
  const double x1 = (PE + P.z) * c.inv_sqrt_s, x2 = (PE - P.z) * c.inv_sqrt_s;
  if (!(x1 > 0.0 && x1 < 1.0 && x2 > 0.0 && x2 < 1.0)) break;
  const double shat = x1 * x2 * c.S;
  if (!(4.0 * c.mt2 < shat)) break;                                // reading A9
  const double h = 0.5 * c.sqrt_s, ish = rcp_fast(shat), rho = 4.0 * c.mt2 * ish;
  const TtLumi<double> lum = tt_lumi<true>(c, x1, x2);                   // the same for every assignment
  const P4 l = p[0], nu = p[1];
  const P4 Wl = l + nu;
  const double swl_m = mdot(Wl, Wl) - c.mW2;
  const double dWl = fma(swl_m, swl_m, c.mWGW2);
  double sum = 0.0;
  const int n_perm = ONE ? 1 : c.n_perm;
  for (int kperm = 0; kperm < n_perm; ++kperm) {
    int sig[4] = {0, 1, 2, 3};
    if (!ONE) jet_assignment(c.n_perm, kperm, sig);
    // the four jets sit in p[2..5]; select by role without dynamic register indexing
    P4 r[4];
#pragma unroll
    for (int role = 0; role < 4; ++role) {
      const int j = sig[role];
      r[role] = ONE ? p[2 + role] : (j == 0) ? p[2] : (j == 1) ? p[3] : (j == 2) ? p[4] : p[5];
    }
    const P4 bh = r[0], bl = r[1], q = r[2], qb = r[3];
    const P4 pt = Wl + bl, Wh = q + qb, ptb = Wh + bh;
    // production: tau1 = (q1.pt + q2.ptb)/s-hat, tau2 = (q2.pt + q1.ptb)/s-hat
    const double tau1 = h * ish * fma(x1, pt.E - pt.z, x2 * (ptb.E + ptb.z));
    const double tau2 = h * ish * fma(x2, pt.E + pt.z, x1 * (ptb.E - ptb.z));
    const double t12 = tau1 * tau2, tt = fma(tau1, tau1, tau2 * tau2);
    // propagators from the momenta; one reciprocal for 1/(tau1 tau2) and the four denominators
    const double st_m = mdot(pt, pt) - c.mt2, stb_m = mdot(ptb, ptb) - c.mt2, swh_m = mdot(Wh, Wh) - c.mW2;
    const double dens = dWl * fma(st_m, st_m, c.mtGt2) * fma(stb_m, stb_m, c.mtGt2) * fma(swh_m, swh_m, c.mWGW2);
    const double inv = rcp_fast(t12 * dens);
    const double iT = inv * dens, props = inv * t12;
    const double Mgg = (iT * (1.0 / 6.0) - 0.375) * (tt + rho - 0.25 * rho * rho * iT);
    const double Mqq = tt + 0.5 * rho;
    const double prod = c.gs4 * fma(lum.gg, Mgg, lum.qq * Mqq);    // flavour sum incl. the PDFs
    // decays, summed over spins, 1/2 per decaying top: (p_t.p_l)(p_b.p_nu) and 3 |V_ud|^2 (p_tbar.p_q)(p_bbar.p_qbar')
    const double dec = (2.0 * c.g4w * c.V_tb2) * mdot(pt, l) * mdot(bl, nu) *
                       (6.0 * c.g4w * c.V_tb2 * c.V_ud2) * mdot(ptb, q) * mdot(bh, qb);
    const double me = prod * props * dec;
    if (isfinite(me)) sum += me;
  }
  w = 4.0 * ish * sum;                                              // 1 / (x1 x2 S / 4)
  } while (false);
  out_w[e] = isfinite(w) ? w : 0.0;
}

}  // namespace memb200
