// oracle/mem_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain single-threaded fp64 oracle for the matrix-element-method hot path of
// arXiv 1407.7595: p = (1/N) sum_i w_i, w = V * J * dPhi * PDF * |M|^2 * TF at
// points drawn from a Philox4x32-10 stream keyed by (seed, event, point).
// It follows the algorithm step by step in the order DESIGN.md states it
// (readings O1-O8, A1-A17 of SURVEY.md section 8(c)); no blocking, fusion or
// reordering.  Built with g++ -O2 -ffp-contract=off, platform libm.
// Shares nothing with paper_1407_7595_b200/csrc/.
//
// Every arithmetic routine is a template over the real type R.  R = double is
// the oracle proper (all orc_* entry points without suffix).  R = long double
// (x87, 64-bit mantissa, libm's *l functions) is the same text instantiated a
// second time and exported as orc_weight_x / orc_eval_points_x: an
// extended-precision referee the tests use to decide which side is wrong at
// points where the fp64 evaluation is ill-conditioned (cancellation in
// s_t = p_t^2 next to the top pole; "cancellation of large
// coefficients").
//
// Pins (tests/test_oracle_*.py): Philox known-answer vectors; Breit-Wigner and
// double-Gaussian normalisation; Dirac-trace and closed-form cross-section
// checks of every matrix element; massless phase-space volume; momentum
// conservation of every configuration; brute-force quadrature of the 1-D and
// 2-D configs; chart independence of config 3; VEGAS grid invariants.
// Config-3/config-4 absolute values and the VEGAS constants (A14):
// "parity unpinned" beyond those factor-wise pins.
#include "mem_oracle.h"

#include <cmath>
#include <cstring>
#include <limits>
#include <vector>

namespace {

const long double kPiL = 3.14159265358979323846264338327950288L;
template <typename R> inline R pi_() { return (R)kPiL; }

template <typename R>
struct V4 {
  R E, x, y, z;
};
template <typename R> inline V4<R> operator+(const V4<R>& a, const V4<R>& b) {
  return {a.E + b.E, a.x + b.x, a.y + b.y, a.z + b.z};
}
template <typename R> inline R dot(const V4<R>& a, const V4<R>& b) {
  return a.E * b.E - a.x * b.x - a.y * b.y - a.z * b.z;
}
template <typename R> inline V4<R> from_arr(const R* a) { return {a[0], a[1], a[2], a[3]}; }
template <typename R> inline void to_arr(const V4<R>& v, R* a) { a[0] = v.E; a[1] = v.x; a[2] = v.y; a[3] = v.z; }

// massless particle from (pT, eta, phi)
template <typename R> inline V4<R> from_pt_eta_phi(R pT, R eta, R phi) {
  return {pT * std::cosh(eta), pT * std::cos(phi), pT * std::sin(phi), pT * std::sinh(eta)};
}
// massless particle from (E, eta, phi): direction n = (cos phi/cosh eta, sin phi/cosh eta, tanh eta)
template <typename R> inline V4<R> from_E_eta_phi(R E, R eta, R phi) {
  R st = R(1) / std::cosh(eta);  // sin(theta)
  return {E, E * st * std::cos(phi), E * st * std::sin(phi), E * std::tanh(eta)};
}

// ---- Neumaier compensated sum, index order (O1) ----
struct NSum {
  double s = 0.0, c = 0.0;
  void add(double v) {
    double t = s + v;
    if (std::fabs(s) >= std::fabs(v)) c += (s - t) + v; else c += (v - t) + s;
    s = t;
  }
  double value() const { return s + c; }
};

// ---- couplings (O8) ----
template <typename R> inline R g2_weak(const orc_params* p) {
  return R(4) * std::sqrt(R(2)) * R(p->G_F) * R(p->m_W) * R(p->m_W);
}
template <typename R> inline R gZ2(const orc_params* p) {
  return R(4) * std::sqrt(R(2)) * R(p->G_F) * R(p->m_Z) * R(p->m_Z);
}
template <typename R> inline R gs2(const orc_params* p) { return R(4) * pi_<R>() * R(p->alpha_s); }
template <typename R> inline void z_couplings(const orc_params* p, bool up, R* L, R* Rr) {
  R T3 = up ? R(0.5) : R(-0.5), Q = up ? R(2) / R(3) : R(-1) / R(3);
  *L = T3 - Q * R(p->sin2_thw);
  *Rr = -Q * R(p->sin2_thw);
}
template <typename R> inline R bw_D(R s_minus_m2, R m, R Gam) {
  return R(1) / (s_minus_m2 * s_minus_m2 + m * m * Gam * Gam);
}
// flavours in the paper's order (d,u,s,c,b); first n_flav are summed.
inline bool flavour_is_up(int i) { return i == 1 || i == 3; }

// --------------------------------------------------------------------------
// O4. toy PDF shape, O5. jet TF, O6. Breit-Wigner map
// --------------------------------------------------------------------------
template <typename R> R pdf_shape(const orc_params* p, R x) {
  return std::pow(x, R(p->pdf_pow_x)) * std::pow(R(1) - x, R(p->pdf_pow_1mx));
}

template <typename R> R gauss(R d, R mu, R sig) {
  R z = (d - mu) / sig;
  return std::exp(R(-0.5) * z * z) / (sig * std::sqrt(R(2) * pi_<R>()));
}
// PAPER.md:58 "double Gaussian"; BASELINE.json:configs[1] parameters; reading A11.
template <typename R> R tf_jet(const orc_params* p, R E_jet, R E) {
  R d = E_jet - E;
  return (R(1) - R(p->tf_w_tail)) * gauss<R>(d, R(p->tf_mu1) * E, R(p->tf_sig1) * E) +
         R(p->tf_w_tail) * gauss<R>(d, R(p->tf_mu2) * E, R(p->tf_sig2) * E);
}

// NEXT-3, grid PDFs ("stored in (x, Q^2) grids for each parton flavor ... evaluated using
// bilinear interpolation within the kernel"; listing PAPER.md:274-306 Fig. A.5, reading A17): uniform
// grid in (ln x, ln Q) with NX x NQ samples per species, sample i at min + i (max - min)/N (the
// listing's step), cell index clamped to [0, N-2] (so points outside the grid extrapolate the edge
// cell), value = sum of the four corners weighted by the opposite areas / (dx dq).
// species: 0 = gluon, 1..5 = d, u, s, c, b (antiquark = quark in the synthesised tables).
template <typename R> R pdf_grid(const orc_params* p, int species, R x, R Q) {
  const int NX = p->pdf_nx, NQ = p->pdf_nq;
  if (species < 0 || species > 5) return R(0);
  const double* data = p->pdf_data + (size_t)species * NX * NQ;
  const R lx = std::log(x), lq = std::log(Q);
  const R dx = (R(p->pdf_lxmax) - R(p->pdf_lxmin)) / R(NX), dq = (R(p->pdf_lqmax) - R(p->pdf_lqmin)) / R(NQ);
  int ix = 0, iq = 0;
  if (R(p->pdf_lxmin) < lx) ix = (int)((lx - R(p->pdf_lxmin)) / dx);
  ix = ix < NX - 1 ? ix : NX - 2;
  if (R(p->pdf_lqmin) < lq) iq = (int)((lq - R(p->pdf_lqmin)) / dq);
  iq = iq < NQ - 1 ? iq : NQ - 2;
  const R c11x = R(p->pdf_lxmin) + dx * R(ix), c11q = R(p->pdf_lqmin) + dq * R(iq);
  const R c22x = R(p->pdf_lxmin) + dx * R(ix + 1), c22q = R(p->pdf_lqmin) + dq * R(iq + 1);
  const R norm = dx * dq;
  const R d00 = data[(size_t)iq * NX + ix], d10 = data[(size_t)(iq + 1) * NX + ix];
  const R d01 = data[(size_t)iq * NX + ix + 1], d11 = data[(size_t)(iq + 1) * NX + ix + 1];
  return d00 / norm * (c22x - lx) * (c22q - lq) + d01 / norm * (lx - c11x) * (c22q - lq) +
         d10 / norm * (c22x - lx) * (lq - c11q) + d11 / norm * (lx - c11x) * (lq - c11q);
}

// sum over initial-state flavours of f_a(x1) f_b(x2) |M_ab|^2 for t tbar production:
// g g, and q qbar + qbar q for the first n_flav quark species.  Toy mode (O4): every species has
// the shape A x^a (1-x)^b; grid mode: pdf_grid at the fixed scale pdf_Q.
template <typename R> R tt_flavour_sum(const orc_params* p, R x1, R x2, R me_gg, R me_qq) {
  if (!p->pdf_mode) {
    const R ff = pdf_shape<R>(p, x1) * pdf_shape<R>(p, x2);
    return ff * (R(p->pdf_A_g) * R(p->pdf_A_g) * me_gg + R(2) * R(p->n_flav) * R(p->pdf_A_q) * R(p->pdf_A_q) * me_qq);
  }
  const R Q = p->pdf_Q;
  R lqq = R(0);
  for (int f = 1; f <= p->n_flav; ++f) lqq += R(2) * pdf_grid<R>(p, f, x1, Q) * pdf_grid<R>(p, f, x2, Q);
  return pdf_grid<R>(p, 0, x1, Q) * pdf_grid<R>(p, 0, x2, Q) * me_gg + lqq * me_qq;
}

// integrate over q^2 of the propagators.  s = m^2 + m Gam tan t.
template <typename R> void bw_window(R m, R Gam, R s_lo, R s_hi, R* t_lo, R* t_hi) {
  *t_lo = std::atan((s_lo - m * m) / (m * Gam));
  *t_hi = std::atan((s_hi - m * m) / (m * Gam));
}
template <typename R> void bw_point(R m, R Gam, R t, R* s_minus_m2, R* dsdt, R* D) {
  R smm = m * Gam * std::tan(t);
  *s_minus_m2 = smm;
  *dsdt = (smm * smm + m * m * Gam * Gam) / (m * Gam);
  *D = bw_D<R>(smm, m, Gam);
}

// --------------------------------------------------------------------------
// matrix elements (SURVEY.md 8(c) "Matrix elements")
// --------------------------------------------------------------------------
// u(qa) dbar(qb) -> W+ -> e+(lep) nu:  g^4 |V_ud|^2 / 12 * u^2 * D_W(s),  u = -2 qa.lep.
// D_W is passed in: for a sampled W mass it is D(m Gam tan t) (reading O6, SURVEY.md 8(c):
// "for a mapped resonance evaluate s - m^2 as m Gam tan t (no cancellation)").
template <typename R> R me_w_D(const orc_params* p, const R qa[4], const R lep[4], R D_W) {
  V4<R> a = from_arr(qa), l = from_arr(lep);
  R uhat = R(-2) * dot(a, l);
  R g2 = g2_weak<R>(p);
  return g2 * g2 * R(p->V_ud) * R(p->V_ud) / R(12) * uhat * uhat * D_W;
}
// the same with D_W from the partonic s-hat = (qa + qb)^2
template <typename R> R me_w(const orc_params* p, const R qa[4], const R qb[4], const R lep[4], const R nu[4]) {
  V4<R> a = from_arr(qa), b = from_arr(qb);
  (void)nu;
  R shat = dot(a + b, a + b);
  return me_w_D<R>(p, qa, lep, bw_D<R>(shat - R(p->m_W) * R(p->m_W), R(p->m_W), R(p->Gam_W)));
}

// q(qa) qbar(qb) -> Z -> b(p1) bbar(p2), Z exchange only, colour factor 1
template <typename R> R me_z(const orc_params* p, int up_type, const R qa[4], const R qb[4], const R p1[4],
                             const R p2[4]) {
  V4<R> a = from_arr(qa), b = from_arr(qb), b1 = from_arr(p1), b2 = from_arr(p2);
  R Lq, Rq, Lb, Rb;
  z_couplings<R>(p, up_type != 0, &Lq, &Rq);
  z_couplings<R>(p, false, &Lb, &Rb);
  R shat = dot(a + b, a + b);
  R uhat = R(-2) * dot(a, b2), that = R(-2) * dot(a, b1);
  R gz = gZ2<R>(p);
  return gz * gz * ((Lq * Lq * Lb * Lb + Rq * Rq * Rb * Rb) * uhat * uhat +
                    (Lq * Lq * Rb * Rb + Rq * Rq * Lb * Lb) * that * that) *
         bw_D<R>(shat - R(p->m_Z) * R(p->m_Z), R(p->m_Z), R(p->Gam_Z));
}

// reading A9: tau1 + tau2 = 1 also off shell, pole mass in rho
template <typename R> void tt_invariants(const orc_params* p, const R q1[4], const R q2[4], const R pt[4],
                                         const R ptb[4], R* t1, R* t2, R* rho) {
  V4<R> a = from_arr(q1), b = from_arr(q2), t = from_arr(pt), tb = from_arr(ptb);
  R shat = dot(a + b, a + b);
  *t1 = (dot(a, t) + dot(b, tb)) / shat;
  *t2 = (dot(b, t) + dot(a, tb)) / shat;
  *rho = R(4) * R(p->m_t) * R(p->m_t) / shat;
}
// the two production matrix elements as functions of (tau1, tau2, rho)
template <typename R> R me_tt_qq_inv(const orc_params* p, R t1, R t2, R rho) {
  R g = gs2<R>(p);
  return g * g * (R(4) / R(9)) * (t1 * t1 + t2 * t2 + rho / R(2));
}
template <typename R> R me_tt_gg_inv(const orc_params* p, R t1, R t2, R rho) {
  R g = gs2<R>(p);
  return g * g * (R(1) / (R(6) * t1 * t2) - R(3) / R(8)) *
         (t1 * t1 + t2 * t2 + rho - rho * rho / (R(4) * t1 * t2));
}
template <typename R> R me_tt_qq(const orc_params* p, const R q1[4], const R q2[4], const R pt[4], const R ptb[4]) {
  R t1, t2, rho;
  tt_invariants<R>(p, q1, q2, pt, ptb, &t1, &t2, &rho);
  return me_tt_qq_inv<R>(p, t1, t2, rho);
}
template <typename R> R me_tt_gg(const orc_params* p, const R q1[4], const R q2[4], const R pt[4], const R ptb[4]) {
  R t1, t2, rho;
  tt_invariants<R>(p, q1, q2, pt, ptb, &t1, &t2, &rho);
  return me_tt_gg_inv<R>(p, t1, t2, rho);
}

// sum over all spins of |M(t -> b W -> b fdown-bar... )|^2 with the pairing
// (p_t . p_fdown)(p_b . p_fup): for t -> b l+ nu, fdown = l+ and fup = nu.
// D_W is passed in: for a sampled W mass it is D(s_W - m_W^2 = m Gam tan t), evaluated
// without recomputing s_W from the momenta (reading O6: "for a mapped
// resonance evaluate s - m^2 as m Gam tan t (no cancellation)").
template <typename R> R me_top_decay_D(const orc_params* p, R n_c, const R pt[4], const R pb[4], const R pf_down[4],
                                       const R pf_up[4], R D_W) {
  V4<R> t = from_arr(pt), b = from_arr(pb), fd = from_arr(pf_down), fu = from_arr(pf_up);
  R g2 = g2_weak<R>(p);
  return n_c * R(4) * g2 * g2 * R(p->V_tb) * R(p->V_tb) * dot(t, fd) * dot(b, fu) * D_W;
}
// the same with D_W from the W momentum fd + fu (unmapped resonance)
template <typename R> R me_top_decay(const orc_params* p, R n_c, const R pt[4], const R pb[4], const R pf_down[4],
                                     const R pf_up[4]) {
  V4<R> fd = from_arr(pf_down), fu = from_arr(pf_up);
  R sW = dot(fd + fu, fd + fu);
  return me_top_decay_D<R>(p, n_c, pt, pb, pf_down, pf_up,
                           bw_D<R>(sW - R(p->m_W) * R(p->m_W), R(p->m_W), R(p->Gam_W)));
}

// O7. pure transverse boost that removes the transverse momentum of P.
template <typename R> void boost_transverse(const R P[4], int n, R* mom) {
  R bx = P[1] / P[0], by = P[2] / P[0];
  R b2 = bx * bx + by * by;
  R gam = R(1) / std::sqrt(R(1) - b2);
  R k2 = gam * gam / (gam + R(1));  // = (gamma-1)/beta^2, finite at beta = 0
  for (int i = 0; i < n; ++i) {
    R* q = mom + 4 * i;
    R bp = bx * q[1] + by * q[2];
    R En = gam * (q[0] - bp);
    R k = k2 * bp - gam * q[0];
    q[1] += k * bx; q[2] += k * by; q[0] = En;
  }
}

// --------------------------------------------------------------------------
// per-configuration weights
// --------------------------------------------------------------------------
// O3: x1, x2 from the (boosted) total momentum.  Returns false when outside (0,1).
template <typename R> bool beam_fractions(const orc_params* p, R PE, R Pz, R* x1, R* x2) {
  *x1 = (PE + Pz) / R(p->sqrt_s);
  *x2 = (PE - Pz) / R(p->sqrt_s);
  return (*x1 > R(0) && *x1 < R(1) && *x2 > R(0) && *x2 < R(1));
}
template <typename R> void beams(const orc_params* p, R x1, R x2, R q1[4], R q2[4]) {
  R h = R(0.5) * R(p->sqrt_s);
  q1[0] = x1 * h; q1[1] = 0; q1[2] = 0; q1[3] = x1 * h;
  q2[0] = x2 * h; q2[1] = 0; q2[2] = 0; q2[3] = -x2 * h;
}

template <typename R> void dbg_store(double* dbg, int sol, int n_final, R x1, R x2, const R* mom) {
  if (!dbg) return;
  double* d = dbg + 1 + sol * (2 + 4 * n_final);
  d[0] = (double)x1; d[1] = (double)x2;
  for (int i = 0; i < 4 * n_final; ++i) d[2 + i] = (double)mom[i];
}

// ---------------- config 1: u dbar -> W+ -> e+ nu, D = 1 ----------------
// rec = [lep_pT, lep_eta, lep_phi, met_x, met_y]   (SURVEY.md 8(c) "Config 1", reading A5)
template <typename R> R weight_w_enu(const orc_params* p, const double* rec, const double* u, double* dbg) {
  const R pT = rec[0], eta = rec[1], phi = rec[2], mx = rec[3], my = rec[4], u0 = u[0];
  const R Pz = p->nu_pz_max, m = p->m_W, G = p->Gam_W, S = R(p->sqrt_s) * R(p->sqrt_s);
  V4<R> l = from_pt_eta_phi<R>(pT, eta, phi);
  R nT = std::sqrt(mx * mx + my * my);
  R a = l.x * mx + l.y * my;                           // l_T . nu_T
  auto s_of = [&](R nz) { return R(2) * (l.E * std::sqrt(nT * nT + nz * nz) - a - l.z * nz); };
  // 1. window in s_W.  Stationary point of s(nu_z): nu_z* = |nu_T| sinh(eta_l), s* = 2(pT nT - a).
  R nz_star = nT * std::sinh(eta);
  R s_star = R(2) * (pT * nT - a);
  R s_min = (nz_star > Pz) ? s_of(Pz) : (nz_star < -Pz) ? s_of(-Pz) : s_star;
  R s_max = std::fmax(s_of(-Pz), s_of(Pz));
  R t_lo, t_hi;
  bw_window<R>(m, G, s_min, s_max, &t_lo, &t_hi);
  R dt = t_hi - t_lo;
  R t = t_lo + dt * u0;
  R smm, dsdt, DW;
  bw_point<R>(m, G, t, &smm, &dsdt, &DW);
  R sW = m * m + smm;
  // 2. roots of s(nu_z) = sW.  disc = c^2 - pT^2 nT^2 = (c - pT nT)(c + pT nT) with
  //    c - pT nT = (sW - s*)/2; sW - s_min = m G (tan t - tan t_lo) = m G sin(dt u)/(cos t cos t_lo)
  //    (cancellation-free near the transverse-mass edge; reading A5b).
  R ds = m * G * std::sin(dt * u0) / (std::cos(t) * std::cos(t_lo));
  R half = R(0.5) * (ds + (s_min - s_star));
  R c = R(0.5) * sW + a;
  R disc = half * (c + pT * nT);
  if (dbg) dbg[0] = 0;
  if (!(disc > R(0))) return R(0);
  R rt = std::sqrt(disc);
  R sum = R(0);
  int n_sol = 0;
  for (int sgn = -1; sgn <= 1; sgn += 2) {
    R nz = (c * l.z + R(sgn) * l.E * rt) / (pT * pT);
    if (!(std::fabs(nz) <= Pz)) continue;
    R En = std::sqrt(nT * nT + nz * nz);
    // |d nu_z / d s| = E_nu / (2 sqrt(disc))   (= 1/|2(E_l nu_z/E_nu - l_z)| at the root)
    R jac = En / (R(2) * rt);
    V4<R> nu = {En, mx, my, nz};
    V4<R> P = l + nu;
    R x1, x2;
    if (!beam_fractions<R>(p, P.E, P.z, &x1, &x2)) continue;
    R q1[4], q2[4], la[4], na[4];
    beams<R>(p, x1, x2, q1, q2); to_arr(l, la); to_arr(nu, na);
    // flavour sum = both beam orderings (u from beam 1 or from beam 2), reading A4; the W mass
    // is the mapped variable, so its propagator is D(m Gam tan t) (reading O6)
    R me = me_w_D<R>(p, q1, la, DW) + me_w_D<R>(p, q2, la, DW);
    R ff = R(p->pdf_A_q) * R(p->pdf_A_q) * pdf_shape<R>(p, x1) * pdf_shape<R>(p, x2);
    R flux = x1 * x2 * S / R(4);                       // |q1||q2|, Eq. 1
    R w_root = ff * me / flux / (R(8) * pi_<R>() * pi_<R>() * S * l.E * En);
    sum += jac * w_root;
    if (dbg) { R mom[8]; to_arr(l, mom); to_arr(nu, mom + 4); dbg_store<R>(dbg, n_sol, 2, x1, x2, mom); }
    ++n_sol;
  }
  if (dbg) dbg[0] = n_sol;
  return dt * dsdt * sum;
}

// ---------------- config 2: q qbar -> Z -> b bbar, D = 2 ----------------
// rec = [E1, eta1, phi1, E2, eta2, phi2]   (SURVEY.md 8(c) "Config 2")
template <typename R> R weight_z_bb(const orc_params* p, const double* rec, const double* u, double* dbg) {
  const R S = R(p->sqrt_s) * R(p->sqrt_s), dr = R(p->jetE_rhi) - R(p->jetE_rlo);
  const R twopi3 = R(8) * pi_<R>() * pi_<R>() * pi_<R>();
  if (dbg) dbg[0] = 0;
  R Ej[2] = {rec[0], rec[3]}, eta[2] = {rec[1], rec[4]}, phi[2] = {rec[2], rec[5]};
  R E[2], mom[8], vol = R(1), tf = R(1), meas = R(1);
  V4<R> P = {0, 0, 0, 0};
  for (int j = 0; j < 2; ++j) {
    E[j] = Ej[j] * (R(p->jetE_rlo) + dr * R(u[j]));
    vol *= Ej[j] * dr;
    tf *= tf_jet<R>(p, Ej[j], E[j]);
    meas *= E[j] * (R(1) / std::cosh(eta[j])) / (R(2) * twopi3);   // E sin(theta) dE / (2 (2pi)^3)
    V4<R> q = from_E_eta_phi<R>(E[j], eta[j], phi[j]);
    to_arr(q, mom + 4 * j);
    P = P + q;
  }
  R Parr[4]; to_arr(P, Parr);
  boost_transverse<R>(Parr, 2, mom);                   // O7
  R PE = mom[0] + mom[4], Pzz = mom[3] + mom[7];
  R x1, x2;
  if (!beam_fractions<R>(p, PE, Pzz, &x1, &x2)) return R(0);
  R q1[4], q2[4];
  beams<R>(p, x1, x2, q1, q2);
  R me = R(0);
  for (int f = 0; f < p->n_flav; ++f)                  // q from beam 1 or beam 2
    me += me_z<R>(p, flavour_is_up(f), q1, q2, mom, mom + 4) + me_z<R>(p, flavour_is_up(f), q2, q1, mom, mom + 4);
  R ff = R(p->pdf_A_q) * R(p->pdf_A_q) * pdf_shape<R>(p, x1) * pdf_shape<R>(p, x2);
  R flux = x1 * x2 * S / R(4);
  dbg_store<R>(dbg, 0, 2, x1, x2, mom);
  if (dbg) dbg[0] = 1;
  return vol * tf * meas * (R(16) * pi_<R>() * pi_<R>() * pi_<R>() * pi_<R>()) * (R(2) / S) * ff * me / flux;
}

// ---------------- config 3: t tbar -> b l nu  bbar q qbar', D = 6 ----------------
// rec = [lep_pT, lep_eta, lep_phi, (E,eta,phi) x {b_had, b_lep, q, qbar'}, met, met_phi]
// (SURVEY.md 8(c) "Config 3", reading A7)
template <typename R> R weight_tt_ljets(const orc_params* p, const double* rec, const double* u, double* dbg) {
  const R S = R(p->sqrt_s) * R(p->sqrt_s), dr = R(p->jetE_rhi) - R(p->jetE_rlo), H = p->nu_eta_max;
  const R twopi3 = R(8) * pi_<R>() * pi_<R>() * pi_<R>();
  if (dbg) dbg[0] = 0;
  const R lpT = rec[0], leta = rec[1], lphi = rec[2], met_phi = rec[16];
  V4<R> l = from_pt_eta_phi<R>(lpT, leta, lphi);
  V4<R> jet[4];
  R vol = R(1), tf = R(1), meas = R(1);
  for (int j = 0; j < 4; ++j) {
    R Ej = rec[3 + 3 * j], eta = rec[4 + 3 * j], phi = rec[5 + 3 * j];
    R E = Ej * (R(p->jetE_rlo) + dr * R(u[j]));
    vol *= Ej * dr;
    tf *= tf_jet<R>(p, Ej, E);
    meas *= E * (R(1) / std::cosh(eta)) / (R(2) * twopi3);
    jet[j] = from_E_eta_phi<R>(E, eta, phi);
  }
  const V4<R> &b_had = jet[0], &b_lep = jet[1], &q = jet[2], &qb = jet[3];
  // neutrino: eta flat in [-H, H]; leptonic W mass BW-mapped; azimuth = MET azimuth
  R eta_nu = -H + R(2) * H * R(u[4]);
  vol *= R(2) * H;
  R mW = p->m_W, GW = p->Gam_W, n = p->bw_nwidths;
  R t_lo, t_hi;
  bw_window<R>(mW, GW, (mW - n * GW) * (mW - n * GW), (mW + n * GW) * (mW + n * GW), &t_lo, &t_hi);
  R t = t_lo + (t_hi - t_lo) * R(u[5]);
  vol *= (t_hi - t_lo);
  R smm, dsdt, DW_lep;
  bw_point<R>(mW, GW, t, &smm, &dsdt, &DW_lep);
  R sW = mW * mW + smm;
  R den = R(2) * lpT * (std::cosh(leta - eta_nu) - std::cos(lphi - met_phi));
  if (!(den > R(0))) return R(0);
  R nuT = sW / den;
  V4<R> nu = from_pt_eta_phi<R>(nuT, eta_nu, met_phi);
  meas *= R(1) / (R(2) * l.E * twopi3);                // lepton: delta TF
  meas *= nuT * nuT / (R(2) * sW * twopi3);            // d^3nu/((2pi)^3 2E) -> ds_W d eta_nu
  V4<R> pt = b_lep + l + nu, ptb = b_had + q + qb;
  R st = dot(pt, pt), stb = dot(ptb, ptb);
  // O7 boost of the six final-state momenta: order l, nu, b_lep, b_had, q, qbar'
  R mom[24];
  to_arr(l, mom); to_arr(nu, mom + 4); to_arr(b_lep, mom + 8); to_arr(b_had, mom + 12);
  to_arr(q, mom + 16); to_arr(qb, mom + 20);
  V4<R> P = pt + ptb;
  R Parr[4]; to_arr(P, Parr);
  if (!(P.x * P.x + P.y * P.y < P.E * P.E)) return R(0);
  boost_transverse<R>(Parr, 6, mom);
  R PE = 0, Pzz = 0;
  for (int i = 0; i < 6; ++i) { PE += mom[4 * i]; Pzz += mom[4 * i + 3]; }
  R x1, x2;
  if (!beam_fractions<R>(p, PE, Pzz, &x1, &x2)) return R(0);
  R shat = x1 * x2 * S;
  if (!(R(4) * R(p->m_t) * R(p->m_t) < shat)) return R(0);     // rho >= 1 -> 0 (A9)
  R q1[4], q2[4], pta[4], ptba[4];
  beams<R>(p, x1, x2, q1, q2);
  for (int k = 0; k < 4; ++k) { pta[k] = mom[k] + mom[4 + k] + mom[8 + k]; ptba[k] = mom[12 + k] + mom[16 + k] + mom[20 + k]; }
  R prod = tt_flavour_sum<R>(p, x1, x2, me_tt_gg<R>(p, q1, q2, pta, ptba), me_tt_qq<R>(p, q1, q2, pta, ptba));   // includes the PDFs
  // narrow-width factorised decays, 1/2 = average over the decaying top's spin.  The leptonic
  // W mass is the mapped variable: its propagator is D(m Gam tan t) (reading O6).
  R dec_lep = R(0.5) * me_top_decay_D<R>(p, R(1), pta, mom + 8, mom, mom + 4, DW_lep);
  R dec_had = R(0.5) * R(p->V_ud) * R(p->V_ud) * me_top_decay<R>(p, R(3), ptba, mom + 12, mom + 16, mom + 20);
  R mt = p->m_t, Gt = p->Gam_t;
  R Dt = bw_D<R>(st - mt * mt, mt, Gt), Dtb = bw_D<R>(stb - mt * mt, mt, Gt);
  R me = prod * Dt * Dtb * dec_lep * dec_had;
  R ff = R(1);                                  // PDFs are inside prod (tt_flavour_sum)
  R flux = x1 * x2 * S / R(4);
  dbg_store<R>(dbg, 0, 6, x1, x2, mom);
  if (dbg) dbg[0] = 1;
  R w = vol * dsdt * tf * meas * (R(16) * pi_<R>() * pi_<R>() * pi_<R>() * pi_<R>()) * (R(2) / S) * ff * me / flux;
  return std::isfinite(w) ? w : R(0);
}

// ---------------- config 4: t tbar -> b l+ nu  bbar l- nubar, D = 8 ----------------
// rec = [(pT,eta,phi) l+, (pT,eta,phi) l-, (E,eta,phi) b, (E,eta,phi) bbar, met_x, met_y]
// (readings A3, A8, A12; Eq. 7-8)

// Largest real root of z^3 + c2 z^2 + c1 z + c0 (textbook: depressed cubic, Cardano for one real
// root, trigonometric form for three), then Newton on the cubic until it stops moving.
template <typename R> R cubic_largest_root(R c2, R c1, R c0) {
  const R sh = c2 / R(3);
  const R P = c1 - c2 * c2 / R(3);
  const R Q = R(2) * c2 * c2 * c2 / R(27) - c2 * c1 / R(3) + c0;
  const R disc = Q * Q / R(4) + P * P * P / R(27);
  R w;
  if (disc > R(0)) {
    const R sq = std::sqrt(disc);
    const R A = (Q > R(0)) ? -std::cbrt(Q / R(2) + sq) : std::cbrt(-Q / R(2) + sq);
    const R B = (A != R(0)) ? -P / (R(3) * A) : R(0);
    w = A + B;
  } else {
    const R m = std::sqrt(-P / R(3));
    if (m == R(0)) w = R(0);
    else {
      R c = (R(-0.5) * Q) / (m * m * m);
      if (c > R(1)) c = R(1);
      if (c < R(-1)) c = R(-1);
      w = R(2) * m * std::cos(std::acos(c) / R(3));
    }
  }
  R z = w - sh;
  for (int it = 0; it < 30; ++it) {
    const R f = ((z + c2) * z + c1) * z + c0;
    const R fp = (R(3) * z + R(2) * c2) * z + c1;
    if (!(fp != R(0))) break;
    const R zn = z - f / fp;
    if (!std::isfinite((double)zn)) break;
    const bool done = std::fabs(zn - z) <= R(4) * std::numeric_limits<R>::epsilon() * std::fabs(zn);
    z = zn;
    if (done) break;
  }
  return z;
}

// Real roots of q4 x^4 + q3 x^3 + q2 x^2 + q1 x + q0 by Ferrari's method: depress, take the
// largest root z0 of the resolvent cubic z^3 + 2p z^2 + (p^2 - 4r) z - q^2, split into
// (y^2 + s y + m)(y^2 - s y + n), s = sqrt(z0), m,n = (p + z0 -+ q/s)/2.  A quadratic factor has
// real roots iff its discriminant is >= 0.  Returns the number of real roots (0, 2 or 4).
template <typename R> int quartic_real_roots(R q4, R q3, R q2, R q1, R q0, R* x) {
  if (!(q4 != R(0))) return 0;
  const R a3 = q3 / q4, a2 = q2 / q4, a1 = q1 / q4, a0 = q0 / q4;
  const R p = a2 - R(3) * a3 * a3 / R(8);
  const R q = a1 - a3 * a2 / R(2) + a3 * a3 * a3 / R(8);
  const R r = a0 - a3 * a1 / R(4) + a3 * a3 * a2 / R(16) - R(3) * a3 * a3 * a3 * a3 / R(256);
  const R shift = -a3 / R(4);
  R z0 = cubic_largest_root<R>(R(2) * p, p * p - R(4) * r, -q * q);
  if (!(z0 > R(0))) z0 = R(0);
  const R s = std::sqrt(z0);
  // q/s = sign(q) sqrt((p + z0)^2 - 4 r) (from the resolvent); use the quotient unless s vanishes
  R qs;
  if (s > R(0)) qs = q / s;
  else { R t = p * p - R(4) * r; qs = (t > R(0)) ? std::sqrt(t) : R(0); }
  const R m = (p + z0 - qs) / R(2), n = (p + z0 + qs) / R(2);
  int cnt = 0;
  const R d1 = z0 - R(4) * m;          // y^2 + s y + m
  if (d1 >= R(0)) {
    const R sq = std::sqrt(d1);
    const R ya = (-s - sq) / R(2);     // the larger-magnitude root first (s >= 0), the other from the product
    const R yb = (ya != R(0)) ? m / ya : (-s + sq) / R(2);
    x[cnt++] = ya + shift; x[cnt++] = yb + shift;
  }
  const R d2 = z0 - R(4) * n;          // y^2 - s y + n
  if (d2 >= R(0)) {
    const R sq = std::sqrt(d2);
    const R ya = (s + sq) / R(2);
    const R yb = (ya != R(0)) ? n / ya : (s - sq) / R(2);
    x[cnt++] = ya + shift; x[cnt++] = yb + shift;
  }
  return cnt;
}

// One top side of PAPER.md:113-118 Eq. 8 (reading A3: ordinary invariant masses): the neutrino
// momenta with (l + nu)^2 = sW and (b + l + nu)^2 = st lie on the plane d.nu = kappa and satisfy
// E_nu = w0 + n_l.nu.  In terms of (x, y) = (nu_x, nu_y):
//   nu_z = al0 + alx x + aly y,   E_nu = la0 + lax x + lay y.
template <typename R> struct TopSide {
  R al0, alx, aly, la0, lax, lay;
  bool ok;
};
template <typename R> TopSide<R> top_side(const V4<R>& l, const V4<R>& b, R sW, R st) {
  TopSide<R> t;
  const R nlx = l.x / l.E, nly = l.y / l.E, nlz = l.z / l.E;
  const R nbx = b.x / b.E, nby = b.y / b.E, nbz = b.z / b.E;
  const R mbl2 = R(2) * dot(b, l);
  const R Delta = st - sW - mbl2;                 // 2 b.nu
  const R w0 = sW / (R(2) * l.E);
  const R kappa = Delta / (R(2) * b.E) - w0;
  const R dx = nlx - nbx, dy = nly - nby, dz = nlz - nbz;
  t.ok = (Delta > R(0)) && (dz != R(0));
  t.al0 = kappa / dz; t.alx = -dx / dz; t.aly = -dy / dz;
  t.la0 = w0 + nlz * t.al0; t.lax = nlx + nlz * t.alx; t.lay = nly + nlz * t.aly;
  return t;
}
// conic a x^2 + b xy + c y^2 + d x + e y + f = 0 expressing E_nu^2 = |nu|^2
template <typename R> void side_conic(const TopSide<R>& t, R* k) {
  k[0] = R(1) + t.alx * t.alx - t.lax * t.lax;
  k[1] = R(2) * (t.alx * t.aly - t.lax * t.lay);
  k[2] = R(1) + t.aly * t.aly - t.lay * t.lay;
  k[3] = R(2) * (t.al0 * t.alx - t.la0 * t.lax);
  k[4] = R(2) * (t.al0 * t.aly - t.la0 * t.lay);
  k[5] = t.al0 * t.al0 - t.la0 * t.la0;
}

// All real solutions (nu, nubar) of the six equations of Eq. 8: two W masses, two top masses and
// nu_T + nubar_T = (Sx, Sy).  Resultant quartic in x = nu_x, y from the linear relation, then
// Newton on g1 = |nu| - E_nu(x,y), g2 = |nubar| - E_nubar(Sx-x, Sy-y) (reading A12).
// sol[k] = {nu (E,x,y,z), nubar (E,x,y,z)}.  Returns the number of solutions (0..4).
template <typename R> int dilep_solve(const V4<R>& lp, const V4<R>& b, const V4<R>& lm, const V4<R>& bb,
                                      R sWp, R st, R sWm, R stb, R Sx, R Sy, R sol[4][8]) {
  const TopSide<R> T1 = top_side<R>(lp, b, sWp, st), T2 = top_side<R>(lm, bb, sWm, stb);
  if (!T1.ok || !T2.ok) return 0;
  R k1[6], kb[6], k2[6];
  side_conic<R>(T1, k1);
  side_conic<R>(T2, kb);                          // in (xbar, ybar) = (Sx - x, Sy - y)
  k2[0] = kb[0]; k2[1] = kb[1]; k2[2] = kb[2];
  k2[3] = -R(2) * kb[0] * Sx - kb[1] * Sy - kb[3];
  k2[4] = -R(2) * kb[2] * Sy - kb[1] * Sx - kb[4];
  k2[5] = kb[0] * Sx * Sx + kb[1] * Sx * Sy + kb[2] * Sy * Sy + kb[3] * Sx + kb[4] * Sy + kb[5];
  // as polynomials in y: p_i y^2 + q_i(x) y + r_i(x), p = c, q = b x + e, r = a x^2 + d x + f
  const R U2 = k1[2] * k2[0] - k2[2] * k1[0], U1 = k1[2] * k2[3] - k2[2] * k1[3], U0 = k1[2] * k2[5] - k2[2] * k1[5];
  const R V1 = k1[2] * k2[1] - k2[2] * k1[1], V0 = k1[2] * k2[4] - k2[2] * k1[4];
  const R W3 = k1[1] * k2[0] - k2[1] * k1[0];
  const R W2 = k1[1] * k2[3] + k1[4] * k2[0] - k2[1] * k1[3] - k2[4] * k1[0];
  const R W1 = k1[1] * k2[5] + k1[4] * k2[3] - k2[1] * k1[5] - k2[4] * k1[3];
  const R W0 = k1[4] * k2[5] - k2[4] * k1[5];
  const R R4 = U2 * U2 - V1 * W3;
  const R R3 = R(2) * U2 * U1 - V1 * W2 - V0 * W3;
  const R R2 = U1 * U1 + R(2) * U2 * U0 - V1 * W1 - V0 * W2;
  const R R1 = R(2) * U1 * U0 - V1 * W0 - V0 * W1;
  const R R0 = U0 * U0 - V0 * W0;
  R xr[4];
  const int nr = quartic_real_roots<R>(R4, R3, R2, R1, R0, xr);
  int ns = 0;
  for (int i = 0; i < nr; ++i) {
    R x = xr[i];
    const R V = V1 * x + V0;
    if (!(V != R(0))) continue;
    R y = -((U2 * x + U1) * x + U0) / V;
    // Newton on the un-squared equations
    R nz = 0, En = 0, nbz = 0, Enb = 0;
    bool good = true;
    for (int it = 0; it < 12; ++it) {
      nz = T1.al0 + T1.alx * x + T1.aly * y;
      En = std::sqrt(x * x + y * y + nz * nz);
      const R xb = Sx - x, yb = Sy - y;
      nbz = T2.al0 + T2.alx * xb + T2.aly * yb;
      Enb = std::sqrt(xb * xb + yb * yb + nbz * nbz);
      const R g1 = En - (T1.la0 + T1.lax * x + T1.lay * y);
      const R g2 = Enb - (T2.la0 + T2.lax * xb + T2.lay * yb);
      const R j11 = (x + nz * T1.alx) / En - T1.lax, j12 = (y + nz * T1.aly) / En - T1.lay;
      const R j21 = -((xb + nbz * T2.alx) / Enb - T2.lax), j22 = -((yb + nbz * T2.aly) / Enb - T2.lay);
      const R det = j11 * j22 - j12 * j21;
      if (!(det != R(0)) || !std::isfinite((double)det)) { good = false; break; }
      const R dxn = (g1 * j22 - g2 * j12) / det, dyn = (j11 * g2 - j21 * g1) / det;
      x -= dxn; y -= dyn;
      if (std::fabs(dxn) + std::fabs(dyn) <= R(8) * std::numeric_limits<R>::epsilon() * (std::fabs(x) + std::fabs(y)))
        break;
    }
    if (!good) continue;
    nz = T1.al0 + T1.alx * x + T1.aly * y;
    const R xb = Sx - x, yb = Sy - y;
    nbz = T2.al0 + T2.alx * xb + T2.aly * yb;
    En = T1.la0 + T1.lax * x + T1.lay * y;        // E from the W-mass equation (linear form)
    Enb = T2.la0 + T2.lax * xb + T2.lay * yb;
    if (!(En > R(0)) || !(Enb > R(0))) continue;   // the squared equation also has E < 0 branches
    // the polished point must still solve the squared equations (a diverged Newton does not)
    const R c1 = std::sqrt(x * x + y * y + nz * nz), c2 = std::sqrt(xb * xb + yb * yb + nbz * nbz);
    if (!(std::fabs(c1 - En) <= R(1e-9) * (c1 + En)) || !(std::fabs(c2 - Enb) <= R(1e-9) * (c2 + Enb))) continue;
    R* s = sol[ns++];
    s[0] = c1; s[1] = x; s[2] = y; s[3] = nz; s[4] = c2; s[5] = xb; s[6] = yb; s[7] = nbz;
  }
  return ns;
}

// |d(s_W+, s_t, s_W-, s_tbar, S_x, S_y)/d(nu, nubar)|^-1 at one solution:
// with A = grad_nu s_W+ = 2(E_l nuhat - l), B = grad_nu s_t = 2((E_l + E_b) nuhat - (l + b)) and
// C, D likewise on the antitop side, the 6x6 determinant equals [(A x B) x (C x D)]_z.
template <typename R> R dilep_jacobian(const V4<R>& lp, const V4<R>& b, const V4<R>& lm, const V4<R>& bb, const R* s) {
  auto grads = [](const V4<R>& l, const V4<R>& bq, const R* nu, R* A, R* B) {
    const R hx = nu[1] / nu[0], hy = nu[2] / nu[0], hz = nu[3] / nu[0];
    A[0] = R(2) * (l.E * hx - l.x); A[1] = R(2) * (l.E * hy - l.y); A[2] = R(2) * (l.E * hz - l.z);
    B[0] = R(2) * ((l.E + bq.E) * hx - (l.x + bq.x)); B[1] = R(2) * ((l.E + bq.E) * hy - (l.y + bq.y));
    B[2] = R(2) * ((l.E + bq.E) * hz - (l.z + bq.z));
  };
  auto cross = [](const R* a, const R* c, R* o) {
    o[0] = a[1] * c[2] - a[2] * c[1]; o[1] = a[2] * c[0] - a[0] * c[2]; o[2] = a[0] * c[1] - a[1] * c[0];
  };
  R A[3], B[3], Cc[3], Dd[3], P[3], Q[3], X[3];
  grads(lp, b, s, A, B);
  grads(lm, bb, s + 4, Cc, Dd);
  cross(A, B, P); cross(Cc, Dd, Q); cross(P, Q, X);
  return R(1) / std::fabs(X[2]);
}

template <typename R> R weight_tt_dilep(const orc_params* p, const double* rec, const double* u, double* dbg) {
  const R S = R(p->sqrt_s) * R(p->sqrt_s), dr = R(p->jetE_rhi) - R(p->jetE_rlo);
  const R twopi3 = R(8) * pi_<R>() * pi_<R>() * pi_<R>();
  if (dbg) dbg[0] = 0;
  V4<R> lp = from_pt_eta_phi<R>(rec[0], rec[1], rec[2]), lm = from_pt_eta_phi<R>(rec[3], rec[4], rec[5]);
  const R met_x = rec[12], met_y = rec[13];
  V4<R> jet[2];
  R vol = R(1), tf = R(1), meas = R(1);
  for (int j = 0; j < 2; ++j) {
    R Ej = rec[6 + 3 * j], eta = rec[7 + 3 * j], phi = rec[8 + 3 * j];
    R E = Ej * (R(p->jetE_rlo) + dr * R(u[j]));
    vol *= Ej * dr;
    tf *= tf_jet<R>(p, Ej, E);
    meas *= E * (R(1) / std::cosh(eta)) / (R(2) * twopi3);
    jet[j] = from_E_eta_phi<R>(E, eta, phi);
  }
  const V4<R> &b = jet[0], &bb = jet[1];
  // four Breit-Wigner mapped masses: u2 -> s_W+, u3 -> s_t, u4 -> s_W-, u5 -> s_tbar (O6)
  const R mW = p->m_W, GW = p->Gam_W, mt = p->m_t, Gt = p->Gam_t, n = p->bw_nwidths;
  R tWlo, tWhi, tTlo, tThi;
  bw_window<R>(mW, GW, (mW - n * GW) * (mW - n * GW), (mW + n * GW) * (mW + n * GW), &tWlo, &tWhi);
  bw_window<R>(mt, Gt, (mt - n * Gt) * (mt - n * Gt), (mt + n * Gt) * (mt + n * Gt), &tTlo, &tThi);
  R smm[4], dsdt[4], Dk[4];
  for (int k = 0; k < 4; ++k) {
    const bool isW = (k == 0 || k == 2);
    const R lo = isW ? tWlo : tTlo, hi = isW ? tWhi : tThi;
    const R t = lo + (hi - lo) * R(u[2 + k]);
    vol *= (hi - lo);
    bw_point<R>(isW ? mW : mt, isW ? GW : Gt, t, &smm[k], &dsdt[k], &Dk[k]);
  }
  const R sWp = mW * mW + smm[0], st = mt * mt + smm[1], sWm = mW * mW + smm[2], stb = mt * mt + smm[3];
  // total neutrino transverse momentum, flat +-n sigma around the measured MET, Gaussian MET TF (A8)
  const R sig = p->met_sigma, ns = p->met_nsigma;
  const R Sx = met_x + sig * ns * (R(2) * R(u[6]) - R(1)), Sy = met_y + sig * ns * (R(2) * R(u[7]) - R(1));
  vol *= (R(2) * ns * sig) * (R(2) * ns * sig);
  const R ddx = met_x - Sx, ddy = met_y - Sy;
  const R tmet = std::exp(-(ddx * ddx + ddy * ddy) / (R(2) * sig * sig)) / (R(2) * pi_<R>() * sig * sig);
  meas *= R(1) / (R(2) * lp.E * twopi3) * R(1) / (R(2) * lm.E * twopi3);   // leptons: delta TF
  R sol[4][8];
  const int nsol = dilep_solve<R>(lp, b, lm, bb, sWp, st, sWm, stb, Sx, Sy, sol);
  R sum = R(0);
  int kept = 0;
  for (int k = 0; k < nsol; ++k) {
    const R J = dilep_jacobian<R>(lp, b, lm, bb, sol[k]);
    V4<R> nu = from_arr(sol[k]), nub = from_arr(sol[k] + 4);
    // O7 boost of the six final momenta: order l+, nu, b, l-, nubar, bbar
    R mom[24];
    to_arr(lp, mom); to_arr(nu, mom + 4); to_arr(b, mom + 8); to_arr(lm, mom + 12); to_arr(nub, mom + 16);
    to_arr(bb, mom + 20);
    V4<R> P = lp + nu + b + lm + nub + bb;
    R Parr[4]; to_arr(P, Parr);
    if (!(P.x * P.x + P.y * P.y < P.E * P.E)) continue;
    boost_transverse<R>(Parr, 6, mom);
    R PE = 0, Pzz = 0;
    for (int i = 0; i < 6; ++i) { PE += mom[4 * i]; Pzz += mom[4 * i + 3]; }
    R x1, x2;
    if (!beam_fractions<R>(p, PE, Pzz, &x1, &x2)) continue;
    const R shat = x1 * x2 * S;
    if (!(R(4) * mt * mt < shat)) continue;                       // A9
    R q1[4], q2[4], pta[4], ptba[4];
    beams<R>(p, x1, x2, q1, q2);
    for (int c = 0; c < 4; ++c) { pta[c] = mom[c] + mom[4 + c] + mom[8 + c]; ptba[c] = mom[12 + c] + mom[16 + c] + mom[20 + c]; }
    const R prod = tt_flavour_sum<R>(p, x1, x2, me_tt_gg<R>(p, q1, q2, pta, ptba), me_tt_qq<R>(p, q1, q2, pta, ptba));   // includes the PDFs
    // t -> b l+ nu: (p_t.p_l+)(p_b.p_nu);  tbar -> bbar l- nubar: (p_tbar.p_l-)(p_bbar.p_nubar)
    const R dec1 = R(0.5) * me_top_decay_D<R>(p, R(1), pta, mom + 8, mom, mom + 4, Dk[0]);
    const R dec2 = R(0.5) * me_top_decay_D<R>(p, R(1), ptba, mom + 20, mom + 12, mom + 16, Dk[2]);
    const R me = prod * Dk[1] * Dk[3] * dec1 * dec2;
    const R ff = R(1);                                  // PDFs are inside prod (tt_flavour_sum)
    const R flux = x1 * x2 * S / R(4);
    const R ws = J / (twopi3 * twopi3 * R(4) * nu.E * nub.E) * ff * me / flux;
    if (!std::isfinite((double)ws)) continue;
    sum += ws;
    dbg_store<R>(dbg, kept, 6, x1, x2, mom);
    ++kept;
  }
  if (dbg) dbg[0] = kept;
  R w = vol * dsdt[0] * dsdt[1] * dsdt[2] * dsdt[3] * tf * tmet * meas *
        (R(16) * pi_<R>() * pi_<R>() * pi_<R>() * pi_<R>()) * (R(2) / S) * sum;
  return std::isfinite((double)w) ? w : R(0);
}

// ---------------- NEXT-4: t tbar H(-> b bbar), dilepton, four b jets, D = 8 ----------------
// PAPER.md:101-109 Eq. 7 (the paper's own benchmark integral: four jet-energy TFs, the two neutrinos
// fixed by the MET delta functions), :111-118 Eq. 8 (neutrino momenta -> q^2 of the W and top
// propagators), :120-137 Eq. 9 (Higgs b-quark energies (E1, E2) -> (f = E1 + E2, m_H^2)), :178-180
// Eq. 11 (the MET entering Eq. 8 is minus the visible transverse momentum of the point, so the total
// transverse momentum vanishes and the O7 boost is the identity: it is not applied).
// rec = [(pT,eta,phi) l+, (pT,eta,phi) l-, (E,eta,phi) x {b, bbar, b1, b2}]: b pairs with l+ (top),
// bbar with l- (antitop), b1 b2 are the Higgs candidates.  No measured MET enters (Eq. 11).
// DESIGN.md "NEXT-4" readings A18-A21.

// Eq. 9 for massless b quarks ("E is set to |p|"): f = E1 + E2, m^2 = 2 E1 E2 K12 with
// K12 = 1 - cos(Delta theta_12).  Inverse: E1 E2 = m^2/(2 K12), so E1, E2 = (f +- sqrt(f^2 - 2 m^2/K12))/2:
// the map is two-to-one (E1 <-> E2) and BOTH orderings are returned (reading A19);
// |d(E1,E2)/d(f,m^2)| = 1/(2 K12 |E1 - E2|).  Returns 0 or 2.
template <typename R> int eq9_roots(R K12, R f, R sH, R E1[2], R E2[2], R* jac) {
  const R disc = f * f - R(2) * sH / K12;
  if (!(disc > R(0))) return 0;
  const R rt = std::sqrt(disc);
  E1[0] = (f + rt) / R(2); E2[0] = (f - rt) / R(2);
  E1[1] = E2[0]; E2[1] = E1[0];
  *jac = R(1) / (R(2) * K12 * rt);
  return 2;
}

// Factorised matrix-element pieces of the two hypotheses (reading A20; SURVEY.md 8(f)-4 "factorised
// t tbar H ME ... a second factorised hypothesis"): radiation of the b bbar system k = p_b1 + p_b2 off the
// top pair, the propagator of what was radiated, and its decay into b bbar.
//   hyp 0, t tbar H: soft-scalar (eikonal) emission off either top, y_t^2 4 m_t^2 (1/X_t + 1/X_tbar)^2 with
//          X = 2 p.k + k^2; Higgs propagator D_H(k^2); sum |M(H -> b bbar)|^2 = 3 y_b^2 2 k^2 (massless b)
//   hyp 1, non-resonant t tbar b bbar: eikonal vector emission g_s^2 (-J^2),
//          J = p_t/(p_t.k) - p_tbar/(p_tbar.k) (>= 0 for timelike k); propagator 1/k^4; splitting g_s^2 k^2;
//          colour factors set to 1.
template <typename R> R tth_radiator(const orc_params* p, const V4<R>& pt, const V4<R>& ptb, const V4<R>& k) {
  const R sH = dot(k, k);
  if (p->tth_hyp == 0) {
    const R Xt = R(2) * dot(pt, k) + sH, Xtb = R(2) * dot(ptb, k) + sH;
    const R a = R(1) / Xt + R(1) / Xtb;
    return R(p->yuk_t) * R(p->yuk_t) * R(4) * R(p->m_t) * R(p->m_t) * a * a;
  }
  const R tk = dot(pt, k), tbk = dot(ptb, k);
  return gs2<R>(p) * (R(2) * dot(pt, ptb) / (tk * tbk) - dot(pt, pt) / (tk * tk) - dot(ptb, ptb) / (tbk * tbk));
}
template <typename R> R tth_decay(const orc_params* p, R sH) {
  if (p->tth_hyp == 0) return R(3) * R(p->yuk_b) * R(p->yuk_b) * R(2) * sH;
  return gs2<R>(p) * sH;
}

// t tbar production next to a third body (reading A20): tau1, tau2 of reading A9 normalised to
// tau1 + tau2 = 1, rho = 4 m_t^2 / (p_t + p_tbar)^2; 0 unless rho < 1.
template <typename R> bool tth_tt_invariants(const orc_params* p, const R q1[4], const R q2[4], const V4<R>& t,
                                             const V4<R>& tb, R* t1, R* t2, R* rho) {
  V4<R> a = from_arr(q1), b = from_arr(q2);
  const R n1 = dot(a, t) + dot(b, tb), n2 = dot(b, t) + dot(a, tb);
  const R stt = dot(t + tb, t + tb);
  if (!(R(4) * R(p->m_t) * R(p->m_t) < stt)) return false;
  *t1 = n1 / (n1 + n2); *t2 = n2 / (n1 + n2);
  *rho = R(4) * R(p->m_t) * R(p->m_t) / stt;
  return true;
}

// Everything that depends on the Higgs b-quark energies (E1, E2): jets b1, b2 with their TFs and measures,
// Eq. 11, the neutrino solutions of Eq. 8, and per solution Jacobian x neutrino measure x PDFs x |M|^2 / flux.
// propH = the propagator factor of the radiated system (D_H from the mapped variable, or 1/k^4).
template <typename R> R tth_core(const orc_params* p, const double* rec, const V4<R>& lp, const V4<R>& lm,
                                 const V4<R>& b, const V4<R>& bb, R E1, R E2, R sWp, R st, R sWm, R stb,
                                 const R Dk[4], R propH, double* dbg, int* kept) {
  const R S = R(p->sqrt_s) * R(p->sqrt_s), mt = p->m_t;
  const R twopi3 = R(8) * pi_<R>() * pi_<R>() * pi_<R>();
  const R Ej1 = rec[12], Ej2 = rec[15];
  const V4<R> b1 = from_E_eta_phi<R>(E1, R(rec[13]), R(rec[14])), b2 = from_E_eta_phi<R>(E2, R(rec[16]), R(rec[17]));
  const R tf12 = tf_jet<R>(p, Ej1, E1) * tf_jet<R>(p, Ej2, E2);
  const R meas12 = E1 * (R(1) / std::cosh(R(rec[13]))) / (R(2) * twopi3) * E2 * (R(1) / std::cosh(R(rec[16]))) / (R(2) * twopi3);
  // Eq. 11: the neutrino pair balances the visible system of THIS point
  const V4<R> vis = lp + lm + b + bb + b1 + b2;
  const R Sx = -vis.x, Sy = -vis.y;
  R sol[4][8];
  const int nsol = dilep_solve<R>(lp, b, lm, bb, sWp, st, sWm, stb, Sx, Sy, sol);
  const V4<R> k = b1 + b2;
  const R sH = dot(k, k);
  R sum = R(0);
  for (int i = 0; i < nsol; ++i) {
    const R J = dilep_jacobian<R>(lp, b, lm, bb, sol[i]);
    V4<R> nu = from_arr(sol[i]), nub = from_arr(sol[i] + 4);
    const V4<R> P = vis + nu + nub;                         // P_T = 0 by construction
    R x1, x2;
    if (!beam_fractions<R>(p, P.E, P.z, &x1, &x2)) continue;
    R q1[4], q2[4];
    beams<R>(p, x1, x2, q1, q2);
    const V4<R> pt = lp + nu + b, ptb = lm + nub + bb;
    R t1, t2, rho;
    if (!tth_tt_invariants<R>(p, q1, q2, pt, ptb, &t1, &t2, &rho)) continue;
    const R prod = tt_flavour_sum<R>(p, x1, x2, me_tt_gg_inv<R>(p, t1, t2, rho), me_tt_qq_inv<R>(p, t1, t2, rho));   // includes the PDFs
    R pta[4], ptba[4], la[4], na[4], ba[4], lma[4], nba[4], bba[4];
    to_arr(pt, pta); to_arr(ptb, ptba); to_arr(lp, la); to_arr(nu, na); to_arr(b, ba);
    to_arr(lm, lma); to_arr(nub, nba); to_arr(bb, bba);
    const R dec1 = R(0.5) * me_top_decay_D<R>(p, R(1), pta, ba, la, na, Dk[0]);
    const R dec2 = R(0.5) * me_top_decay_D<R>(p, R(1), ptba, bba, lma, nba, Dk[2]);
    const R me = prod * tth_radiator<R>(p, pt, ptb, k) * propH * tth_decay<R>(p, sH) * Dk[1] * Dk[3] * dec1 * dec2;
    const R flux = x1 * x2 * S / R(4);
    const R ws = J / (twopi3 * twopi3 * R(4) * nu.E * nub.E) * me / flux;
    if (!std::isfinite((double)ws)) continue;
    sum += ws;
    if (dbg && *kept < 8) {
      R mom[32];
      to_arr(lp, mom); to_arr(nu, mom + 4); to_arr(b, mom + 8); to_arr(lm, mom + 12); to_arr(nub, mom + 16);
      to_arr(bb, mom + 20); to_arr(b1, mom + 24); to_arr(b2, mom + 28);
      dbg_store<R>(dbg, *kept, 8, x1, x2, mom);
    }
    ++*kept;
  }
  (void)mt;
  return tf12 * meas12 * sum;
}

template <typename R> R weight_tth_dilep(const orc_params* p, const double* rec, const double* u, double* dbg) {
  const R S = R(p->sqrt_s) * R(p->sqrt_s), rlo = p->jetE_rlo, rhi = p->jetE_rhi, dr = rhi - rlo;
  const R twopi3 = R(8) * pi_<R>() * pi_<R>() * pi_<R>();
  if (dbg) dbg[0] = 0;
  V4<R> lp = from_pt_eta_phi<R>(rec[0], rec[1], rec[2]), lm = from_pt_eta_phi<R>(rec[3], rec[4], rec[5]);
  V4<R> jet[2];
  R vol = R(1), tf = R(1), meas = R(1);
  for (int j = 0; j < 2; ++j) {                              // b (top side), bbar (antitop side): O5
    R Ej = rec[6 + 3 * j], eta = rec[7 + 3 * j], phi = rec[8 + 3 * j];
    R E = Ej * (rlo + dr * R(u[j]));
    vol *= Ej * dr;
    tf *= tf_jet<R>(p, Ej, E);
    meas *= E * (R(1) / std::cosh(eta)) / (R(2) * twopi3);
    jet[j] = from_E_eta_phi<R>(E, eta, phi);
  }
  const V4<R> &b = jet[0], &bb = jet[1];
  // four Breit-Wigner mapped masses: u2 -> s_W+, u3 -> s_t, u4 -> s_W-, u5 -> s_tbar (O6), as in config 4
  const R mW = p->m_W, GW = p->Gam_W, mt = p->m_t, Gt = p->Gam_t, n = p->bw_nwidths;
  R tWlo, tWhi, tTlo, tThi;
  bw_window<R>(mW, GW, (mW - n * GW) * (mW - n * GW), (mW + n * GW) * (mW + n * GW), &tWlo, &tWhi);
  bw_window<R>(mt, Gt, (mt - n * Gt) * (mt - n * Gt), (mt + n * Gt) * (mt + n * Gt), &tTlo, &tThi);
  R smm[4], dsdt[4], Dk[4];
  for (int k = 0; k < 4; ++k) {
    const bool isW = (k == 0 || k == 2);
    const R lo = isW ? tWlo : tTlo, hi = isW ? tWhi : tThi;
    const R t = lo + (hi - lo) * R(u[2 + k]);
    vol *= (hi - lo);
    bw_point<R>(isW ? mW : mt, isW ? GW : Gt, t, &smm[k], &dsdt[k], &Dk[k]);
  }
  const R sWp = mW * mW + smm[0], st = mt * mt + smm[1], sWm = mW * mW + smm[2], stb = mt * mt + smm[3];
  meas *= R(1) / (R(2) * lp.E * twopi3) * R(1) / (R(2) * lm.E * twopi3);   // leptons: delta TF
  // Higgs candidates b1, b2
  const R Ej1 = rec[12], Ej2 = rec[15];
  const V4<R> n1 = from_E_eta_phi<R>(R(1), R(rec[13]), R(rec[14])), n2 = from_E_eta_phi<R>(R(1), R(rec[16]), R(rec[17]));
  const R K12 = dot(n1, n2);                                 // 1 - cos(Delta theta_12)
  const R mH = p->m_H, GH = p->Gam_H;
  // window of k^2 = (p_b1 + p_b2)^2.  hyp 0: Breit-Wigner window of the Higgs, mapped by O6;
  // hyp 1: everything the two energy windows allow, s in 2 K12 Ej1 Ej2 [rlo^2, rhi^2], mapped with
  // s = s_lo (s_hi/s_lo)^u (flat in ln s, ds/du = s ln(s_hi/s_lo))
  R tHlo = 0, tHhi = 0;
  if (p->tth_hyp == 0) bw_window<R>(mH, GH, (mH - n * GH) * (mH - n * GH), (mH + n * GH) * (mH + n * GH), &tHlo, &tHhi);
  const R s_lo = R(2) * K12 * Ej1 * Ej2 * rlo * rlo, lnr = R(2) * std::log(rhi / rlo);
  int kept = 0;
  R sum = R(0);
  if (p->tth_chart == 0) {
    // Eq. 9 chart: u6 -> k^2, u7 -> f = E1 + E2 flat over the sum of the two energy windows
    R sH, propH, jac_map;
    if (p->tth_hyp == 0) {
      const R t = tHlo + (tHhi - tHlo) * R(u[6]);
      R smH, dsdtH, DH;
      bw_point<R>(mH, GH, t, &smH, &dsdtH, &DH);
      sH = mH * mH + smH; propH = DH; jac_map = (tHhi - tHlo) * dsdtH;
    } else {
      sH = s_lo * std::exp(lnr * R(u[6]));
      propH = R(1) / (sH * sH); jac_map = lnr * sH;
    }
    const R f = (Ej1 + Ej2) * (rlo + dr * R(u[7]));
    const R volf = (Ej1 + Ej2) * dr;
    R E1[2], E2[2], jac9;
    const int nroot = eq9_roots<R>(K12, f, sH, E1, E2, &jac9);
    for (int r = 0; r < nroot; ++r) {
      // a root counts only inside both parton-energy windows, so that the chart covers exactly the box of O5
      if (!(E1[r] >= rlo * Ej1 && E1[r] <= rhi * Ej1 && E2[r] >= rlo * Ej2 && E2[r] <= rhi * Ej2)) continue;
      sum += jac_map * volf * jac9 * tth_core<R>(p, rec, lp, lm, b, bb, E1[r], E2[r], sWp, st, sWm, stb, Dk, propH, dbg, &kept);
    }
  } else {
    // pin chart (tests only): (E1, E2) flat in their windows, k^2 from the momenta
    const R E1 = Ej1 * (rlo + dr * R(u[6])), E2 = Ej2 * (rlo + dr * R(u[7]));
    const R sH = R(2) * E1 * E2 * K12;
    R propH;
    bool inside = true;
    if (p->tth_hyp == 0) {
      inside = (sH >= (mH - n * GH) * (mH - n * GH)) && (sH <= (mH + n * GH) * (mH + n * GH));
      propH = bw_D<R>(sH - mH * mH, mH, GH);
    } else {
      propH = R(1) / (sH * sH);
    }
    if (inside) sum = Ej1 * dr * Ej2 * dr * tth_core<R>(p, rec, lp, lm, b, bb, E1, E2, sWp, st, sWm, stb, Dk, propH, dbg, &kept);
  }
  if (dbg) dbg[0] = kept < 8 ? kept : 8;
  R w = vol * dsdt[0] * dsdt[1] * dsdt[2] * dsdt[3] * tf * meas *
        (R(16) * pi_<R>() * pi_<R>() * pi_<R>() * pi_<R>()) * (R(2) / S) * sum;
  return std::isfinite((double)w) ? w : R(0);
}

// NEXT-1 (Eq. 7: "The outer sum is over all permutations of assigning measured
// jets to partons in the matrix element").  The sum over
// assignments sits outside the integral, i.e. every sample point is evaluated for each assignment:
// w(u) = sum_sigma w(record with its jets reordered by sigma, u).  Parton role r takes measured jet
// sigma[r]; the energy variable u_r stays with the role.  Assignments in lexicographic order.
inline int jet_perms(int process, int n_perm, int perm[24][4]) {
  static const int id[4] = {0, 1, 2, 3};
  int n = 0;
  auto push = [&](int a, int b, int c, int d) { perm[n][0] = a; perm[n][1] = b; perm[n][2] = c; perm[n][3] = d; ++n; };
  if (process == ORC_TT_LJETS && n_perm == 24) {
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) for (int c = 0; c < 4; ++c) for (int d = 0; d < 4; ++d)
      if (a != b && a != c && a != d && b != c && b != d && c != d) push(a, b, c, d);
  } else if (process == ORC_TT_LJETS && n_perm == 4) {
    push(0, 1, 2, 3); push(0, 1, 3, 2); push(1, 0, 2, 3); push(1, 0, 3, 2);
  } else if (process == ORC_TT_DILEP && n_perm == 2) {
    push(0, 1, 2, 3); push(1, 0, 2, 3);
  } else if (process == ORC_TTH_DILEP && n_perm == 12) {
    // roles (b, bbar, b1, b2); the integrand is symmetric in b1 <-> b2 (both Eq. 9 orderings are summed),
    // so the 4!/2 = 12 distinct assignments are the ordered choices of (b, bbar), the remaining two jets
    // in ascending order
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) {
      if (a == b) continue;
      int rest[2], m = 0;
      for (int c = 0; c < 4; ++c) if (c != a && c != b) rest[m++] = c;
      push(a, b, rest[0], rest[1]);
    }
  } else {
    push(id[0], id[1], id[2], id[3]);
  }
  return n;
}

template <typename R> R weight_permuted(int process, const orc_params* p, const double* rec, const double* u,
                                        double* dbg) {
  int perm[24][4];
  const int n = jet_perms(process, p->n_perm, perm);
  const int first_jet = (process == ORC_TT_LJETS) ? 3 : 6;   // record offset of the first (E, eta, phi) triple
  const int n_jets = (process == ORC_TT_DILEP) ? 2 : 4;
  const int nf = orc_n_fields(process);
  R sum = R(0);
  for (int k = 0; k < n; ++k) {
    double r2[32];
    for (int f = 0; f < nf; ++f) r2[f] = rec[f];
    for (int role = 0; role < n_jets; ++role)
      for (int c = 0; c < 3; ++c) r2[first_jet + 3 * role + c] = rec[first_jet + 3 * perm[k][role] + c];
    sum += (process == ORC_TT_LJETS)   ? weight_tt_ljets<R>(p, r2, u, k == 0 ? dbg : nullptr)
           : (process == ORC_TT_DILEP) ? weight_tt_dilep<R>(p, r2, u, k == 0 ? dbg : nullptr)
                                       : weight_tth_dilep<R>(p, r2, u, k == 0 ? dbg : nullptr);
  }
  return sum;
}

// NEXT-2, parton-level mode (Table 2): "the transfer functions are delta
// functions", no integration -- the integrand of Eq. 1 without dPhi at a fully specified partonic
// configuration, summed over the jet-parton assignments (n_perm) and the initial-state flavours:
//   w = sum_sigma  f(x1) f(x2) / (|q1||q2|) * |M|^2(l, nu, b_had, b_lep, q, qbar' [jets reordered by sigma])
// mom = six four-vectors (E, px, py, pz) in the order l, nu, b_had, b_lep, q, qbar'.  The transverse
// boost O7 is applied (identity for a balanced event); all four propagators come from the momenta.
template <typename R> R parton_weight_tt_ljets(const orc_params* p, const double* mom_in) {
  const R S = R(p->sqrt_s) * R(p->sqrt_s), mt = p->m_t, Gt = p->Gam_t;
  int perm[24][4];
  const int n = jet_perms(ORC_TT_LJETS, p->n_perm, perm);
  R sum = R(0);
  for (int k = 0; k < n; ++k) {
    // internal order for the boost: l, nu, b_lep, b_had, q, qbar'
    R mom[24];
    const int role_src[4] = {2 + perm[k][0], 2 + perm[k][1], 2 + perm[k][2], 2 + perm[k][3]};   // b_had, b_lep, q, qbar'
    for (int c = 0; c < 4; ++c) {
      mom[c] = mom_in[c]; mom[4 + c] = mom_in[4 + c];
      mom[8 + c] = mom_in[4 * role_src[1] + c];     // b_lep
      mom[12 + c] = mom_in[4 * role_src[0] + c];    // b_had
      mom[16 + c] = mom_in[4 * role_src[2] + c];    // q
      mom[20 + c] = mom_in[4 * role_src[3] + c];    // qbar'
    }
    R P[4] = {0, 0, 0, 0};
    for (int i = 0; i < 6; ++i) for (int c = 0; c < 4; ++c) P[c] += mom[4 * i + c];
    if (!(P[1] * P[1] + P[2] * P[2] < P[0] * P[0])) continue;
    boost_transverse<R>(P, 6, mom);
    R PE = 0, Pz = 0;
    for (int i = 0; i < 6; ++i) { PE += mom[4 * i]; Pz += mom[4 * i + 3]; }
    R x1, x2;
    if (!beam_fractions<R>(p, PE, Pz, &x1, &x2)) continue;
    const R shat = x1 * x2 * S;
    if (!(R(4) * mt * mt < shat)) continue;                          // A9
    R q1[4], q2[4], pt[4], ptb[4];
    beams<R>(p, x1, x2, q1, q2);
    for (int c = 0; c < 4; ++c) { pt[c] = mom[c] + mom[4 + c] + mom[8 + c]; ptb[c] = mom[12 + c] + mom[16 + c] + mom[20 + c]; }
    const R prod = tt_flavour_sum<R>(p, x1, x2, me_tt_gg<R>(p, q1, q2, pt, ptb), me_tt_qq<R>(p, q1, q2, pt, ptb));   // includes the PDFs
    const R dec_lep = R(0.5) * me_top_decay<R>(p, R(1), pt, mom + 8, mom, mom + 4);
    const R dec_had = R(0.5) * R(p->V_ud) * R(p->V_ud) * me_top_decay<R>(p, R(3), ptb, mom + 12, mom + 16, mom + 20);
    V4<R> t4 = from_arr(pt), tb4 = from_arr(ptb);
    const R Dt = bw_D<R>(dot(t4, t4) - mt * mt, mt, Gt), Dtb = bw_D<R>(dot(tb4, tb4) - mt * mt, mt, Gt);
    const R ff = R(1);                                  // PDFs are inside prod (tt_flavour_sum)
    const R w = ff * prod * Dt * Dtb * dec_lep * dec_had / (x1 * x2 * S / R(4));
    if (std::isfinite((double)w)) sum += w;
  }
  return sum;
}

template <typename R> double weight_any(int process, const orc_params* p, const double* rec, const double* u,
                                        double* dbg) {
  R w = R(0);
  switch (process) {
    case ORC_W_ENU: w = weight_w_enu<R>(p, rec, u, dbg); break;
    case ORC_Z_BB: w = weight_z_bb<R>(p, rec, u, dbg); break;
    case ORC_TT_LJETS: w = weight_permuted<R>(process, p, rec, u, dbg); break;
    case ORC_TT_DILEP: w = weight_permuted<R>(process, p, rec, u, dbg); break;
    case ORC_TTH_DILEP: w = weight_permuted<R>(process, p, rec, u, dbg); break;
    default: return std::nan("");
  }
  double wd = (double)w;
  return std::isfinite(wd) ? wd : 0.0;   // non-finite points contribute 0
}

// VEGAS map (config 5; SURVEY.md 8(c) "Config 5", reading A14)
template <typename R> void vegas_map(const double* edges, int bins, int n_dims, const double* u, R* z, int* k, R* jac) {
  R j = R(1);
  for (int d = 0; d < n_dims; ++d) {
    const double* x = edges + (size_t)d * (bins + 1);
    R y = R(u[d]) * R(bins);
    int kk = (int)std::floor(y);
    if (kk > bins - 1) kk = bins - 1;
    R width = R(x[kk + 1]) - R(x[kk]);
    z[d] = R(x[kk]) + (y - R(kk)) * width;
    j *= R(bins) * width;
    if (k) k[d] = kk;
  }
  *jac = j;
}

void load_record(const double* events, int64_t n_events, int64_t e, int nf, double* rec) {
  for (int f = 0; f < nf; ++f) rec[f] = events[(size_t)f * n_events + e];
}

}  // namespace

extern "C" {

// --------------------------------------------------------------------------
// parameters
// --------------------------------------------------------------------------
int orc_n_fields(int process) {
  switch (process) { case ORC_W_ENU: return 5; case ORC_Z_BB: return 6;
                     case ORC_TT_LJETS: return 17; case ORC_TT_DILEP: return 14; case ORC_TTH_DILEP: return 18; }
  return -1;
}
int orc_n_dims(int process) {
  switch (process) { case ORC_W_ENU: return 1; case ORC_Z_BB: return 2;
                     case ORC_TT_LJETS: return 6; case ORC_TT_DILEP: return 8; case ORC_TTH_DILEP: return 8; }
  return -1;
}

int orc_params_default(int process, orc_params* p) {
  if (!p || orc_n_fields(process) < 0) return 1;
  std::memset(p, 0, sizeof(*p));
  p->sqrt_s = 14000.0;                       // BASELINE.json:configs[0]
  p->G_F = 1.16637e-5; p->alpha_s = 0.118; p->sin2_thw = 0.2312;
  p->m_W = 80.4; p->Gam_W = 2.09;            // configs[0]
  p->m_Z = 91.1876; p->Gam_Z = 2.4952;
  p->m_t = 173.0; p->Gam_t = 1.4;            // configs[2]
  p->V_ud = 1.0; p->V_tb = 1.0;
  p->pdf_A_q = 1.0; p->pdf_A_g = 1.0; p->pdf_pow_x = -0.5; p->pdf_pow_1mx = 3.0;  // configs[0]
  p->tf_w_tail = 0.3; p->tf_mu1 = 0.0; p->tf_sig1 = 0.15; p->tf_mu2 = -0.1; p->tf_sig2 = 0.35;  // configs[1]
  p->jetE_rlo = 0.5; p->jetE_rhi = 2.0; p->bw_nwidths = 15.0;
  p->nu_pz_max = 500.0;                      // configs[0]
  p->nu_eta_max = 5.0; p->met_sigma = 10.0; p->met_nsigma = 4.0;
  p->vegas_alpha = 0.5; p->vegas_points = 1 << 17; p->vegas_iters = 0; p->vegas_bins = 50;  // configs[4]
  p->n_flav = (process == ORC_Z_BB) ? 3 : 5; // configs[1] "u,d,s"; PAPER.md:141 (d,u,s,c,b)
  // NEXT-4 (reading A21; the paper gives none): m_H = 125, Gamma_H = 4.07 MeV ("very narrow"),
  // Yukawa couplings y_f = m_f sqrt(2 sqrt2 G_F) with m_b = 4.18 in the coupling only (kinematics massless)
  p->m_H = 125.0; p->Gam_H = 0.00407;
  p->yuk_t = p->m_t * std::sqrt(2.0 * std::sqrt(2.0) * p->G_F);
  p->yuk_b = 4.18 * std::sqrt(2.0 * std::sqrt(2.0) * p->G_F);
  p->tth_hyp = 0; p->tth_chart = 0;
  return 0;
}

// --------------------------------------------------------------------------
// O2. Philox4x32-10 and the 52-bit uniform
// --------------------------------------------------------------------------
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t m0 = (uint64_t)0xD2511F53u * c0;
    uint64_t m1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t hi0 = (uint32_t)(m0 >> 32), lo0 = (uint32_t)m0;
    uint32_t hi1 = (uint32_t)(m1 >> 32), lo1 = (uint32_t)m1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

double orc_u52(uint32_t a, uint32_t b) {
  uint64_t k = ((uint64_t)(a >> 6) << 26) | (uint64_t)(b >> 6);   // 52 bits
  return ((double)k + 0.5) * (1.0 / 4503599627370496.0);          // 2^-52, exact, in (0,1)
}

void orc_uniforms(uint64_t seed, uint64_t event, uint64_t point, uint32_t iteration,
                  int n_dims, double* u) {
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  for (int j = 0; 2 * j < n_dims; ++j) {
    uint32_t ctr[4] = {(uint32_t)point, (uint32_t)(point >> 32), (uint32_t)event,
                       iteration * 256u + (uint32_t)j};
    uint32_t r[4];
    orc_philox4x32_10(ctr, key, r);
    u[2 * j] = orc_u52(r[0], r[1]);
    if (2 * j + 1 < n_dims) u[2 * j + 1] = orc_u52(r[2], r[3]);
  }
}

// --------------------------------------------------------------------------
// building blocks, fp64 instantiations
// --------------------------------------------------------------------------
double orc_pdf_shape(const orc_params* p, double x) { return pdf_shape<double>(p, x); }
double orc_tf_jet(const orc_params* p, double E_jet, double E) { return tf_jet<double>(p, E_jet, E); }
void orc_bw_window(double m, double Gam, double s_lo, double s_hi, double* t_lo, double* t_hi) {
  bw_window<double>(m, Gam, s_lo, s_hi, t_lo, t_hi);
}
void orc_bw_point(double m, double Gam, double t, double* s_minus_m2, double* dsdt, double* D) {
  bw_point<double>(m, Gam, t, s_minus_m2, dsdt, D);
}
double orc_me_w(const orc_params* p, const double qa[4], const double qb[4], const double lep[4], const double nu[4]) {
  return me_w<double>(p, qa, qb, lep, nu);
}
double orc_me_z(const orc_params* p, int up_type, const double qa[4], const double qb[4], const double p1[4],
                const double p2[4]) {
  return me_z<double>(p, up_type, qa, qb, p1, p2);
}
double orc_me_tt_qq(const orc_params* p, const double q1[4], const double q2[4], const double pt[4], const double ptb[4]) {
  return me_tt_qq<double>(p, q1, q2, pt, ptb);
}
double orc_me_tt_gg(const orc_params* p, const double q1[4], const double q2[4], const double pt[4], const double ptb[4]) {
  return me_tt_gg<double>(p, q1, q2, pt, ptb);
}
double orc_me_top_decay(const orc_params* p, double n_c, const double pt[4], const double pb[4],
                        const double pf_down[4], const double pf_up[4]) {
  return me_top_decay<double>(p, n_c, pt, pb, pf_down, pf_up);
}
void orc_boost_transverse(const double P[4], int n, double* mom) { boost_transverse<double>(P, n, mom); }

// config-4 building blocks (pinned by tests/test_oracle_dilep.py)
int orc_quartic_real_roots(const double q[5], double x[4]) {
  return quartic_real_roots<double>(q[4], q[3], q[2], q[1], q[0], x);
}
int orc_dilep_solve(const double lp[4], const double b[4], const double lm[4], const double bb[4],
                    double sWp, double st, double sWm, double stb, double Sx, double Sy,
                    double* sol /* [4][8] */, double* jac /* [4] */) {
  V4<double> a = from_arr(lp), c = from_arr(b), d = from_arr(lm), e = from_arr(bb);
  double s[4][8];
  int n = dilep_solve<double>(a, c, d, e, sWp, st, sWm, stb, Sx, Sy, s);
  for (int k = 0; k < n; ++k) {
    for (int i = 0; i < 8; ++i) sol[8 * k + i] = s[k][i];
    jac[k] = dilep_jacobian<double>(a, c, d, e, s[k]);
  }
  return n;
}

// NEXT-2: parton-level weights of n_events configurations, SoA field-major [24][n_events]
int orc_parton_weights(int process, const orc_params* p, const double* mom, int64_t n_events, int extended,
                       double* out_w) {
  if (process != ORC_TT_LJETS || !p || !mom || !out_w) return 1;
  for (int64_t e = 0; e < n_events; ++e) {
    double m[24];
    for (int f = 0; f < 24; ++f) m[f] = mom[(size_t)f * n_events + e];
    double w = extended ? (double)parton_weight_tt_ljets<long double>(p, m) : (double)parton_weight_tt_ljets<double>(p, m);
    out_w[e] = std::isfinite(w) ? w : 0.0;
  }
  return 0;
}

double orc_pdf_grid(const orc_params* p, int species, double x, double Q) { return pdf_grid<double>(p, species, x, Q); }

// NEXT-4 building blocks (pinned by tests/test_oracle_tth.py)
int orc_eq9_roots(double K12, double f, double sH, double E1[2], double E2[2], double* jac) {
  return eq9_roots<double>(K12, f, sH, E1, E2, jac);
}
double orc_tth_radiator(const orc_params* p, const double pt[4], const double ptb[4], const double k[4]) {
  return tth_radiator<double>(p, from_arr(pt), from_arr(ptb), from_arr(k));
}
double orc_tth_decay(const orc_params* p, double sH) { return tth_decay<double>(p, sH); }
int orc_tth_tt_invariants(const orc_params* p, const double q1[4], const double q2[4], const double pt[4],
                          const double ptb[4], double* t1, double* t2, double* rho) {
  return tth_tt_invariants<double>(p, q1, q2, from_arr(pt), from_arr(ptb), t1, t2, rho) ? 1 : 0;
}
double orc_me_tt_gg_inv(const orc_params* p, double t1, double t2, double rho) { return me_tt_gg_inv<double>(p, t1, t2, rho); }
double orc_me_tt_qq_inv(const orc_params* p, double t1, double t2, double rho) { return me_tt_qq_inv<double>(p, t1, t2, rho); }
double orc_tt_flavour_sum(const orc_params* p, double x1, double x2, double me_gg, double me_qq) {
  return tt_flavour_sum<double>(p, x1, x2, me_gg, me_qq);
}
// sum over all spins of |M(t -> b f fbar')|^2 with the W propagator passed in (mapped resonance, O6)
double orc_me_top_decay_D(const orc_params* p, double n_c, const double pt[4], const double pb[4],
                          const double pf_down[4], const double pf_up[4], double D_W) {
  return me_top_decay_D<double>(p, n_c, pt, pb, pf_down, pf_up, D_W);
}

// post-processing of PAPER.md:45 (1/sigma) and :143 Eq. 10 (reading A22): sigma as the importance-sampled
// acceptance integral (1/n) sum_e p_e / g_e over events drawn from the density g; D = log10 of the ratio of
// the two normalised likelihoods.
double orc_normalisation(const double* p, const double* g, int64_t n) {
  NSum s;
  for (int64_t e = 0; e < n; ++e) s.add(p[e] / g[e]);
  return s.value() / (double)n;
}
void orc_discriminant(const double* p_sig, const double* p_bkg, int64_t n, double sigma_sig, double sigma_bkg,
                      double* out_D) {
  for (int64_t e = 0; e < n; ++e) out_D[e] = std::log10((p_sig[e] / sigma_sig) / (p_bkg[e] / sigma_bkg));
}

double orc_weight(int process, const orc_params* p, const double* rec, const double* u, double* dbg) {
  return weight_any<double>(process, p, rec, u, dbg);
}
// extended-precision referee: the same algorithm in long double, rounded to double at the end
double orc_weight_x(int process, const orc_params* p, const double* rec, const double* u) {
  return weight_any<long double>(process, p, rec, u, nullptr);
}

// --------------------------------------------------------------------------
// VEGAS (config 5; SURVEY.md 8(c) "Config 5", reading A14)
// --------------------------------------------------------------------------
void orc_vegas_map(const double* edges, int bins, int n_dims, const double* u, double* z, int* k, double* jac) {
  vegas_map<double>(edges, bins, n_dims, u, z, k, jac);
}

void orc_vegas_refine(const double* hist, double* edges, int bins, double alpha) {
  const int B = bins;
  std::vector<double> h(B), r(B);
  // smooth (1,6,1)/8 with (7,1)/8 at the ends
  if (B == 1) h[0] = hist[0];
  else {
    h[0] = (7.0 * hist[0] + hist[1]) / 8.0;
    for (int k = 1; k < B - 1; ++k) h[k] = (hist[k - 1] + 6.0 * hist[k] + hist[k + 1]) / 8.0;
    h[B - 1] = (hist[B - 2] + 7.0 * hist[B - 1]) / 8.0;
  }
  double tot = 0.0;
  for (int k = 0; k < B; ++k) tot += h[k];
  if (!(tot > 0.0) || !std::isfinite(tot)) return;      // leave the grid
  // compress
  double rsum = 0.0;
  for (int k = 0; k < B; ++k) {
    double rk = h[k] / tot;
    if (rk <= 0.0) r[k] = 0.0;
    else if (rk >= 1.0) r[k] = 1.0;
    else r[k] = std::pow((1.0 - rk) / std::log(1.0 / rk), alpha);
    rsum += r[k];
  }
  // new edges = j/B quantiles of the piecewise-constant density r on the old bins
  std::vector<double> nx(B + 1);
  nx[0] = edges[0]; nx[B] = edges[B];
  double per = rsum / B, acc = 0.0;
  int k = 0;
  for (int j = 1; j < B; ++j) {
    double target = j * per;
    while (k < B - 1 && acc + r[k] < target) { acc += r[k]; ++k; }
    double frac = (r[k] > 0.0) ? (target - acc) / r[k] : 0.0;
    if (frac < 0.0) frac = 0.0;
    if (frac > 1.0) frac = 1.0;
    nx[j] = edges[k] + frac * (edges[k + 1] - edges[k]);
  }
  for (int j = 0; j <= B; ++j) edges[j] = nx[j];
}

// --------------------------------------------------------------------------
// drivers
// --------------------------------------------------------------------------
int orc_eval_points(int process, const orc_params* p, const double* events, int64_t n_events,
                    int64_t event, uint64_t event_offset, int64_t first_point, int64_t n,
                    uint64_t seed, int32_t iteration, const double* grid, double* out_w) {
  int nf = orc_n_fields(process), D = orc_n_dims(process);
  if (nf < 0 || !p || !events || !out_w || event < 0 || event >= n_events) return 1;
  double rec[32], u[16], z[16];
  load_record(events, n_events, event, nf, rec);
  const int B = p->vegas_bins;
  for (int64_t i = 0; i < n; ++i) {
    orc_uniforms(seed, event_offset + (uint64_t)event, (uint64_t)(first_point + i), (uint32_t)iteration, D, u);
    if (grid) {
      double jac;
      orc_vegas_map(grid + (size_t)event * D * (B + 1), B, D, u, z, nullptr, &jac);
      out_w[i] = jac * orc_weight(process, p, rec, z, nullptr);
    } else {
      out_w[i] = orc_weight(process, p, rec, u, nullptr);
    }
  }
  return 0;
}

// referee version of orc_eval_points.  With a grid the warp u -> z and its Jacobian are the fp64 ones of
// orc_vegas_map (the warped point is itself a rounded fp64 quantity on both sides); the integrand at z is
// evaluated in long double.
int orc_eval_points_x(int process, const orc_params* p, const double* events, int64_t n_events,
                      int64_t event, uint64_t event_offset, int64_t first_point, int64_t n,
                      uint64_t seed, int32_t iteration, const double* grid, double* out_w) {
  int nf = orc_n_fields(process), D = orc_n_dims(process);
  if (nf < 0 || !p || !events || !out_w || event < 0 || event >= n_events) return 1;
  double rec[32], u[16], z[16];
  load_record(events, n_events, event, nf, rec);
  const int B = p->vegas_bins;
  for (int64_t i = 0; i < n; ++i) {
    orc_uniforms(seed, event_offset + (uint64_t)event, (uint64_t)(first_point + i), (uint32_t)iteration, D, u);
    if (grid) {
      double jac;
      orc_vegas_map(grid + (size_t)event * D * (B + 1), B, D, u, z, nullptr, &jac);
      out_w[i] = (double)((long double)jac * (long double)orc_weight_x(process, p, rec, z));
    } else {
      out_w[i] = orc_weight_x(process, p, rec, u);
    }
  }
  return 0;
}

// O1 (PAPER.md:76 Eq. 5, :80 Eq. 6, reading A1)
static void estimate(const NSum& s1, const NSum& s2, int64_t N, double* mean, double* err) {
  double m = s1.value() / (double)N;
  double var = s2.value() / (double)N - m * m;
  if (var < 0.0) var = 0.0;
  *mean = m;
  *err = std::sqrt(var / (double)(N - 1));
}

int orc_integrate(int process, const orc_params* p, const double* events, int64_t n_events,
                  uint64_t event_offset, int64_t n_points, uint64_t seed, double* out_p, double* out_err) {
  int nf = orc_n_fields(process), D = orc_n_dims(process);
  if (nf < 0 || !p || n_points < 2) return 1;
  double rec[32], u[16];
  for (int64_t e = 0; e < n_events; ++e) {
    load_record(events, n_events, e, nf, rec);
    NSum s1, s2;
    for (int64_t i = 0; i < n_points; ++i) {
      orc_uniforms(seed, event_offset + (uint64_t)e, (uint64_t)i, 0u, D, u);
      double w = orc_weight(process, p, rec, u, nullptr);
      s1.add(w); s2.add(w * w);
    }
    estimate(s1, s2, n_points, &out_p[e], &out_err[e]);
  }
  return 0;
}

int orc_vegas_integrate(int process, const orc_params* p, const double* events, int64_t n_events,
                        uint64_t event_offset, int64_t n_points, uint64_t seed,
                        double* out_p, double* out_err, double* grid_out) {
  int nf = orc_n_fields(process), D = orc_n_dims(process);
  const int B = p->vegas_bins;
  if (nf < 0 || !p || n_points < 2 || B < 1) return 1;
  double rec[32], u[16], z[16];
  int k[16];
  std::vector<double> edges((size_t)D * (B + 1)), hist((size_t)D * B);
  for (int64_t e = 0; e < n_events; ++e) {
    load_record(events, n_events, e, nf, rec);
    for (int d = 0; d < D; ++d)
      for (int j = 0; j <= B; ++j) edges[(size_t)d * (B + 1) + j] = (double)j / (double)B;
    for (int it = 0; it < p->vegas_iters; ++it) {
      std::fill(hist.begin(), hist.end(), 0.0);
      for (int64_t i = 0; i < p->vegas_points; ++i) {
        orc_uniforms(seed, event_offset + (uint64_t)e, (uint64_t)i, (uint32_t)it, D, u);
        double jac;
        orc_vegas_map(edges.data(), B, D, u, z, k, &jac);
        double w = jac * orc_weight(process, p, rec, z, nullptr);
        for (int d = 0; d < D; ++d) hist[(size_t)d * B + k[d]] += w * w;
      }
      for (int d = 0; d < D; ++d)
        orc_vegas_refine(hist.data() + (size_t)d * B, edges.data() + (size_t)d * (B + 1), B, p->vegas_alpha);
    }
    NSum s1, s2;
    for (int64_t i = 0; i < n_points; ++i) {
      orc_uniforms(seed, event_offset + (uint64_t)e, (uint64_t)i, (uint32_t)p->vegas_iters, D, u);
      double jac;
      orc_vegas_map(edges.data(), B, D, u, z, nullptr, &jac);
      double w = jac * orc_weight(process, p, rec, z, nullptr);
      s1.add(w); s2.add(w * w);
    }
    estimate(s1, s2, n_points, &out_p[e], &out_err[e]);
    if (grid_out) std::memcpy(grid_out + (size_t)e * D * (B + 1), edges.data(), edges.size() * sizeof(double));
  }
  return 0;
}

}  // extern "C"
