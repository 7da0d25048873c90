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
template <typename R> R me_tt_qq(const orc_params* p, const R q1[4], const R q2[4], const R pt[4], const R ptb[4]) {
  R t1, t2, rho;
  tt_invariants<R>(p, q1, q2, pt, ptb, &t1, &t2, &rho);
  R g = gs2<R>(p);
  return g * g * (R(4) / R(9)) * (t1 * t1 + t2 * t2 + rho / R(2));
}
template <typename R> R me_tt_gg(const orc_params* p, const R q1[4], const R q2[4], const R pt[4], const R ptb[4]) {
  R t1, t2, rho;
  tt_invariants<R>(p, q1, q2, pt, ptb, &t1, &t2, &rho);
  R g = gs2<R>(p);
  return g * g * (R(1) / (R(6) * t1 * t2) - R(3) / R(8)) *
         (t1 * t1 + t2 * t2 + rho - rho * rho / (R(4) * t1 * t2));
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
  R prod = R(p->pdf_A_g) * R(p->pdf_A_g) * me_tt_gg<R>(p, q1, q2, pta, ptba) +
           R(2) * R(p->n_flav) * R(p->pdf_A_q) * R(p->pdf_A_q) * me_tt_qq<R>(p, q1, q2, pta, ptba);
  // narrow-width factorised decays, 1/2 = average over the decaying top's spin.  The leptonic
  // W mass is the mapped variable: its propagator is D(m Gam tan t) (reading O6).
  R dec_lep = R(0.5) * me_top_decay_D<R>(p, R(1), pta, mom + 8, mom, mom + 4, DW_lep);
  R dec_had = R(0.5) * R(p->V_ud) * R(p->V_ud) * me_top_decay<R>(p, R(3), ptba, mom + 12, mom + 16, mom + 20);
  R mt = p->m_t, Gt = p->Gam_t;
  R Dt = bw_D<R>(st - mt * mt, mt, Gt), Dtb = bw_D<R>(stb - mt * mt, mt, Gt);
  R me = prod * Dt * Dtb * dec_lep * dec_had;
  R ff = pdf_shape<R>(p, x1) * pdf_shape<R>(p, x2);
  R flux = x1 * x2 * S / R(4);
  dbg_store<R>(dbg, 0, 6, x1, x2, mom);
  if (dbg) dbg[0] = 1;
  R w = vol * dsdt * tf * meas * (R(16) * pi_<R>() * pi_<R>() * pi_<R>() * pi_<R>()) * (R(2) / S) * ff * me / flux;
  return std::isfinite(w) ? w : R(0);
}

template <typename R> double weight_any(int process, const orc_params* p, const double* rec, const double* u,
                                        double* dbg) {
  R w = R(0);
  switch (process) {
    case ORC_W_ENU: w = weight_w_enu<R>(p, rec, u, dbg); break;
    case ORC_Z_BB: w = weight_z_bb<R>(p, rec, u, dbg); break;
    case ORC_TT_LJETS: w = weight_tt_ljets<R>(p, rec, u, dbg); break;
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
                     case ORC_TT_LJETS: return 17; case ORC_TT_DILEP: return 14; }
  return -1;
}
int orc_n_dims(int process) {
  switch (process) { case ORC_W_ENU: return 1; case ORC_Z_BB: return 2;
                     case ORC_TT_LJETS: return 6; case ORC_TT_DILEP: return 8; }
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

// referee version of orc_eval_points (no grid: the warped point z is itself a rounded fp64
// quantity on both sides, so grid parity is tested through orc_eval_points)
int orc_eval_points_x(int process, const orc_params* p, const double* events, int64_t n_events,
                      int64_t event, uint64_t event_offset, int64_t first_point, int64_t n,
                      uint64_t seed, int32_t iteration, double* out_w) {
  int nf = orc_n_fields(process), D = orc_n_dims(process);
  if (nf < 0 || !p || !events || !out_w || event < 0 || event >= n_events) return 1;
  double rec[32], u[16];
  load_record(events, n_events, event, nf, rec);
  for (int64_t i = 0; i < n; ++i) {
    orc_uniforms(seed, event_offset + (uint64_t)event, (uint64_t)(first_point + i), (uint32_t)iteration, D, u);
    out_w[i] = orc_weight_x(process, p, rec, u);
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
