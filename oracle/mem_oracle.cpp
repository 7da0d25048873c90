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

const double kPi = 3.14159265358979323846264338327950288;

struct V4 {
  double E, x, y, z;
};
inline V4 operator+(const V4& a, const V4& b) { return {a.E + b.E, a.x + b.x, a.y + b.y, a.z + b.z}; }
inline double dot(const V4& a, const V4& b) { return a.E * b.E - a.x * b.x - a.y * b.y - a.z * b.z; }
inline V4 from_arr(const double* a) { return {a[0], a[1], a[2], a[3]}; }

// massless particle from (pT, eta, phi)
inline V4 from_pt_eta_phi(double pT, double eta, double phi) {
  return {pT * std::cosh(eta), pT * std::cos(phi), pT * std::sin(phi), pT * std::sinh(eta)};
}
// massless particle from (E, eta, phi): direction n = (cos phi/cosh eta, sin phi/cosh eta, tanh eta)
inline V4 from_E_eta_phi(double E, double eta, double phi) {
  double st = 1.0 / std::cosh(eta);  // sin(theta)
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
inline double g2_weak(const orc_params* p) { return 4.0 * std::sqrt(2.0) * p->G_F * p->m_W * p->m_W; }
inline double gZ2(const orc_params* p) { return 4.0 * std::sqrt(2.0) * p->G_F * p->m_Z * p->m_Z; }
inline double gs2(const orc_params* p) { return 4.0 * kPi * p->alpha_s; }
inline void z_couplings(const orc_params* p, bool up, double* L, double* R) {
  double T3 = up ? 0.5 : -0.5, Q = up ? 2.0 / 3.0 : -1.0 / 3.0;
  *L = T3 - Q * p->sin2_thw;
  *R = -Q * p->sin2_thw;
}
inline double bw_D(double s_minus_m2, double m, double Gam) {
  return 1.0 / (s_minus_m2 * s_minus_m2 + m * m * Gam * Gam);
}
// flavours in the paper's order (d,u,s,c,b); first n_flav are summed.
inline bool flavour_is_up(int i) { return i == 1 || i == 3; }

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
// O4. toy PDF shape, O5. jet TF, O6. Breit-Wigner map
// --------------------------------------------------------------------------
double orc_pdf_shape(const orc_params* p, double x) {
  return std::pow(x, p->pdf_pow_x) * std::pow(1.0 - x, p->pdf_pow_1mx);
}

static double gauss(double d, double mu, double sig) {
  double z = (d - mu) / sig;
  return std::exp(-0.5 * z * z) / (sig * std::sqrt(2.0 * kPi));
}
// PAPER.md:58 "double Gaussian"; BASELINE.json:configs[1] parameters; reading A11.
double orc_tf_jet(const orc_params* p, double E_jet, double E) {
  double d = E_jet - E;
  return (1.0 - p->tf_w_tail) * gauss(d, p->tf_mu1 * E, p->tf_sig1 * E) +
         p->tf_w_tail * gauss(d, p->tf_mu2 * E, p->tf_sig2 * E);
}

// integrate over q^2 of the propagators.  s = m^2 + m Gam tan t.
void orc_bw_window(double m, double Gam, double s_lo, double s_hi, double* t_lo, double* t_hi) {
  *t_lo = std::atan((s_lo - m * m) / (m * Gam));
  *t_hi = std::atan((s_hi - m * m) / (m * Gam));
}
void orc_bw_point(double m, double Gam, double t, double* s_minus_m2, double* dsdt, double* D) {
  double smm = m * Gam * std::tan(t);
  *s_minus_m2 = smm;
  *dsdt = (smm * smm + m * m * Gam * Gam) / (m * Gam);
  *D = bw_D(smm, m, Gam);
}

// --------------------------------------------------------------------------
// matrix elements (SURVEY.md 8(c) "Matrix elements")
// --------------------------------------------------------------------------
// u(qa) dbar(qb) -> W+ -> e+(lep) nu:  g^4 |V_ud|^2 / 12 * u^2 * D_W(s),  u = -2 qa.lep
double orc_me_w(const orc_params* p, const double qa[4], const double qb[4],
                const double lep[4], const double nu[4]) {
  V4 a = from_arr(qa), b = from_arr(qb), l = from_arr(lep);
  (void)nu;
  double shat = dot(a + b, a + b);
  double uhat = -2.0 * dot(a, l);
  double g2 = g2_weak(p);
  return g2 * g2 * p->V_ud * p->V_ud / 12.0 * uhat * uhat * bw_D(shat - p->m_W * p->m_W, p->m_W, p->Gam_W);
}

// q(qa) qbar(qb) -> Z -> b(p1) bbar(p2), Z exchange only, colour factor 1
double orc_me_z(const orc_params* p, int up_type, const double qa[4], const double qb[4],
                const double p1[4], const double p2[4]) {
  V4 a = from_arr(qa), b = from_arr(qb), b1 = from_arr(p1), b2 = from_arr(p2);
  double Lq, Rq, Lb, Rb;
  z_couplings(p, up_type != 0, &Lq, &Rq);
  z_couplings(p, false, &Lb, &Rb);
  double shat = dot(a + b, a + b);
  double uhat = -2.0 * dot(a, b2), that = -2.0 * dot(a, b1);
  double gz = gZ2(p);
  return gz * gz * ((Lq * Lq * Lb * Lb + Rq * Rq * Rb * Rb) * uhat * uhat +
                    (Lq * Lq * Rb * Rb + Rq * Rq * Lb * Lb) * that * that) *
         bw_D(shat - p->m_Z * p->m_Z, p->m_Z, p->Gam_Z);
}

// reading A9: tau1 + tau2 = 1 also off shell, pole mass in rho
static void tt_invariants(const orc_params* p, const double q1[4], const double q2[4],
                          const double pt[4], const double ptb[4], double* t1, double* t2, double* rho) {
  V4 a = from_arr(q1), b = from_arr(q2), t = from_arr(pt), tb = from_arr(ptb);
  double shat = dot(a + b, a + b);
  *t1 = (dot(a, t) + dot(b, tb)) / shat;
  *t2 = (dot(b, t) + dot(a, tb)) / shat;
  *rho = 4.0 * p->m_t * p->m_t / shat;
}
double orc_me_tt_qq(const orc_params* p, const double q1[4], const double q2[4],
                    const double pt[4], const double ptb[4]) {
  double t1, t2, rho;
  tt_invariants(p, q1, q2, pt, ptb, &t1, &t2, &rho);
  double g = gs2(p);
  return g * g * (4.0 / 9.0) * (t1 * t1 + t2 * t2 + rho / 2.0);
}
double orc_me_tt_gg(const orc_params* p, const double q1[4], const double q2[4],
                    const double pt[4], const double ptb[4]) {
  double t1, t2, rho;
  tt_invariants(p, q1, q2, pt, ptb, &t1, &t2, &rho);
  double g = gs2(p);
  return g * g * (1.0 / (6.0 * t1 * t2) - 3.0 / 8.0) *
         (t1 * t1 + t2 * t2 + rho - rho * rho / (4.0 * t1 * t2));
}

// sum over all spins of |M(t -> b W -> b fdown-bar... )|^2 with the pairing
// (p_t . p_fdown)(p_b . p_fup): for t -> b l+ nu, fdown = l+ and fup = nu.
double orc_me_top_decay(const orc_params* p, double n_c, const double pt[4], const double pb[4],
                        const double pf_down[4], const double pf_up[4]) {
  V4 t = from_arr(pt), b = from_arr(pb), fd = from_arr(pf_down), fu = from_arr(pf_up);
  double sW = dot(fd + fu, fd + fu);
  double g2 = g2_weak(p);
  return n_c * 4.0 * g2 * g2 * p->V_tb * p->V_tb * dot(t, fd) * dot(b, fu) *
         bw_D(sW - p->m_W * p->m_W, p->m_W, p->Gam_W);
}

// O7. pure transverse boost that removes the transverse momentum of P.
void orc_boost_transverse(const double P[4], int n, double* mom) {
  double bx = P[1] / P[0], by = P[2] / P[0];
  double b2 = bx * bx + by * by;
  double gam = 1.0 / std::sqrt(1.0 - b2);
  double k2 = gam * gam / (gam + 1.0);  // = (gamma-1)/beta^2, finite at beta = 0
  for (int i = 0; i < n; ++i) {
    double* q = mom + 4 * i;
    double bp = bx * q[1] + by * q[2];
    double En = gam * (q[0] - bp);
    double k = k2 * bp - gam * q[0];
    q[1] += k * bx; q[2] += k * by; q[0] = En;
  }
}

}  // extern "C"

// --------------------------------------------------------------------------
// per-configuration weights
// --------------------------------------------------------------------------
namespace {

// O3: x1, x2 from the (boosted) total momentum.  Returns false when outside (0,1).
bool beam_fractions(const orc_params* p, double PE, double Pz, double* x1, double* x2) {
  *x1 = (PE + Pz) / p->sqrt_s;
  *x2 = (PE - Pz) / p->sqrt_s;
  return (*x1 > 0.0 && *x1 < 1.0 && *x2 > 0.0 && *x2 < 1.0);
}
void beams(const orc_params* p, double x1, double x2, double q1[4], double q2[4]) {
  double h = 0.5 * p->sqrt_s;
  q1[0] = x1 * h; q1[1] = 0; q1[2] = 0; q1[3] = x1 * h;
  q2[0] = x2 * h; q2[1] = 0; q2[2] = 0; q2[3] = -x2 * h;
}
void to_arr(const V4& v, double* a) { a[0] = v.E; a[1] = v.x; a[2] = v.y; a[3] = v.z; }

void dbg_store(double* dbg, int sol, int n_final, double x1, double x2, const double* mom) {
  if (!dbg) return;
  double* d = dbg + 1 + sol * (2 + 4 * n_final);
  d[0] = x1; d[1] = x2;
  for (int i = 0; i < 4 * n_final; ++i) d[2 + i] = mom[i];
}

// ---------------- config 1: u dbar -> W+ -> e+ nu, D = 1 ----------------
// rec = [lep_pT, lep_eta, lep_phi, met_x, met_y]   (SURVEY.md 8(c) "Config 1", reading A5)
double weight_w_enu(const orc_params* p, const double* rec, const double* u, double* dbg) {
  const double pT = rec[0], eta = rec[1], phi = rec[2], mx = rec[3], my = rec[4];
  const double Pz = p->nu_pz_max, m = p->m_W, G = p->Gam_W, S = p->sqrt_s * p->sqrt_s;
  V4 l = from_pt_eta_phi(pT, eta, phi);
  double nT = std::sqrt(mx * mx + my * my);
  double a = l.x * mx + l.y * my;                      // l_T . nu_T
  auto s_of = [&](double nz) { return 2.0 * (l.E * std::sqrt(nT * nT + nz * nz) - a - l.z * nz); };
  // 1. window in s_W.  Stationary point of s(nu_z): nu_z* = |nu_T| sinh(eta_l), s* = 2(pT nT - a).
  double nz_star = nT * std::sinh(eta);
  double s_star = 2.0 * (pT * nT - a);
  double s_min = (nz_star > Pz) ? s_of(Pz) : (nz_star < -Pz) ? s_of(-Pz) : s_star;
  double s_max = std::fmax(s_of(-Pz), s_of(Pz));
  double t_lo, t_hi;
  orc_bw_window(m, G, s_min, s_max, &t_lo, &t_hi);
  double dt = t_hi - t_lo;
  double t = t_lo + dt * u[0];
  double smm, dsdt, DW;
  orc_bw_point(m, G, t, &smm, &dsdt, &DW);
  double sW = m * m + smm;
  // 2. roots of s(nu_z) = sW.  disc = c^2 - pT^2 nT^2 = (c - pT nT)(c + pT nT) with
  //    c - pT nT = (sW - s*)/2; sW - s_min = m G (tan t - tan t_lo) = m G sin(dt u)/(cos t cos t_lo)
  //    (cancellation-free near the transverse-mass edge; reading A5b).
  double ds = m * G * std::sin(dt * u[0]) / (std::cos(t) * std::cos(t_lo));
  double half = 0.5 * (ds + (s_min - s_star));
  double c = 0.5 * sW + a;
  double disc = half * (c + pT * nT);
  if (dbg) dbg[0] = 0;
  if (!(disc > 0.0)) return 0.0;
  double rt = std::sqrt(disc);
  double sum = 0.0;
  int n_sol = 0;
  for (int sgn = -1; sgn <= 1; sgn += 2) {
    double nz = (c * l.z + sgn * l.E * rt) / (pT * pT);
    if (!(std::fabs(nz) <= Pz)) continue;
    double En = std::sqrt(nT * nT + nz * nz);
    // |d nu_z / d s| = E_nu / (2 sqrt(disc))   (= 1/|2(E_l nu_z/E_nu - l_z)| at the root)
    double jac = En / (2.0 * rt);
    V4 nu = {En, mx, my, nz};
    V4 P = l + nu;
    double x1, x2;
    if (!beam_fractions(p, P.E, P.z, &x1, &x2)) continue;
    double q1[4], q2[4], la[4], na[4];
    beams(p, x1, x2, q1, q2); to_arr(l, la); to_arr(nu, na);
    // flavour sum = both beam orderings (u from beam 1 or from beam 2), reading A4
    double me = orc_me_w(p, q1, q2, la, na) + orc_me_w(p, q2, q1, la, na);
    double ff = p->pdf_A_q * p->pdf_A_q * orc_pdf_shape(p, x1) * orc_pdf_shape(p, x2);
    double flux = x1 * x2 * S / 4.0;                   // |q1||q2|, Eq. 1
    double w_root = ff * me / flux / (8.0 * kPi * kPi * S * l.E * En);
    sum += jac * w_root;
    if (dbg) { double mom[8]; to_arr(l, mom); to_arr(nu, mom + 4); dbg_store(dbg, n_sol, 2, x1, x2, mom); }
    ++n_sol;
  }
  if (dbg) dbg[0] = n_sol;
  return dt * dsdt * sum;
}

// ---------------- config 2: q qbar -> Z -> b bbar, D = 2 ----------------
// rec = [E1, eta1, phi1, E2, eta2, phi2]   (SURVEY.md 8(c) "Config 2")
double weight_z_bb(const orc_params* p, const double* rec, const double* u, double* dbg) {
  const double S = p->sqrt_s * p->sqrt_s, dr = p->jetE_rhi - p->jetE_rlo;
  const double twopi3 = 8.0 * kPi * kPi * kPi;
  if (dbg) dbg[0] = 0;
  double Ej[2] = {rec[0], rec[3]}, eta[2] = {rec[1], rec[4]}, phi[2] = {rec[2], rec[5]};
  double E[2], mom[8], vol = 1.0, tf = 1.0, meas = 1.0;
  V4 P = {0, 0, 0, 0};
  for (int j = 0; j < 2; ++j) {
    E[j] = Ej[j] * (p->jetE_rlo + dr * u[j]);
    vol *= Ej[j] * dr;
    tf *= orc_tf_jet(p, Ej[j], E[j]);
    meas *= E[j] * (1.0 / std::cosh(eta[j])) / (2.0 * twopi3);   // E sin(theta) dE / (2 (2pi)^3)
    V4 q = from_E_eta_phi(E[j], eta[j], phi[j]);
    to_arr(q, mom + 4 * j);
    P = P + q;
  }
  double Parr[4]; to_arr(P, Parr);
  orc_boost_transverse(Parr, 2, mom);                  // O7
  double PE = mom[0] + mom[4], Pzz = mom[3] + mom[7];
  double x1, x2;
  if (!beam_fractions(p, PE, Pzz, &x1, &x2)) return 0.0;
  double q1[4], q2[4];
  beams(p, x1, x2, q1, q2);
  double me = 0.0;
  for (int f = 0; f < p->n_flav; ++f)                  // q from beam 1 or beam 2
    me += orc_me_z(p, flavour_is_up(f), q1, q2, mom, mom + 4) + orc_me_z(p, flavour_is_up(f), q2, q1, mom, mom + 4);
  double ff = p->pdf_A_q * p->pdf_A_q * orc_pdf_shape(p, x1) * orc_pdf_shape(p, x2);
  double flux = x1 * x2 * S / 4.0;
  dbg_store(dbg, 0, 2, x1, x2, mom);
  if (dbg) dbg[0] = 1;
  return vol * tf * meas * (16.0 * kPi * kPi * kPi * kPi) * (2.0 / S) * ff * me / flux;
}

// ---------------- config 3: t tbar -> b l nu  bbar q qbar', D = 6 ----------------
// rec = [lep_pT, lep_eta, lep_phi, (E,eta,phi) x {b_had, b_lep, q, qbar'}, met, met_phi]
// (SURVEY.md 8(c) "Config 3", reading A7)
double weight_tt_ljets(const orc_params* p, const double* rec, const double* u, double* dbg) {
  const double S = p->sqrt_s * p->sqrt_s, dr = p->jetE_rhi - p->jetE_rlo, H = p->nu_eta_max;
  const double twopi3 = 8.0 * kPi * kPi * kPi;
  if (dbg) dbg[0] = 0;
  const double lpT = rec[0], leta = rec[1], lphi = rec[2], met_phi = rec[16];
  V4 l = from_pt_eta_phi(lpT, leta, lphi);
  V4 jet[4];
  double vol = 1.0, tf = 1.0, meas = 1.0;
  for (int j = 0; j < 4; ++j) {
    double Ej = rec[3 + 3 * j], eta = rec[4 + 3 * j], phi = rec[5 + 3 * j];
    double E = Ej * (p->jetE_rlo + dr * u[j]);
    vol *= Ej * dr;
    tf *= orc_tf_jet(p, Ej, E);
    meas *= E * (1.0 / std::cosh(eta)) / (2.0 * twopi3);
    jet[j] = from_E_eta_phi(E, eta, phi);
  }
  const V4 &b_had = jet[0], &b_lep = jet[1], &q = jet[2], &qb = jet[3];
  // neutrino: eta flat in [-H, H]; leptonic W mass BW-mapped; azimuth = MET azimuth
  double eta_nu = -H + 2.0 * H * u[4];
  vol *= 2.0 * H;
  double mW = p->m_W, GW = p->Gam_W, n = p->bw_nwidths;
  double t_lo, t_hi;
  orc_bw_window(mW, GW, (mW - n * GW) * (mW - n * GW), (mW + n * GW) * (mW + n * GW), &t_lo, &t_hi);
  double t = t_lo + (t_hi - t_lo) * u[5];
  vol *= (t_hi - t_lo);
  double smm, dsdt, DW_lep;
  orc_bw_point(mW, GW, t, &smm, &dsdt, &DW_lep);
  double sW = mW * mW + smm;
  double den = 2.0 * lpT * (std::cosh(leta - eta_nu) - std::cos(lphi - met_phi));
  if (!(den > 0.0)) return 0.0;
  double nuT = sW / den;
  V4 nu = from_pt_eta_phi(nuT, eta_nu, met_phi);
  meas *= 1.0 / (2.0 * l.E * twopi3);                  // lepton: delta TF
  meas *= nuT * nuT / (2.0 * sW * twopi3);             // d^3nu/((2pi)^3 2E) -> ds_W d eta_nu
  V4 pt = b_lep + l + nu, ptb = b_had + q + qb;
  double st = dot(pt, pt), stb = dot(ptb, ptb);
  // O7 boost of the six final-state momenta: order l, nu, b_lep, b_had, q, qbar'
  double mom[24];
  to_arr(l, mom); to_arr(nu, mom + 4); to_arr(b_lep, mom + 8); to_arr(b_had, mom + 12);
  to_arr(q, mom + 16); to_arr(qb, mom + 20);
  V4 P = pt + ptb;
  double Parr[4]; to_arr(P, Parr);
  if (!(P.x * P.x + P.y * P.y < P.E * P.E)) return 0.0;
  orc_boost_transverse(Parr, 6, mom);
  double PE = 0, Pzz = 0;
  for (int i = 0; i < 6; ++i) { PE += mom[4 * i]; Pzz += mom[4 * i + 3]; }
  double x1, x2;
  if (!beam_fractions(p, PE, Pzz, &x1, &x2)) return 0.0;
  double shat = x1 * x2 * S;
  if (!(4.0 * p->m_t * p->m_t < shat)) return 0.0;     // rho >= 1 -> 0 (A9)
  double q1[4], q2[4], pta[4], ptba[4];
  beams(p, x1, x2, q1, q2);
  for (int k = 0; k < 4; ++k) { pta[k] = mom[k] + mom[4 + k] + mom[8 + k]; ptba[k] = mom[12 + k] + mom[16 + k] + mom[20 + k]; }
  double prod = p->pdf_A_g * p->pdf_A_g * orc_me_tt_gg(p, q1, q2, pta, ptba) +
                2.0 * p->n_flav * p->pdf_A_q * p->pdf_A_q * orc_me_tt_qq(p, q1, q2, pta, ptba);
  // narrow-width factorised decays, 1/2 = average over the decaying top's spin
  double dec_lep = 0.5 * orc_me_top_decay(p, 1.0, pta, mom + 8, mom, mom + 4);
  double dec_had = 0.5 * p->V_ud * p->V_ud * orc_me_top_decay(p, 3.0, ptba, mom + 12, mom + 16, mom + 20);
  double Dt = bw_D(st - p->m_t * p->m_t, p->m_t, p->Gam_t), Dtb = bw_D(stb - p->m_t * p->m_t, p->m_t, p->Gam_t);
  double me = prod * Dt * Dtb * dec_lep * dec_had;
  double ff = orc_pdf_shape(p, x1) * orc_pdf_shape(p, x2);
  double flux = x1 * x2 * S / 4.0;
  dbg_store(dbg, 0, 6, x1, x2, mom);
  if (dbg) dbg[0] = 1;
  double w = vol * dsdt * tf * meas * (16.0 * kPi * kPi * kPi * kPi) * (2.0 / S) * ff * me / flux;
  return std::isfinite(w) ? w : 0.0;
}

}  // namespace

extern "C" {

double orc_weight(int process, const orc_params* p, const double* rec, const double* u, double* dbg) {
  double w = 0.0;
  switch (process) {
    case ORC_W_ENU: w = weight_w_enu(p, rec, u, dbg); break;
    case ORC_Z_BB: w = weight_z_bb(p, rec, u, dbg); break;
    case ORC_TT_LJETS: w = weight_tt_ljets(p, rec, u, dbg); break;
    default: return std::nan("");
  }
  return std::isfinite(w) ? w : 0.0;   // non-finite points contribute 0
}

// --------------------------------------------------------------------------
// VEGAS (config 5; SURVEY.md 8(c) "Config 5", reading A14)
// --------------------------------------------------------------------------
void orc_vegas_map(const double* edges, int bins, int n_dims, const double* u, double* z, int* k, double* jac) {
  double j = 1.0;
  for (int d = 0; d < n_dims; ++d) {
    const double* x = edges + (size_t)d * (bins + 1);
    double y = u[d] * bins;
    int kk = (int)std::floor(y);
    if (kk > bins - 1) kk = bins - 1;
    double width = x[kk + 1] - x[kk];
    z[d] = x[kk] + (y - kk) * width;
    j *= bins * width;
    if (k) k[d] = kk;
  }
  *jac = j;
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
static void load_record(const double* events, int64_t n_events, int64_t e, int nf, double* rec) {
  for (int f = 0; f < nf; ++f) rec[f] = events[(size_t)f * n_events + e];
}

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
