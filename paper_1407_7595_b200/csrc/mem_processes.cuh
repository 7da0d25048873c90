// mem_processes.cuh -- S0, S2-S7 of the hot path for each process hypothesis.
//
// Each process is a struct with
//   D, NF, NC               integration dimensions, record fields, per-event constants
//   prepare(c, ev, n, e, ec) S0: read event e of the SoA record array, write the per-event
//                            constants ec[NC] (everything that does not depend on the point)
//   weight(c, ec, u)         S2-S7: the integrand w at the unit-cube point u[D]
// The formulas restate DESIGN.md "Readings" O3-O8 (PAPER.md:45-58 Eq. 1-3, :103-111 Eq. 7)
// with every point-independent factor folded into one per-event constant C0 and with
// Lorentz-invariant products written through per-event angular constants
//   a.b = E_a E_b K_ab,  K_ab = 1 - n_a.n_b = 2 (sinh^2(d eta/2) + sin^2(d phi/2)) / (cosh eta_a cosh eta_b)
// (massless partons), so that no point needs six boosted four-vectors in
// registers (the paper's own register-pressure finding).
#pragma once
#include <type_traits>

#include "mem_common.cuh"

namespace memb200 {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double kTwoPi3 = 8.0 * kPi * kPi * kPi;        // (2 pi)^3
constexpr double kTwoPi4 = 16.0 * kPi * kPi * kPi * kPi; // (2 pi)^4

// 1 - n_a.n_b for two directions given by (eta, phi), without cancellation
__device__ inline double one_minus_cos(double eta_a, double phi_a, double eta_b, double phi_b) {
  const double sh = sinh(0.5 * (eta_a - eta_b)), sn = sin(0.5 * (phi_a - phi_b));
  return 2.0 * (sh * sh + sn * sn) / (cosh(eta_a) * cosh(eta_b));
}

// NEXT-1 (Eq. 7): the k-th jet-parton assignment, role r takes measured jet sig[r].
// n_perm = 24: all permutations of four jets in lexicographic order; 4: b-tags known, order
// (0123), (0132), (1023), (1032); 2: the two b jets swapped; otherwise the record order.
__device__ inline void jet_assignment(int n_perm, int k, int (&sig)[4]) {
  sig[0] = 0; sig[1] = 1; sig[2] = 2; sig[3] = 3;
  if (n_perm == 24) {
    int pool[4] = {0, 1, 2, 3};
    int div = 6, rem = k;
    for (int r = 0; r < 4; ++r) {
      const int idx = rem / div;
      rem -= idx * div;
      sig[r] = pool[idx];
      for (int j = idx; j < 3 - r; ++j) pool[j] = pool[j + 1];
      if (r < 2) div /= (3 - r);
    }
  } else if (n_perm == 4) {
    if (k & 2) { sig[0] = 1; sig[1] = 0; }
    if (k & 1) { sig[2] = 3; sig[3] = 2; }
  } else if (n_perm == 2) {
    if (k & 1) { sig[0] = 1; sig[1] = 0; }
  }
}

// =========================================================================================
// config 1: u dbar -> W+ -> e+ nu, D = 1.  rec = [lep_pT, lep_eta, lep_phi, met_x, met_y]
// DESIGN.md "Config 1" (reading A5): nu_z in [-P, P] charted by s_W with a Breit-Wigner map,
// both roots summed.
// =========================================================================================
struct ProcWenu {
  using real = double;
  static constexpr bool kCompact = false;   // lane compaction in the plain integrate kernel
  static constexpr int kClasses = 0, kPreStages = 0;
  static constexpr bool kSplitC0 = false;
  static constexpr int D = 1, NF = 5, NC = 16;
  enum { LM, LP, LE, LZ, PT, NT2, A, CLO, CHI, DT, ISCLO, DSM, PTNT, IPT2, C0, _N };

  __device__ static void prepare(const DevConst& c, const double* ev, int64_t n, int64_t e, int k, double* ec) {
    const double pT = ev[0 * n + e], eta = ev[1 * n + e], phi = ev[2 * n + e];
    const double mx = ev[3 * n + e], my = ev[4 * n + e];
    const double Pz = c.nu_pz_max;
    const double lE = pT * cosh(eta), lx = pT * cos(phi), ly = pT * sin(phi), lz = pT * sinh(eta);
    const double nT2 = mx * mx + my * my, nT = sqrt(nT2);
    const double a = lx * mx + ly * my;
    // s(nu_z) = 2 (E_l sqrt(nT^2 + nz^2) - a - l_z nz); stationary at nz* = nT sinh(eta)
    const double nz_star = nT * sinh(eta);
    const double s_star = 2.0 * (pT * nT - a);
    const double s_p = 2.0 * (lE * sqrt(nT2 + Pz * Pz) - a - lz * Pz);
    const double s_m = 2.0 * (lE * sqrt(nT2 + Pz * Pz) - a + lz * Pz);
    const double s_min = (nz_star > Pz) ? s_p : (nz_star < -Pz) ? s_m : s_star;
    const double s_max = fmax(s_p, s_m);
    // Breit-Wigner angle through its complement c = pi/2 - t = atan2(m Gam, s - m^2) in (0, pi):
    // events far above the W pole have t within 1e-3 of pi/2, where t itself loses 3-4 digits
    const double c_lo = atan2(c.mWGW, s_min - c.mW2), c_hi = atan2(c.mWGW, s_max - c.mW2);
    const double dt = c_lo - c_hi;
    ec[LM] = pT * exp(-eta);            // E_l - l_z
    ec[LP] = pT * exp(eta);             // E_l + l_z
    ec[LE] = lE; ec[LZ] = lz; ec[PT] = pT; ec[NT2] = nT2; ec[A] = a;
    ec[CLO] = c_lo; ec[CHI] = c_hi; ec[DT] = dt; ec[ISCLO] = 1.0 / sin(c_lo);   // sin(c_lo) = cos(t_lo)
    // s_min - s* without cancellation: E_l E_nu - l_z nu_z = pT nT cosh(eta - y_nu), so at the
    // boundary nu_z = +-P (y_P = +-asinh(P / nT)):  s(+-P) - s* = 4 pT nT sinh^2((eta - y_P) / 2)
    {
      const double yP = asinh(Pz / nT);
      const double shp = sinh(0.5 * (eta - yP)), shm = sinh(0.5 * (eta + yP));
      ec[DSM] = (nz_star > Pz) ? 4.0 * pT * nT * shp * shp : (nz_star < -Pz) ? 4.0 * pT * nT * shm * shm : 0.0;
    }
    ec[PTNT] = pT * nT;
    ec[IPT2] = 1.0 / (pT * pT);
    // dt * (ds/dt * D_W = 1/(m Gam)) * g^4 |V_ud|^2 / 12 * A_q^2 * (4 / (x1 x2 S)) * (4 h^2 = S)
    //    * 1 / (8 pi^2 S E_l E_nu) * (jac = E_nu / (2 rt))
    ec[C0] = dt / c.mWGW * c.g4w * c.V_ud2 / 12.0 * c.A_q2 * 4.0 / (8.0 * kPi * kPi * c.S * lE) * 0.5;
  }

  template <bool PERM, bool GRIDPDF, bool TAB>
  __device__ static double weight_t(const DevConst& c, const double* ec, const double (&u)[D]) { return weight(c, ec, u); }

  __device__ static double weight(const DevConst& c, const double* ec, const double (&u)[D]) {
    // pi/2 - t = c_lo (1 - u) + c_hi u: positive terms only (1 - u is exact)
    const double cc_t = fma(ec[CLO], 1.0 - u[0], ec[CHI] * u[0]);
    double sc, cs;
    sincos_0pi(cc_t, &sc, &cs);
    const double isc = rcp_fast(sc);                  // sc = sin(pi/2 - t) = cos t > 0 inside the window
    const double smm = c.mWGW * (cs * isc);           // m Gam tan t = m Gam cot(pi/2 - t)
    const double sW = c.mW2 + smm;
    // s_W - s_min = m Gam (tan t - tan t_lo) = m Gam sin(dt u) / (cos t cos t_lo): no cancellation
    // at the transverse-mass edge
    double sdt, cdt;
    sincos_0pi(ec[DT] * u[0], &sdt, &cdt);
    const double ds = c.mWGW * sdt * (isc * ec[ISCLO]);
    const double half = 0.5 * (ds + ec[DSM]);
    const double cc = 0.5 * sW + ec[A];
    const double disc = half * (cc + ec[PTNT]);
    if (!(disc > 0.0)) return 0.0;
    const double irt = rsqrt_fast(disc), rt = disc * irt;
    double sum = 0.0;
#pragma unroll
    for (int sgn = -1; sgn <= 1; sgn += 2) {
      const double nz = (cc * ec[LZ] + sgn * ec[LE] * rt) * ec[IPT2];
      if (!(fabs(nz) <= c.nu_pz_max)) continue;
      const double En = sqrt(ec[NT2] + nz * nz);
      const double PE = ec[LE] + En, Pz = ec[LZ] + nz;
      const double x1 = (PE + Pz) * c.inv_sqrt_s, x2 = (PE - Pz) * c.inv_sqrt_s;
      if (!(x1 > 0.0 && x1 < 1.0 && x2 > 0.0 && x2 < 1.0)) continue;
      // both beam orderings: u^2 + t^2 = S (x1^2 (E_l - l_z)^2 + x2^2 (E_l + l_z)^2)
      const double a1 = x1 * ec[LM], a2 = x2 * ec[LP];
      const double me = fma(a1, a1, a2 * a2);
      if (c.pdf_fast) {
        // f f / (x1 x2) = (x1 x2)^(-3/2) ((1 - x1)(1 - x2))^3 = (r yy)^3 with r = (x1 x2)^(-1/2): no division
        const double r = rsqrt_fast(x1 * x2), ry = r * ((1.0 - x1) * (1.0 - x2));
        sum = fma(ry * ry * ry, me, sum);
      } else {
        sum += pdf_pair(c, x1, x2) / (x1 * x2) * me;
      }
    }
    const double w = ec[C0] * sum * irt;
    return isfinite(w) ? w : 0.0;
  }
};

// =========================================================================================
// jets shared by configs 2-4 (O5): E = E_jet (rlo + dr u); direction fixed by the record.
// per-event block of 5 constants per jet: E_jet rlo, E_jet dr, n_x, n_y, n_z
// =========================================================================================
template <typename T> struct JetR { T E, x, y, z; };
using Jet = JetR<double>;

__device__ inline void jet_prepare(const DevConst& c, double Ej, double eta, double phi, double* o) {
  const double st = 1.0 / cosh(eta);
  o[0] = Ej * c.rlo; o[1] = Ej * c.dr;
  o[2] = st * cos(phi); o[3] = st * sin(phi); o[4] = tanh(eta);
}

// returns the parton momentum; tf accumulates E * T(E_jet; E) (see tf_accum)
template <typename T>
__device__ __forceinline__ JetR<T> jet_point(const DevConstR<T>& c, const T* o, T u, TfAcc<T>& tf) {
  const T x = fma(c.dr, u, c.rlo);
  tf_accum<true>(c, rcp_fast(x), tf);
  JetR<T> j;
  j.E = fma(o[1], u, o[0]);
  j.x = j.E * o[2]; j.y = j.E * o[3]; j.z = j.E * o[4];
  return j;
}

// parton momentum alone (the transfer functions are accumulated separately)
template <typename T>
__device__ __forceinline__ JetR<T> jet_mom(const T* o, T u) {
  JetR<T> j;
  j.E = fma(o[1], u, o[0]);
  j.x = j.E * o[2]; j.y = j.E * o[3]; j.z = j.E * o[4];
  return j;
}

// =========================================================================================
// config 2: q qbar -> Z -> b bbar, D = 2.  rec = [E1, eta1, phi1, E2, eta2, phi2]
// DESIGN.md "Config 2"; transverse boost O7 (reading A6)
// =========================================================================================
struct ProcZbb {
  using real = double;
  static constexpr bool kCompact = false;   // lane compaction in the plain integrate kernel
  static constexpr int kClasses = 0, kPreStages = 0;
  static constexpr bool kSplitC0 = false;
  static constexpr int D = 2, NF = 6, NC = 12;
  enum { J0 = 0, J1 = 5, C0 = 10, KT = 11 };

  __device__ static void prepare(const DevConst& c, const double* ev, int64_t n, int64_t e, int k, double* ec) {
    double vol = 1.0, sth = 1.0, eta[2], phi[2];
    for (int j = 0; j < 2; ++j) {
      const double Ej = ev[(3 * j) * n + e];
      eta[j] = ev[(3 * j + 1) * n + e]; phi[j] = ev[(3 * j + 2) * n + e];
      jet_prepare(c, Ej, eta[j], phi[j], ec + 5 * j);
      vol *= Ej * c.dr;
      sth *= (1.0 / cosh(eta[j])) / (2.0 * kTwoPi3);
    }
    // 1 - n1T.n2T = (cosh eta1 cosh eta2 - cos dphi)/(cosh eta1 cosh eta2), as a sum of squares
    const double sp = sinh(0.5 * (eta[0] + eta[1])), sm = sinh(0.5 * (eta[0] - eta[1])), sn = sin(0.5 * (phi[0] - phi[1]));
    ec[KT] = (sp * sp + sm * sm + 2.0 * sn * sn) / (cosh(eta[0]) * cosh(eta[1]));
    // the slot n_y of jet 0 is not needed: it holds K12 = 1 - n1.n2
    ec[J0 + 3] = one_minus_cos(eta[0], phi[0], eta[1], phi[1]);
    // vol * prod sin(theta)/(2 (2pi)^3) * (2pi)^4 * (2/S) * g_Z^4 * A_q^2 * 4 (flux) * S (u^2, t^2 carry 4 h^2)
    ec[C0] = vol * sth * kTwoPi4 * (2.0 * c.inv_S) * c.gz4 * c.A_q2 * 4.0 * c.S;
  }

  template <bool PERM, bool GRIDPDF, bool TAB>
  __device__ static double weight_t(const DevConst& c, const double* ec, const double (&u)[D]) { return weight(c, ec, u); }

  __device__ static double weight(const DevConst& c, const double* ec, const double (&u)[D]) {
    TfAcc<double> tfa{0.0, 1.0};
    const Jet p1 = jet_point(c, ec + J0, u[0], tfa), p2 = jet_point(c, ec + J1, u[1], tfa);
    const double tf = tfa.fac * exp_tab<true>(-tfa.esum);
    // O7 without the cancellation in 1 - beta^2 (nearly collinear jets): with P = p1 + p2,
    //   P_E'^2 = P_E^2 - P_T^2 = p1z^2 + p2z^2 + 2 E1 E2 (1 - n1T.n2T)
    //   E_i'   = gamma (E_i - beta.p_iT) = (p_iz^2 + E1 E2 (1 - n1T.n2T)) / P_E'
    //   s-hat  = 2 E1 E2 (1 - n1.n2) = (P_E' + P_z)(P_E' - P_z)
    const double e12 = p1.E * p2.E, ekt = e12 * ec[KT];
    const double Pz = p1.z + p2.z;
    const double PEb2 = fma(p1.z, p1.z, fma(p2.z, p2.z, 2.0 * ekt));
    const double iPEb = rsqrt_fast(PEb2), PEb = PEb2 * iPEb;
    const double E1 = fma(p1.z, p1.z, ekt) * iPEb, E2 = fma(p2.z, p2.z, ekt) * iPEb;
    const double shat = 2.0 * e12 * ec[J0 + 3];
    const double Xb = PEb + fabs(Pz), Xs = shat * rcp_fast(Xb);
    const double x1 = (Pz >= 0.0 ? Xb : Xs) * c.inv_sqrt_s, x2 = (Pz >= 0.0 ? Xs : Xb) * c.inv_sqrt_s;
    if (!(x1 > 0.0 && x1 < 1.0 && x2 > 0.0 && x2 < 1.0)) return 0.0;
    // u = -2 qa.p2', t = -2 qa.p1' for qa = q1 and qa = q2 (both beam orderings), in units of -2h
    const double u1 = x1 * (E2 - p2.z), t1 = x1 * (E1 - p1.z);
    const double u2 = x2 * (E2 + p2.z), t2 = x2 * (E1 + p1.z);
    const double me = c.z_cu * (u1 * u1 + u2 * u2) + c.z_ct * (t1 * t1 + t2 * t2);
    const double dz = shat - c.mZ2;
    const double w = ec[C0] * tf * pdf_pair(c, x1, x2) * me * rcp_fast(shat * fma(dz, dz, c.mZGZ2));
    return isfinite(w) ? w : 0.0;
  }
};

// =========================================================================================
// config 3: t tbar -> b l nu  bbar q qbar', D = 6 (also the config-5 integrand).
// rec = [lep_pT, lep_eta, lep_phi, (E, eta, phi) x {b_had, b_lep, q, qbar'}, met, met_phi]
// DESIGN.md "Config 3" (reading A7): u0..u3 jet energies, u4 eta_nu flat in [-H, H],
// u5 leptonic s_W through the Breit-Wigner map; nu azimuth = MET azimuth.
// =========================================================================================
template <typename T>
struct ProcTTljetsR {
  using real = T;
  static constexpr bool kCompact = false;
  static constexpr int kClasses = 0, kPreStages = 0;
  static constexpr int D = 6, NF = 17, NC = 44;
  static constexpr bool kSplitC0 = !std::is_same<T, double>::value;
  enum { LE, LX, LY, LZ, ELI, EL, LPT2, OMC, CPN, SPN,   // lepton, neutrino azimuth
         J0 = 10, J1 = 15, J2 = 20, J3 = 25,            // b_had, b_lep, q, qbar'
         KBL = 30,                                      // b_lep . l / E_b
         K02, K23, K03,                                 // 1 - n.n of (b_had,q), (q,qbar'), (b_had,qbar')
         NA, NB, NC_,                                   // b_lep . nu = E_b nuT (NA e^eta + NB e^-eta - NC_)
         C0, SW0, _N };

  __device__ static void prepare(const DevConst& c, const double* ev, int64_t n, int64_t e, int k, double* ec) {
    const double lpT = ev[0 * n + e], leta = ev[1 * n + e], lphi = ev[2 * n + e];
    const double mphi = ev[16 * n + e];
    const double lE = lpT * cosh(leta);
    ec[LE] = lE; ec[LX] = lpT * cos(lphi); ec[LY] = lpT * sin(lphi); ec[LZ] = lpT * sinh(leta);
    ec[EL] = exp(leta); ec[ELI] = exp(-leta);
    ec[LPT2] = 2.0 * lpT;
    const double sd = sin(0.5 * (lphi - mphi));
    ec[OMC] = 2.0 * sd * sd;            // 1 - cos(phi_l - phi_nu)
    ec[CPN] = cos(mphi); ec[SPN] = sin(mphi);
    int sig[4];
    jet_assignment(c.n_perm, k, sig);                  // role j takes measured jet sig[j]
    double vol = 1.0, sth = 1.0, eta_j[4], phi_j[4];
    for (int j = 0; j < 4; ++j) {
      const double Ej = ev[(3 + 3 * sig[j]) * n + e];
      eta_j[j] = ev[(4 + 3 * sig[j]) * n + e]; phi_j[j] = ev[(5 + 3 * sig[j]) * n + e];
      jet_prepare(c, Ej, eta_j[j], phi_j[j], ec + J0 + 5 * j);
      vol *= Ej * c.dr;
      sth *= (1.0 / cosh(eta_j[j])) / (2.0 * kTwoPi3);
    }
    {   // b_lep . l = E_b * lpT (cosh(d eta) - cos(d phi)) / cosh(eta_b)
      const double sh = sinh(0.5 * (eta_j[1] - leta)), sn = sin(0.5 * (phi_j[1] - lphi));
      ec[KBL] = lpT * 2.0 * (sh * sh + sn * sn) / cosh(eta_j[1]);
    }
    ec[K02] = one_minus_cos(eta_j[0], phi_j[0], eta_j[2], phi_j[2]);
    ec[K23] = one_minus_cos(eta_j[2], phi_j[2], eta_j[3], phi_j[3]);
    ec[K03] = one_minus_cos(eta_j[0], phi_j[0], eta_j[3], phi_j[3]);
    {   // b_lep . nu = E_b nuT (cosh(eta_nu - eta_b) - cos(phi_nu - phi_b)) / cosh(eta_b)
      const double chb = cosh(eta_j[1]);
      ec[NA] = 0.5 * exp(-eta_j[1]) / chb; ec[NB] = 0.5 * exp(eta_j[1]) / chb;
      ec[NC_] = cos(mphi - phi_j[1]) / chb;
    }
    const double H = c.nu_eta_max;
    // vol: jets, 2H, dt_W; jets' sin(theta)/(2 (2pi)^3); lepton 1/(2 E_l (2pi)^3); neutrino 1/(2 (2pi)^3)
    // [nuT^2/s_W stays in the point]; (2pi)^4 (2/S); flux 4/(x1 x2 S) [1/s-hat stays];
    // ds_W/dt * D_W(s_W) = 1/(m_W Gam_W); g_s^4; decays (1/2)(4 g^4 V_tb^2) and (1/2) 3 (4 g^4 V_tb^2) V_ud^2
    ec[C0] = vol * (2.0 * H) * c.tW_dt * sth / (2.0 * lE * kTwoPi3) / (2.0 * kTwoPi3) * kTwoPi4 * (2.0 * c.inv_S) *
             4.0 / c.mWGW * c.gs4 * (2.0 * c.g4w * c.V_tb2) * (6.0 * c.g4w * c.V_tb2 * c.V_ud2);
    ec[SW0] = 0.0;
    for (int k = _N; k < NC; ++k) ec[k] = 0.0;
  }

  __device__ static T weight(const DevConstR<T>& c, const T* ec, const T (&u)[D]) {
    return weight_t<false, false, false>(c, ec, u);
  }

  // PERM = false: the record's own jet-parton assignment (ec = one block of NC constants).
  // PERM = true: NEXT-1, the sum over c.n_perm assignments (Eq. 7), ec = n_perm
  // blocks.  Everything that depends only on the point -- energy fractions, transfer functions
  // (functions of E / E_jet alone), the neutrino -- is computed once; only the jet momenta, the
  // invariants, the boost and the matrix element are repeated per assignment.
  // TAB: table-driven exp (fp64); true in every integrate kernel (mem_kernels.cuh).
  template <bool PERM, bool GRIDPDF, bool TAB>
  __device__ static T weight_t(const DevConstR<T>& c, const T* ec0, const T (&u)[D]) {
    const T* ec = ec0;
    // ---- S2: jet energy fractions x_j = E_j / E_jet, neutrino rapidity.
    // g = e^(eta_nu - eta_l); cosh(d eta) - cos(d phi) = ((g-1)^2/2 + (1 - cos d phi) g) / g =: denp / (LPT2 g)
    const T x0 = fma(c.dr, u[0], c.rlo), x1j = fma(c.dr, u[1], c.rlo), x2j = fma(c.dr, u[2], c.rlo), x3 = fma(c.dr, u[3], c.rlo);
    const T H = c.nu_eta_max;
    const T eta_nu = fma(T(2.0) * H, u[4], -H);
    const T en = b_exp<TAB>(eta_nu);
    const T g = en * ec[ELI];
    const T gm1 = g - T(1.0);
    const T denp = ec[LPT2] * fma(T(0.5) * gm1, gm1, ec[OMC] * g);
    if (!(denp > T(0))) return T(0);
    // one reciprocal for the six divisors (product tree, then back-substitution)
    const T p01 = x0 * x1j, p23 = x2j * x3, p45 = en * denp, p03 = p01 * p23;
    const T inv = rcp_fast(p03 * p45);
    const T i45 = inv * p03, i03 = inv * p45;
    const T eni = i45 * denp, idenp = i45 * en;
    const T i01 = i03 * p23, i23 = i03 * p01;
    const T ix0 = i01 * x1j, ix1 = i01 * x0, ix2 = i23 * x3, ix3 = i23 * x2j;
    // ---- S6: transfer functions (one exponential per jet and one for the sum, see tf_accum)
    TfAcc<T> tfa{T(0), T(1)};
    tf_accum<TAB>(c, ix0, tfa); tf_accum<TAB>(c, ix1, tfa); tf_accum<TAB>(c, ix2, tfa); tf_accum<TAB>(c, ix3, tfa);
    const T tf = tfa.fac * x_exp<TAB>(-tfa.esum);
    // ---- S2: neutrino from the mapped leptonic W mass
    const T t = fma(c.tW_dt, u[5], c.tW_lo);
    const T smm = c.mWGW * m_tan(t);
    const T sW = c.mW2 + smm;
    const T iden = g * idenp;                                                    // 1 / (2 pT_l (cosh - cos))
    const T nuT = sW * iden;
    const T hnuT = T(0.5) * nuT;
    const T nE = hnuT * (en + eni), nx = nuT * ec[CPN], ny = nuT * ec[SPN], nz = hnuT * (en - eni);
    T sum = T(0);
    const int n_perm = PERM ? c.n_perm : 1;
    for (int k = 0; k < n_perm; ++k, ec += NC) {
    const JetR<T> bh = jet_mom(ec + J0, u[0]), bl = jet_mom(ec + J1, u[1]);
    const JetR<T> q = jet_mom(ec + J2, u[2]), qb = jet_mom(ec + J3, u[3]);
    // ---- S3: invariants through per-event angular constants
    const T bl_nu = bl.E * nuT * (fma(ec[NA], en, ec[NB] * eni) - ec[NC_]);
    const T bl_l = bl.E * ec[KBL];
    const T st_m = fma(T(2.0), bl_l + bl_nu, smm + (c.mW2 - c.mt2));           // s_t - m_t^2
    const T bh_q = bh.E * q.E * ec[K02], q_qb = q.E * qb.E * ec[K23], bh_qb = bh.E * qb.E * ec[K03];
    const T swh_m = fma(T(2.0), q_qb, -c.mW2);                                 // s_Whad - m_W^2
    const T stb_m = fma(T(2.0), bh_q + q_qb + bh_qb, -c.mt2);                  // s_tbar - m_t^2
    // ---- S3: top momenta, transverse boost O7 (only the two boosted energies are needed)
    const T tE = bl.E + ec[LE] + nE, tx = bl.x + ec[LX] + nx, ty = bl.y + ec[LY] + ny, tz = bl.z + ec[LZ] + nz;
    const T aE = bh.E + q.E + qb.E, ax = bh.x + q.x + qb.x, ay = bh.y + q.y + qb.y, az = bh.z + q.z + qb.z;
    const T PE = tE + aE, Px = tx + ax, Py = ty + ay, Pz = tz + az;
    // gamma (E - beta.p) = (E P_E - p_T.P_T) / sqrt(P_E^2 - P_T^2): no division by P_E
    const T M2 = fma(PE, PE, -fma(Px, Px, Py * Py));
    bool ok = M2 > T(0);                     // cuts are predicates: the select at the end discards the point
    const T rM = m_rsqrt(M2);
    // the boosted total energy is sqrt(P_E^2 - P_T^2) itself; the antitop's is the rest
    const T tEb = rM * fma(tE, PE, -fma(Px, tx, Py * ty));
    const T PEb = M2 * rM, aEb = PEb - tEb;
    const T x1 = (PEb + Pz) * c.inv_sqrt_s, x2 = (PEb - Pz) * c.inv_sqrt_s;
    ok = ok && x1 > T(0) && x1 < T(1.0) && x2 > T(0) && x2 < T(1.0);
    const T xx = x1 * x2, shat = xx * c.S;
    ok = ok && T(4.0) * c.mt2 < shat;                                             // reading A9
    // ---- S5: production.  tau1 = (q1.pt + q2.ptb)/s-hat, tau2 = (q2.pt + q1.ptb)/s-hat
    // one reciprocal square root serves 1/s-hat and the toy PDF's (x1 x2)^(-1/2) = sqrt(S) / sqrt(s-hat)
    const T rs = m_rsqrt(shat);
    const T ish = rs * rs;
    const T hs = T(0.5) * c.sqrt_s * ish;
    const T tau1 = hs * fma(x1, tEb - tz, x2 * (aEb + az));
    const T tau2 = hs * fma(x2, tEb + tz, x1 * (aEb - az));
    const T rho = T(4.0) * c.mt2 * ish;
    const T t12 = tau1 * tau2;
    // ---- S5: propagators and decays
    const T t_l = fma(T(0.5), sW, bl_l);                                       // p_t . l
    const T a_q = bh_q + q_qb;                                                 // p_tbar . q
    T decprop, iT;                                                             // decays x propagators, 1/(tau1 tau2)
    if constexpr (kSplitC0) {
      // fp32: keep every intermediate inside the single-precision range
      iT = rcp_fast(t12);
      decprop = (t_l * bl_nu * rcp_fast(fma(st_m, st_m, c.mtGt2))) * (a_q * rcp_fast(fma(stb_m, stb_m, c.mtGt2))) *
                (bh_qb * rcp_fast(fma(swh_m, swh_m, c.mWGW2)));
    } else {
      // one reciprocal for 1/(tau1 tau2) and the three propagator denominators
      const T dens = fma(st_m, st_m, c.mtGt2) * fma(stb_m, stb_m, c.mtGt2) * fma(swh_m, swh_m, c.mWGW2);
      const T inv = rcp_fast(t12 * dens);
      iT = inv * dens;
      decprop = t_l * bl_nu * a_q * bh_qb * (inv * t12);
    }
    const T tt = fma(tau1, tau1, tau2 * tau2);
    const T Mgg = fma(iT, T(1.0) / T(6.0), -T(0.375)) * (tt + rho - T(0.25) * rho * rho * iT);
    const T Mqq = tt + T(0.5) * rho;
    const TtLumi<T> lum = tt_lumi<GRIDPDF>(c, x1, x2, rs * c.sqrt_s);
    const T prod = fma(lum.gg, Mgg, lum.qq * Mqq);                             // flavour sum incl. the PDFs
    // ---- S4, S7
    const T core = ish * prod * decprop;
    if constexpr (PERM) { if (ok && isfinite(core)) sum += core; }
    else sum = ok ? core : T(0);                            // a non-finite value is caught by the final test
    }
    const T pt = tf * (nuT * iden) * sum;
    // fp64: the per-event constant (identical for every assignment) is applied here; fp32: by the
    // caller in fp64 (it would underflow)
    const T w = kSplitC0 ? pt : ec0[C0] * pt;
    return isfinite(w) ? w : T(0);
  }
};
using ProcTTljets = ProcTTljetsR<double>;
using ProcTTljetsF = ProcTTljetsR<float>;   // reading A15

// =========================================================================================
// config 4: t tbar -> b l+ nu  bbar l- nubar, D = 8.
// rec = [(pT, eta, phi) l+, (pT, eta, phi) l-, (E, eta, phi) b, (E, eta, phi) bbar, met_x, met_y]
// DESIGN.md "Config 4" (readings A3, A8, A12; Eq. 7-8): u0,u1 jet energies,
// u2..u5 the Breit-Wigner mapped s_W+, s_t, s_W-, s_tbar, u6,u7 the total neutrino pT around the
// measured MET (Gaussian MET TF).  Every (nu, nubar) solution of Eq. 8 is summed.
//
// Lepton and jet directions are fixed per event, so on each top side the plane normal
// d = n_l - n_b, the slopes of nu_z and E_nu in (nu_x, nu_y) and the quadratic part (a, b, c) of
// the conic E_nu^2 = |nu|^2 are per-event constants; a point only moves the offsets al0, la0.
// Likewise p_b.p_nu = Delta/2 and p_t.p_l = b.l + s_W/2 are fixed by the sampled masses, so the
// decay factors do not depend on the solution.
// =========================================================================================

// largest real root of z^3 + c2 z^2 + c1 z + c0: Cardano / trigonometric form as a single-precision START (cube
// root through cbrtf; cos(acos(c)/3) = T(s), s = sqrt((1 + c)/2), as a degree-6 polynomial: both ~1e-6), then three
// Newton steps on the cubic in fp64, which converge to the root to rounding.  The closed forms in fp64 (libdevice
// cbrt, acos) cost ~130 instructions with both branches of a diverged warp and 8 KB of code; this is ~50.
__device__ __forceinline__ double cubic_largest_root(double c2, double c1, double c0) {
  const double sh = c2 * (1.0 / 3.0);
  const double P3 = fma(-c2, sh, c1) * (1.0 / 3.0);                  // P/3, P = c1 - c2^2/3
  const double Qh = 0.5 * fma(sh, fma(2.0 * sh, sh, -c1), c0);       // Q/2, Q = 2 c2^3/27 - c2 c1/3 + c0
  const double disc = fma(Qh, Qh, P3 * P3 * P3);
  double w;
  if (disc > 0.0) {
    const double sq = sqrt(disc);
    const double a3 = (Qh > 0.0) ? -(Qh + sq) : (sq - Qh);           // A^3
    const double aa = fabs(a3);
    double A;
    if (aa > 1e-30 && aa < 1e30) A = (double)cbrtf((float)a3);
    else A = cbrt(a3);                                               // outside the comfortable float range: rare
    w = (A != 0.0) ? fma(-P3, rcp_fast(A), A) : 0.0;
  } else {
    const double m2 = -P3, m = sqrt(m2);
    if (m == 0.0) {
      w = 0.0;
    } else {
      double c = -Qh * rcp_fast(m2 * m);
      c = fmin(1.0, fmax(-1.0, c));
      // T(s) = cos((2/3) acos(s)) on [0, 1] (own Chebyshev fit, 4e-7)
      const float sf = sqrtf(0.5f * (1.0f + (float)c));
      float T = -0.002122052712365985f;
      T = fmaf(T, sf, 0.010519994422793388f);
      T = fmaf(T, sf, -0.026367755606770515f);
      T = fmaf(T, sf, 0.05142129212617874f);
      T = fmaf(T, sf, -0.11077950149774551f);
      T = fmaf(T, sf, 0.5773273706436157f);
      T = fmaf(T, sf, 0.5000004172325134f);
      w = 2.0 * m * (double)T;
    }
  }
  double z = w - sh;
#pragma unroll
  for (int it = 0; it < 3; ++it) {
    const double f = fma(fma(z + c2, z, c1), z, c0);
    const double fp = fma(fma(3.0, z, 2.0 * c2), z, c1);
    const double zn = fma(-f, rcp_fast(fp), z);
    if (isfinite(zn)) z = zn;
  }
  return z;
}

// real roots of x^4 + a3 x^3 + a2 x^2 + a1 x + a0 (Ferrari; reading A12); returns 0, 2 or 4.
// Roots of the factor y^2 + s y + m come first, then those of y^2 - s y + n.
__device__ __forceinline__ int quartic_real_roots(double a3, double a2, double a1, double a0, double (&x)[4]) {
  const double a32 = a3 * a3;
  const double p = fma(-0.375, a32, a2);
  const double q = fma(a3, fma(0.125, a32, -0.5 * a2), a1);
  const double r = fma(a3, fma(a3, fma(-3.0 / 256.0, a32, a2 * (1.0 / 16.0)), -0.25 * a1), a0);
  const double shift = -0.25 * a3;
  double z0 = cubic_largest_root(2.0 * p, fma(p, p, -4.0 * r), -q * q);
  if (!(z0 > 0.0)) z0 = 0.0;
  const double s = sqrt(z0);
  double qs;
  if (s > 0.0) qs = q * rcp_fast(s);
  else { const double t = fma(p, p, -4.0 * r); qs = (t > 0.0) ? sqrt(t) : 0.0; }
  const double m = 0.5 * (p + z0 - qs), n = 0.5 * (p + z0 + qs);
  int cnt = 0;
  const double d1 = fma(-4.0, m, z0), d2 = fma(-4.0, n, z0);
  if (d1 >= 0.0) {
    const double ya = 0.5 * (-s - sqrt(d1));
    const double yb = (ya != 0.0) ? m * rcp_fast(ya) : 0.5 * (-s + sqrt(d1));
    x[0] = ya + shift; x[1] = yb + shift; cnt = 2;
  }
  if (d2 >= 0.0) {
    const double ya = 0.5 * (s + sqrt(d2));
    const double yb = (ya != 0.0) ? n * rcp_fast(ya) : 0.5 * (s - sqrt(d2));
    if (cnt == 0) { x[0] = ya + shift; x[1] = yb + shift; }
    else { x[2] = ya + shift; x[3] = yb + shift; }
    cnt += 2;
  }
  return cnt;
}

struct ProcTTdilep {
  using real = double;
  static constexpr bool kCompact = true;   // lane compaction in the plain integrate kernel
  static constexpr bool kSplitC0 = false;
  static constexpr int D = 8, NF = 14, NC = 64;
  static constexpr int kNewton = 3;      // Newton steps on the un-squared equations per root
  // stages of the lane-compacting loop (mem_kernels.cuh) and the classes its queues sort points into
  static constexpr int kModeFull = 0, kModeClassify = 1, kModeCheap = 2;
  static constexpr int kClasses = 2;     // 2 or 4 real roots of the resultant quartic
  static constexpr int kPreStages = 0;         // the b.nu > 0 test rejects only ~15 % of the points: classify directly
  static constexpr int kCheapBlock = 0;
  __device__ static double cheap_test(const DevConst&, const double*, double, double) { return 1.0; }
  // per top side s (0: l+, b; 1: l-, bbar), 14 constants each, at S0 + 14 s:
  //   LE LX LY LZ   lepton four-momentum
  //   I2EL          1 / (2 E_l)
  //   ELK           E_l (1 - n_l.n_b)                      (b.l = E_b ELK)
  //   IDZ NLZ       1 / d_z, n_l,z                         (al0 = kappa IDZ, la0 = w0 + NLZ al0)
  //   AX AY LAX LAY slopes of nu_z and E_nu
  //   MX MY         (n_l x n_b)_x,y                        (Jacobian)
  // then DX DY DZ of each side, the conics' quadratic parts, the resultant's constant
  // coefficients, jets, MET, C0.
  enum { LE, LX, LY, LZ, I2EL, ELK, IDZ, NLZ, AX, AY, LAX, LAY, MX, MY, SIDE = 14,
         S0 = 0, S1 = 14,
         DX0 = 28, DY0, DZ0, DX1, DY1, DZ1,                 // 28..33
         CA0 = 34, CB0, CC0, CA1, CB1, CC1,                 // 34..39 conic a, b, c
         U2 = 40, V1, W3, IR4,                              // 40..43
         J0 = 44, J1 = 49,                                  // jets: E rlo, E dr, n_x, n_y, n_z
         IEJ0 = 54, IEJ1,                                   // 1 / E_jet
         METX = 56, METY, MSPAN, MEXP, C0, PTX, PTY, _N };  // 56..62

  __device__ static void prepare(const DevConst& c, const double* ev, int64_t n, int64_t e, int k, double* ec) {
    for (int k = 0; k < NC; ++k) ec[k] = 0.0;
    int sig[4];
    jet_assignment(c.n_perm, k, sig);                  // top side s pairs its lepton with measured jet sig[s]
    double vol = 1.0, sth = 1.0, ptx = 0.0, pty = 0.0, lE[2];
    for (int s = 0; s < 2; ++s) {
      const double pT = ev[(3 * s) * n + e], eta = ev[(3 * s + 1) * n + e], phi = ev[(3 * s + 2) * n + e];
      const double Ej = ev[(6 + 3 * sig[s]) * n + e], jeta = ev[(7 + 3 * sig[s]) * n + e], jphi = ev[(8 + 3 * sig[s]) * n + e];
      double* o = ec + S0 + SIDE * s;
      const double E = pT * cosh(eta);
      lE[s] = E;
      o[LE] = E; o[LX] = pT * cos(phi); o[LY] = pT * sin(phi); o[LZ] = pT * sinh(eta);
      o[I2EL] = 0.5 / E;
      const double stl = 1.0 / cosh(eta), stb = 1.0 / cosh(jeta);
      const double nlx = stl * cos(phi), nly = stl * sin(phi), nlz = tanh(eta);
      const double nbx = stb * cos(jphi), nby = stb * sin(jphi), nbz = tanh(jeta);
      o[ELK] = E * one_minus_cos(eta, phi, jeta, jphi);
      const double dx = nlx - nbx, dy = nly - nby;
      // d_z = tanh(eta_l) - tanh(eta_b) = sinh(eta_l - eta_b) / (cosh eta_l cosh eta_b)
      const double dz = sinh(eta - jeta) * stl * stb;
      const double idz = 1.0 / dz;
      o[IDZ] = idz; o[NLZ] = nlz;
      const double ax = -dx * idz, ay = -dy * idz;
      const double lax = nlx + nlz * ax, lay = nly + nlz * ay;
      o[AX] = ax; o[AY] = ay; o[LAX] = lax; o[LAY] = lay;
      o[MX] = nly * nbz - nlz * nby; o[MY] = nlz * nbx - nlx * nbz;
      ec[DX0 + 3 * s] = dx; ec[DY0 + 3 * s] = dy; ec[DZ0 + 3 * s] = dz;
      ec[CA0 + 3 * s] = 1.0 + ax * ax - lax * lax;
      ec[CB0 + 3 * s] = 2.0 * (ax * ay - lax * lay);
      ec[CC0 + 3 * s] = 1.0 + ay * ay - lay * lay;
      jet_prepare(c, Ej, jeta, jphi, ec + J0 + 5 * s);
      ec[IEJ0 + s] = 1.0 / Ej;
      vol *= Ej * c.dr;
      sth *= stb / (2.0 * kTwoPi3);
      ptx += o[LX]; pty += o[LY];
    }
    ec[PTX] = ptx; ec[PTY] = pty;
    const double a1 = ec[CA0], b1 = ec[CB0], c1 = ec[CC0], a2 = ec[CA1], b2 = ec[CB1], c2 = ec[CC1];
    ec[U2] = c1 * a2 - c2 * a1; ec[V1] = c1 * b2 - c2 * b1; ec[W3] = b1 * a2 - b2 * a1;
    ec[IR4] = 1.0 / (ec[U2] * ec[U2] - ec[V1] * ec[W3]);
    ec[METX] = ev[12 * n + e]; ec[METY] = ev[13 * n + e];
    const double span = c.met_sigma * c.met_nsigma;
    ec[MSPAN] = span;
    ec[MEXP] = -0.5 * c.met_nsigma * c.met_nsigma;
    // vol: jets, dt_W^2 dt_t^2, (2 n sigma)^2; jets' sin(theta)/(2 (2pi)^3); leptons 1/(2 E_l (2pi)^3);
    // (2pi)^4 (2/S); prod_k ds_k/dt_k D_k = 1/(m_W Gam_W)^2 1/(m_t Gam_t)^2; neutrinos 1/((2pi)^6 4) and
    // J/(E_nu E_nubar) = 1/(16 E_l+ E_l- E_b E_bbar |..|) [1/(E_b E_bbar |..|) stays in the point];
    // flux 4/(x1 x2 S) [1/s-hat stays]; T_MET norm 1/(2 pi sigma^2); g_s^4; decays (1/2)(4 g^4 V_tb^2) each
    ec[C0] = vol * c.tW_dt * c.tW_dt * c.tT_dt * c.tT_dt * (4.0 * span * span) * sth /
             (2.0 * lE[0] * kTwoPi3) / (2.0 * lE[1] * kTwoPi3) * kTwoPi4 * (2.0 * c.inv_S) /
             (c.mWGW * c.mWGW * c.mtGt * c.mtGt) / (kTwoPi3 * kTwoPi3 * 4.0) / (16.0 * lE[0] * lE[1]) * 4.0 /
             (2.0 * kPi * c.met_sigma * c.met_sigma) * c.gs4 * (2.0 * c.g4w * c.V_tb2) * (2.0 * c.g4w * c.V_tb2);
  }

  // PERM = true: NEXT-1, both assignments of the two b jets (ec = 2 blocks of NC constants)
  template <bool PERM, bool GRIDPDF, bool TAB_UNUSED>
  __device__ static double weight_t(const DevConst& c, const double* ec, const double (&u)[D]) {
    if (!PERM) return weight_rt<GRIDPDF, true>(c, ec, u, kModeFull);
    double w = 0.0;
#pragma unroll 1
    for (int k = 0; k < c.n_perm; ++k) w += weight_rt<GRIDPDF, false>(c, ec + k * NC, u, kModeFull);
    return w;
  }

  __device__ static double weight(const DevConst& c, const double* ec, const double (&u)[D]) {
    return weight_rt<false, true>(c, ec, u, kModeFull);
  }

  // mode (a warp-uniform run-time flag: kModeCheap returns 1 after the cheap kinematic tests, kModeClassify the
  // class of the point, 0 = no real root, 1 = two, 2 = four; see the staged loop in mem_kernels.cuh).  Formerly
  // count_only (a warp-uniform run-time flag, so that the prelude exists once in the kernel: the
  // config-4 kernel is instruction-cache bound, profiles/r01_ncu_config4.md): stop after the resultant
  // quartic and return its number of real roots (0, 2, 4) -- what the lane-compacting loop
  // (mem_kernels.cuh) sorts points by before it runs the per-solution part on full warps.
  // TAB: table-driven exp (+5.8 % in the single-assignment kernel; the two-assignment kernel, tighter on
  // registers, loses 9 % with it and keeps libdevice's exp)
  template <bool GRIDPDF, bool TAB>
  __device__ static double weight_rt(const DevConst& c, const double* ec, const double (&u)[D], int mode) {
    // ---- S2: jets
    const double xb0 = fma(c.dr, u[0], c.rlo), xb1 = fma(c.dr, u[1], c.rlo);
    const double ixb0 = rcp_fast(xb0), ixb1 = rcp_fast(xb1);
    const double Eb0 = fma(ec[J0 + 1], u[0], ec[J0]), Eb1 = fma(ec[J1 + 1], u[1], ec[J1]);
    const double iEb0 = ixb0 * ec[IEJ0], iEb1 = ixb1 * ec[IEJ1];
    // ---- S2: the four mapped masses, s_k - m_k^2 = m Gam tan t_k (O6)
    const double tk[4] = {fma(c.tW_dt, u[2], c.tW_lo), fma(c.tT_dt, u[3], c.tT_lo), fma(c.tW_dt, u[4], c.tW_lo),
                          fma(c.tT_dt, u[5], c.tT_lo)};
    double tn[4];
    tan_bw_n<4>(tk, tn);
    const double smW0 = c.mWGW * tn[0], smT0 = c.mtGt * tn[1], smW1 = c.mWGW * tn[2], smT1 = c.mtGt * tn[3];
    const double sW0 = c.mW2 + smW0, sW1 = c.mW2 + smW1;
    const double dm2 = c.mt2 - c.mW2;
    // Delta/(2 E_b) = b.nu / E_b = ((s_t - s_W)/2 - b.l) / E_b must be positive
    const double hD0 = fma(0.5 * (dm2 + (smT0 - smW0)), iEb0, -ec[S0 + ELK]);
    const double hD1 = fma(0.5 * (dm2 + (smT1 - smW1)), iEb1, -ec[S1 + ELK]);
    if (!(hD0 > 0.0 && hD1 > 0.0)) return 0.0;
    if (mode == kModeCheap) return 1.0;
    // ---- S2: total neutrino pT and the Gaussian MET transfer function (A8)
    const double g6 = fma(2.0, u[6], -1.0), g7 = fma(2.0, u[7], -1.0);
    const double Sx = fma(ec[MSPAN], g6, ec[METX]), Sy = fma(ec[MSPAN], g7, ec[METY]);
    // ---- everything of the point that does not depend on the solution, folded into one factor now (the full pass
    // only), so that it need not stay live -- or be spilled -- across the solution loop: S5 decays (p_t.p_l)(p_b.p_nu)
    // per side, S6 jet transfer functions and the MET Gaussian (one shared exponential), 1/(E_b E_bbar) of the Jacobian
    double pre = 0.0;
    if (mode == kModeFull) {
      TfAcc<double> tfa{0.0, 1.0};
      tf_accum<TAB>(c, ixb0, tfa);
      tf_accum<TAB>(c, ixb1, tfa);
      const double targ = fma(ec[MEXP], fma(g6, g6, g7 * g7), -tfa.esum);
      const double tf_tmet = tfa.fac * (TAB ? exp_tab<true>(targ) : exp(targ));
      const double dec = fma(Eb0, ec[S0 + ELK], 0.5 * sW0) * (Eb0 * hD0) * fma(Eb1, ec[S1 + ELK], 0.5 * sW1) * (Eb1 * hD1);
      pre = ec[C0] * tf_tmet * dec * (iEb0 * iEb1);
    }
    // ---- S2: offsets of nu_z and E_nu on each side, conic linear/constant parts
    const double w00 = sW0 * ec[S0 + I2EL], w01 = sW1 * ec[S1 + I2EL];
    const double al0 = (hD0 - w00) * ec[S0 + IDZ], al1 = (hD1 - w01) * ec[S1 + IDZ];
    const double la0 = fma(ec[S0 + NLZ], al0, w00), la1 = fma(ec[S1 + NLZ], al1, w01);
    const double a1 = ec[CA0], b1 = ec[CB0], c1 = ec[CC0], a2 = ec[CA1], b2 = ec[CB1], c2 = ec[CC1];
    const double d1 = 2.0 * fma(al0, ec[S0 + AX], -la0 * ec[S0 + LAX]);
    const double e1 = 2.0 * fma(al0, ec[S0 + AY], -la0 * ec[S0 + LAY]);
    const double f1 = (al0 - la0) * (al0 + la0);
    const double db = 2.0 * fma(al1, ec[S1 + AX], -la1 * ec[S1 + LAX]);
    const double eb = 2.0 * fma(al1, ec[S1 + AY], -la1 * ec[S1 + LAY]);
    const double fb = (al1 - la1) * (al1 + la1);
    // antitop conic moved from (Sx - x, Sy - y) to (x, y)
    const double d2 = -fma(2.0 * a2, Sx, fma(b2, Sy, db));
    const double e2 = -fma(2.0 * c2, Sy, fma(b2, Sx, eb));
    const double f2 = fma(fma(a2, Sx, fma(b2, Sy, db)), Sx, fma(fma(c2, Sy, eb), Sy, fb));
    // ---- resultant in y: quartic R(x) = U(x)^2 - V(x) W(x), y = -U/V
    const double U1 = fma(c1, d2, -c2 * d1), U0 = fma(c1, f2, -c2 * f1);
    const double V0 = fma(c1, e2, -c2 * e1);
    const double W2 = (fma(b1, d2, e1 * a2) - fma(b2, d1, e2 * a1));
    const double W1 = (fma(b1, f2, e1 * d2) - fma(b2, f1, e2 * d1));
    const double W0 = fma(e1, f2, -e2 * f1);
    const double uu2 = ec[U2], vv1 = ec[V1], ir4 = ec[IR4];
    const double R3 = fma(2.0 * uu2, U1, -fma(vv1, W2, V0 * ec[W3]));
    const double R2 = fma(U1, U1, fma(2.0 * uu2, U0, -fma(vv1, W1, V0 * W2)));
    const double R1 = fma(2.0 * U1, U0, -fma(vv1, W0, V0 * W1));
    const double R0 = fma(U0, U0, -V0 * W0);
    double xr[4];
    const int nr = quartic_real_roots(R3 * ir4, R2 * ir4, R1 * ir4, R0 * ir4, xr);
    if (nr == 0) return 0.0;
    if (mode == kModeClassify) return (double)(nr >> 1);
    // ---- solution-independent pieces
    // (the visible momenta of the two tops are rebuilt from E_b, E_bbar inside the solution loop: eight values fewer to
    // keep live across it)
    double sum = 0.0;
    // one copy of the per-solution code (the roots stay in registers: selected, not indexed)
#pragma unroll 1
    for (int k = 0; k < nr; ++k) {
      double x = (k == 0) ? xr[0] : (k == 1) ? xr[1] : (k == 2) ? xr[2] : xr[3];
      const double V = fma(vv1, x, V0);
      if (!(V != 0.0)) continue;
      double y = -fma(fma(uu2, x, U1), x, U0) * rcp_fast(V);
      double nz, nbz, xb, yb;
      // one Newton step on g1 = |nu| - E_nu(x, y), g2 = |nubar| - E_nubar(Sx - x, Sy - y); returns |dx| + |dy|
      auto newton = [&]() {
        nz = fma(ec[S0 + AX], x, fma(ec[S0 + AY], y, al0));
        xb = Sx - x; yb = Sy - y;
        nbz = fma(ec[S1 + AX], xb, fma(ec[S1 + AY], yb, al1));
        const double n2 = fma(x, x, fma(y, y, nz * nz)), nb2 = fma(xb, xb, fma(yb, yb, nbz * nbz));
        const double iEn = rsqrt(n2), iEnb = rsqrt(nb2);
        const double g1 = n2 * iEn - fma(ec[S0 + LAX], x, fma(ec[S0 + LAY], y, la0));
        const double g2 = nb2 * iEnb - fma(ec[S1 + LAX], xb, fma(ec[S1 + LAY], yb, la1));
        const double j11 = fma(fma(nz, ec[S0 + AX], x), iEn, -ec[S0 + LAX]);
        const double j12 = fma(fma(nz, ec[S0 + AY], y), iEn, -ec[S0 + LAY]);
        const double j21 = -fma(fma(nbz, ec[S1 + AX], xb), iEnb, -ec[S1 + LAX]);
        const double j22 = -fma(fma(nbz, ec[S1 + AY], yb), iEnb, -ec[S1 + LAY]);
        const double idet = rcp_fast(fma(j11, j22, -j12 * j21));
        const double dxn = fma(g1, j22, -g2 * j12) * idet, dyn = fma(j11, g2, -j21 * g1) * idet;
        x -= dxn; y -= dyn;
        return fabs(dxn) + fabs(dyn);
      };
#pragma unroll 1
      for (int it = 0; it < kNewton; ++it) newton();
      double EnL, EnbL, En, Enb;
      bool good = false;
#pragma unroll 1
      for (int attempt = 0; attempt < 2; ++attempt) {
        nz = fma(ec[S0 + AX], x, fma(ec[S0 + AY], y, al0));
        xb = Sx - x; yb = Sy - y;
        nbz = fma(ec[S1 + AX], xb, fma(ec[S1 + AY], yb, al1));
        EnL = fma(ec[S0 + LAX], x, fma(ec[S0 + LAY], y, la0));
        EnbL = fma(ec[S1 + LAX], xb, fma(ec[S1 + LAY], yb, la1));
        En = sqrt(fma(x, x, fma(y, y, nz * nz))); Enb = sqrt(fma(xb, xb, fma(yb, yb, nbz * nbz)));
        good = fabs(En - EnL) <= 1e-9 * (En + EnL) && fabs(Enb - EnbL) <= 1e-9 * (Enb + EnbL);
        if (good || attempt == 1) break;
        // rare: the Ferrari root was a poor start (the resultant's coefficients lose 6-8 digits to cancellation next
        // to a tangency of the conics); polish until the point stops moving, as the oracle does
#pragma unroll 1
        for (int it = kNewton; it < 12; ++it) {
          const double mv = newton();
          if (!(mv > 0x1p-49 * (fabs(x) + fabs(y)))) break;
        }
      }
      if (!(good && EnL > 0.0 && EnbL > 0.0)) continue;
      // Jacobian: E_nu (A x B)/(4 E_l E_b) = nu x d + E_nu (n_l x n_b), x and y components
      const double px = fma(y, ec[DZ0], fma(-nz, ec[DY0], En * ec[S0 + MX]));
      const double py = fma(nz, ec[DX0], fma(-x, ec[DZ0], En * ec[S0 + MY]));
      const double qx = fma(yb, ec[DZ1], fma(-nbz, ec[DY1], Enb * ec[S1 + MX]));
      const double qy = fma(nbz, ec[DX1], fma(-xb, ec[DZ1], Enb * ec[S1 + MY]));
      const double xz = fabs(fma(px, qy, -py * qx));
      // ---- S3: transverse boost O7 of the two tops
      const double tE = ec[S0 + LE] + Eb0 + En, tz = fma(Eb0, ec[J0 + 4], ec[S0 + LZ]) + nz;
      const double aE = ec[S1 + LE] + Eb1 + Enb, az = fma(Eb1, ec[J1 + 4], ec[S1 + LZ]) + nbz;
      const double tx = fma(Eb0, ec[J0 + 2], ec[S0 + LX]) + x, ty = fma(Eb0, ec[J0 + 3], ec[S0 + LY]) + y;
      const double ax = fma(Eb1, ec[J1 + 2], ec[S1 + LX]) + xb, ay = fma(Eb1, ec[J1 + 3], ec[S1 + LY]) + yb;
      const double PE = tE + aE, Pz = tz + az;
      const double iPE = rcp_fast(PE);
      const double bx = (tx + ax) * iPE, by = (ty + ay) * iPE;           // total transverse momentum / P_E
      const double omb = 1.0 - fma(bx, bx, by * by);
      if (!(omb > 0.0)) continue;
      const double gam = rsqrt(omb);
      const double tEb = gam * (tE - fma(bx, tx, by * ty)), aEb = gam * (aE - fma(bx, ax, by * ay));
      const double PEb = tEb + aEb;
      const double x1 = (PEb + Pz) * c.inv_sqrt_s, x2 = (PEb - Pz) * c.inv_sqrt_s;
      if (!(x1 > 0.0 && x1 < 1.0 && x2 > 0.0 && x2 < 1.0)) continue;
      const double shat = x1 * x2 * c.S;
      if (!(4.0 * c.mt2 < shat)) continue;                                     // reading A9
      // ---- S5: production
      const double ish = rcp_fast(shat);
      const double hs = 0.5 * c.sqrt_s * ish;
      const double tau1 = hs * fma(x1, tEb - tz, x2 * (aEb + az));
      const double tau2 = hs * fma(x2, tEb + tz, x1 * (aEb - az));
      const double rho = 4.0 * c.mt2 * ish;
      const double T = tau1 * tau2, iT = rcp_fast(T);
      const double tt = fma(tau1, tau1, tau2 * tau2);
      const double Mgg = fma(iT, 1.0 / 6.0, -0.375) * (tt + rho - 0.25 * rho * rho * iT);
      const double Mqq = tt + 0.5 * rho;
      const TtLumi<double> lum = tt_lumi<GRIDPDF>(c, x1, x2);
      const double ws = fma(lum.gg, Mgg, lum.qq * Mqq) * ish * rcp_fast(xz);  // flavour sum incl. the PDFs
      if (isfinite(ws)) sum += ws;
    }
    const double w = pre * sum;
    return isfinite(w) ? w : 0.0;
  }
};

}  // namespace memb200
