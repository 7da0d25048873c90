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

// =========================================================================================
// config 1: u dbar -> W+ -> e+ nu, D = 1.  rec = [lep_pT, lep_eta, lep_phi, met_x, met_y]
// DESIGN.md "Config 1" (reading A5): nu_z in [-P, P] charted by s_W with a Breit-Wigner map,
// both roots summed.
// =========================================================================================
struct ProcWenu {
  static constexpr int D = 1, NF = 5, NC = 16;
  enum { LM, LP, LE, LZ, PT, NT2, A, CLO, CHI, DT, SCLO, DSM, PTNT, IPT2, C0, _N };

  __device__ static void prepare(const DevConst& c, const double* ev, int64_t n, int64_t e, double* ec) {
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
    ec[CLO] = c_lo; ec[CHI] = c_hi; ec[DT] = dt; ec[SCLO] = sin(c_lo);   // sin(c_lo) = cos(t_lo)
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

  __device__ static double weight(const DevConst& c, const double* ec, const double (&u)[D]) {
    // pi/2 - t = c_lo (1 - u) + c_hi u: positive terms only (1 - u is exact)
    const double cc_t = fma(ec[CLO], 1.0 - u[0], ec[CHI] * u[0]);
    double sc, cs;
    sincos(cc_t, &sc, &cs);
    const double smm = c.mWGW * (cs / sc);            // m Gam tan t = m Gam cot(pi/2 - t)
    const double sW = c.mW2 + smm;
    // s_W - s_min = m Gam (tan t - tan t_lo) = m Gam sin(dt u) / (cos t cos t_lo): no cancellation
    // at the transverse-mass edge
    const double ds = c.mWGW * sin(ec[DT] * u[0]) / (sc * ec[SCLO]);
    const double half = 0.5 * (ds + ec[DSM]);
    const double cc = 0.5 * sW + ec[A];
    const double disc = half * (cc + ec[PTNT]);
    if (!(disc > 0.0)) return 0.0;
    const double rt = sqrt(disc);
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
      sum += pdf_pair(c, x1, x2) / (x1 * x2) * (a1 * a1 + a2 * a2);
    }
    const double w = ec[C0] * sum / rt;
    return isfinite(w) ? w : 0.0;
  }
};

// =========================================================================================
// jets shared by configs 2-4 (O5): E = E_jet (rlo + dr u); direction fixed by the record.
// per-event block of 5 constants per jet: E_jet rlo, E_jet dr, n_x, n_y, n_z
// =========================================================================================
struct Jet { double E, x, y, z; };

__device__ inline void jet_prepare(const DevConst& c, double Ej, double eta, double phi, double* o) {
  const double st = 1.0 / cosh(eta);
  o[0] = Ej * c.rlo; o[1] = Ej * c.dr;
  o[2] = st * cos(phi); o[3] = st * sin(phi); o[4] = tanh(eta);
}

// returns the parton momentum; tf accumulates E * T(E_jet; E)
__device__ __forceinline__ Jet jet_point(const DevConst& c, const double* o, double u, double& tf) {
  const double x = fma(c.dr, u, c.rlo);
  tf *= tf_times_E(c, rcp_fast(x));
  Jet j;
  j.E = fma(o[1], u, o[0]);
  j.x = j.E * o[2]; j.y = j.E * o[3]; j.z = j.E * o[4];
  return j;
}

// =========================================================================================
// config 2: q qbar -> Z -> b bbar, D = 2.  rec = [E1, eta1, phi1, E2, eta2, phi2]
// DESIGN.md "Config 2"; transverse boost O7 (reading A6)
// =========================================================================================
struct ProcZbb {
  static constexpr int D = 2, NF = 6, NC = 12;
  enum { J0 = 0, J1 = 5, C0 = 10, KT = 11 };

  __device__ static void prepare(const DevConst& c, const double* ev, int64_t n, int64_t e, double* ec) {
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

  __device__ static double weight(const DevConst& c, const double* ec, const double (&u)[D]) {
    double tf = 1.0;
    const Jet p1 = jet_point(c, ec + J0, u[0], tf), p2 = jet_point(c, ec + J1, u[1], tf);
    // O7 without the cancellation in 1 - beta^2 (nearly collinear jets): with P = p1 + p2,
    //   P_E'^2 = P_E^2 - P_T^2 = p1z^2 + p2z^2 + 2 E1 E2 (1 - n1T.n2T)
    //   E_i'   = gamma (E_i - beta.p_iT) = (p_iz^2 + E1 E2 (1 - n1T.n2T)) / P_E'
    //   s-hat  = 2 E1 E2 (1 - n1.n2) = (P_E' + P_z)(P_E' - P_z)
    const double e12 = p1.E * p2.E, ekt = e12 * ec[KT];
    const double Pz = p1.z + p2.z;
    const double PEb = sqrt(fma(p1.z, p1.z, fma(p2.z, p2.z, 2.0 * ekt)));
    const double iPEb = rcp_fast(PEb);
    const double E1 = fma(p1.z, p1.z, ekt) * iPEb, E2 = fma(p2.z, p2.z, ekt) * iPEb;
    const double shat = 2.0 * e12 * ec[J0 + 3];
    const double Xb = PEb + fabs(Pz), Xs = shat / Xb;
    const double x1 = (Pz >= 0.0 ? Xb : Xs) * c.inv_sqrt_s, x2 = (Pz >= 0.0 ? Xs : Xb) * c.inv_sqrt_s;
    if (!(x1 > 0.0 && x1 < 1.0 && x2 > 0.0 && x2 < 1.0)) return 0.0;
    // u = -2 qa.p2', t = -2 qa.p1' for qa = q1 and qa = q2 (both beam orderings), in units of -2h
    const double u1 = x1 * (E2 - p2.z), t1 = x1 * (E1 - p1.z);
    const double u2 = x2 * (E2 + p2.z), t2 = x2 * (E1 + p1.z);
    const double me = c.z_cu * (u1 * u1 + u2 * u2) + c.z_ct * (t1 * t1 + t2 * t2);
    const double dz = shat - c.mZ2;
    const double w = ec[C0] * tf * pdf_pair(c, x1, x2) * me / (shat * (dz * dz + c.mZGZ2));
    return isfinite(w) ? w : 0.0;
  }
};

// =========================================================================================
// config 3: t tbar -> b l nu  bbar q qbar', D = 6 (also the config-5 integrand).
// rec = [lep_pT, lep_eta, lep_phi, (E, eta, phi) x {b_had, b_lep, q, qbar'}, met, met_phi]
// DESIGN.md "Config 3" (reading A7): u0..u3 jet energies, u4 eta_nu flat in [-H, H],
// u5 leptonic s_W through the Breit-Wigner map; nu azimuth = MET azimuth.
// =========================================================================================
struct ProcTTljets {
  static constexpr int D = 6, NF = 17, NC = 44;
  enum { LE, LX, LY, LZ, ELI, EL, LPT2, OMC, CPN, SPN,   // lepton, neutrino azimuth
         J0 = 10, J1 = 15, J2 = 20, J3 = 25,            // b_had, b_lep, q, qbar'
         KBL = 30,                                      // b_lep . l / E_b
         K02, K23, K03,                                 // 1 - n.n of (b_had,q), (q,qbar'), (b_had,qbar')
         NA, NB, NC_,                                   // b_lep . nu = E_b nuT (NA e^eta + NB e^-eta - NC_)
         C0, SW0, _N };

  __device__ static void prepare(const DevConst& c, const double* ev, int64_t n, int64_t e, double* ec) {
    const double lpT = ev[0 * n + e], leta = ev[1 * n + e], lphi = ev[2 * n + e];
    const double mphi = ev[16 * n + e];
    const double lE = lpT * cosh(leta);
    ec[LE] = lE; ec[LX] = lpT * cos(lphi); ec[LY] = lpT * sin(lphi); ec[LZ] = lpT * sinh(leta);
    ec[EL] = exp(leta); ec[ELI] = exp(-leta);
    ec[LPT2] = 2.0 * lpT;
    const double sd = sin(0.5 * (lphi - mphi));
    ec[OMC] = 2.0 * sd * sd;            // 1 - cos(phi_l - phi_nu)
    ec[CPN] = cos(mphi); ec[SPN] = sin(mphi);
    double vol = 1.0, sth = 1.0, eta_j[4], phi_j[4];
    for (int j = 0; j < 4; ++j) {
      const double Ej = ev[(3 + 3 * j) * n + e];
      eta_j[j] = ev[(4 + 3 * j) * n + e]; phi_j[j] = ev[(5 + 3 * j) * n + e];
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

  __device__ static double weight(const DevConst& c, const double* ec, const double (&u)[D]) {
    // ---- S2: jets and their transfer functions
    double tf = 1.0;
    const Jet bh = jet_point(c, ec + J0, u[0], tf), bl = jet_point(c, ec + J1, u[1], tf);
    const Jet q = jet_point(c, ec + J2, u[2], tf), qb = jet_point(c, ec + J3, u[3], tf);
    // ---- S2: neutrino.  g = e^(eta_nu - eta_l); cosh(d eta) - cos(d phi) = (g-1)^2/(2g) + (1 - cos d phi)
    const double H = c.nu_eta_max;
    const double eta_nu = fma(2.0 * H, u[4], -H);
    const double en = exp(eta_nu), eni = rcp_fast(en);
    const double g = en * ec[ELI], gi = eni * ec[EL];
    const double gm1 = g - 1.0;
    const double den = ec[LPT2] * fma(0.5 * gm1 * gm1, gi, ec[OMC]);
    if (!(den > 0.0)) return 0.0;
    const double t = fma(c.tW_dt, u[5], c.tW_lo);
    const double smm = c.mWGW * tan(t);
    const double sW = c.mW2 + smm;
    const double iden = rcp_fast(den);
    const double nuT = sW * iden;
    const double chn = 0.5 * (en + eni), shn = 0.5 * (en - eni);
    const double nE = nuT * chn, nx = nuT * ec[CPN], ny = nuT * ec[SPN], nz = nuT * shn;
    // ---- S3: invariants through per-event angular constants
    const double bl_nu = bl.E * nuT * (fma(ec[NA], en, ec[NB] * eni) - ec[NC_]);
    const double bl_l = bl.E * ec[KBL];
    const double st_m = fma(2.0, bl_l + bl_nu, smm + (c.mW2 - c.mt2));           // s_t - m_t^2
    const double bh_q = bh.E * q.E * ec[K02], q_qb = q.E * qb.E * ec[K23], bh_qb = bh.E * qb.E * ec[K03];
    const double swh_m = fma(2.0, q_qb, -c.mW2);                                 // s_Whad - m_W^2
    const double stb_m = fma(2.0, bh_q + q_qb + bh_qb, -c.mt2);                  // s_tbar - m_t^2
    // ---- S3: top momenta, transverse boost O7 (only the two boosted energies are needed)
    const double tE = bl.E + ec[LE] + nE, tx = bl.x + ec[LX] + nx, ty = bl.y + ec[LY] + ny, tz = bl.z + ec[LZ] + nz;
    const double aE = bh.E + q.E + qb.E, ax = bh.x + q.x + qb.x, ay = bh.y + q.y + qb.y, az = bh.z + q.z + qb.z;
    const double PE = tE + aE, Px = tx + ax, Py = ty + ay, Pz = tz + az;
    const double iPE = rcp_fast(PE);
    const double bx = Px * iPE, by = Py * iPE;
    const double omb = 1.0 - (bx * bx + by * by);
    if (!(omb > 0.0)) return 0.0;
    const double gam = rsqrt(omb);
    const double tEb = gam * (tE - bx * tx - by * ty), aEb = gam * (aE - bx * ax - by * ay);
    const double PEb = tEb + aEb;
    const double x1 = (PEb + Pz) * c.inv_sqrt_s, x2 = (PEb - Pz) * c.inv_sqrt_s;
    if (!(x1 > 0.0 && x1 < 1.0 && x2 > 0.0 && x2 < 1.0)) return 0.0;
    const double xx = x1 * x2, shat = xx * c.S;
    if (!(4.0 * c.mt2 < shat)) return 0.0;                                       // reading A9
    // ---- S5: production.  tau1 = (q1.pt + q2.ptb)/s-hat, tau2 = (q2.pt + q1.ptb)/s-hat
    const double ish = rcp_fast(shat);
    const double hs = 0.5 * c.sqrt_s * ish;
    const double tau1 = hs * fma(x1, tEb - tz, x2 * (aEb + az));
    const double tau2 = hs * fma(x2, tEb + tz, x1 * (aEb - az));
    const double rho = 4.0 * c.mt2 * ish;
    const double T = tau1 * tau2, iT = rcp_fast(T);
    const double tt = fma(tau1, tau1, tau2 * tau2);
    const double Mgg = fma(iT, 1.0 / 6.0, -0.375) * (tt + rho - 0.25 * rho * rho * iT);
    const double Mqq = tt + 0.5 * rho;
    const double prod = fma(c.A_g2, Mgg, (2.0 * c.n_flav * (4.0 / 9.0)) * c.A_q2 * Mqq);
    // ---- S5: propagators and decays
    const double dens = fma(st_m, st_m, c.mtGt2) * fma(stb_m, stb_m, c.mtGt2) * fma(swh_m, swh_m, c.mWGW2);
    const double t_l = fma(0.5, sW, bl_l);                                       // p_t . l
    const double a_q = bh_q + q_qb;                                              // p_tbar . q
    const double dec = t_l * bl_nu * a_q * bh_qb;
    // ---- S4, S7
    const double w = ec[C0] * tf * (nuT * iden) * (pdf_pair(c, x1, x2) * ish) * prod * dec * rcp_fast(dens);
    return isfinite(w) ? w : 0.0;
  }
};

}  // namespace memb200
