// mem_tth.cuh -- NEXT-4: t tbar H(-> b bbar), dileptonic top decays, four b jets, D = 8: the paper's own
// benchmark integral (Eq. 7), with the neutrino momenta traded for the W and top
// propagator invariants (Eq. 8), the Higgs b-quark energies (E1, E2) traded for
// (f = E1 + E2, m_H^2) (Eq. 9) and the missing transverse momentum of Eq. 8 defined
// point by point as minus the visible transverse momentum (Eq. 11).
// readings A18-A22.  Also the post-processing the paper does with the result: 1/sigma (PAPER.md:45
// Eq. 1) and the discriminant D = log10(p_ttH / p_ttbb) (Eq. 10).
//
// rec = [(pT, eta, phi) l+, (pT, eta, phi) l-, (E, eta, phi) x {b, bbar, b1, b2}]   (18 fields)
// u0, u1 -> E_b, E_bbar (O5);  u2..u5 -> s_W+, s_t, s_W-, s_tbar (O6);  u6 -> k^2 = (p_b1 + p_b2)^2
// (hypothesis 0: Breit-Wigner map of the Higgs; hypothesis 1: flat in ln k^2 over what the energy
// windows allow);  u7 -> f flat over the sum of the two energy windows.  Both orderings of Eq. 9's
// inverse are summed, each only inside both parton-energy windows.
//
// The dilepton system is the one of config 4 (mem_processes.cuh: ProcTTdilep) and its per-event
// constants are laid out the same way; the total neutrino transverse momentum now moves with the
// point (Eq. 11), there is no MET transfer function, and with P_T = 0 there is no boost.
#pragma once
#include "mem_processes.cuh"

namespace memb200 {

// the k-th of the 4!/2 = 12 distinct assignments of four b jets to the roles (b, bbar, {b1, b2}):
// ordered choices of (b, bbar) in lexicographic order, the remaining two jets ascending
__device__ inline void tth_assignment(int n_perm, int k, int (&sig)[4]) {
  sig[0] = 0; sig[1] = 1; sig[2] = 2; sig[3] = 3;
  if (n_perm != 12) return;
  const int a = k / 3;
  int b = k - 3 * a;
  if (b >= a) ++b;
  sig[0] = a; sig[1] = b;
  int m = 2;
  for (int j = 0; j < 4; ++j)
    if (j != a && j != b) sig[m++] = j;
}

struct ProcTTHdilep {
  using real = double;
  static constexpr bool kCompact = true;    // staged lane compaction in the plain integrate kernel
  static constexpr bool kSplitC0 = false;
  static constexpr int D = 8, NF = 18, NC = 80;
  static constexpr int kNewton = 3;
  // stages of the lane-compacting loop (mem_kernels.cuh).  Classes by the real roots (nr0, nr1) of the two orderings'
  // quartics, so that a batch has one trip count: 1 = one ordering with 2 roots, 2 = one with 4, 3 = (2,2), 4 = (2,4),
  // 5 = (4,2), 6 = (4,4)
  static constexpr int kModeFull = 0, kModeClassify = 1, kModeCheap = 2;
  static constexpr int kClasses = 6;
  // one cheap-test stage before the classification: Eq. 9 has a root inside both energy windows for at least one
  // ordering.  It needs u6, u7 only (Philox word block 3) and 39 % of the points of the closure records pass; the
  // b.nu > 0 test (70 % of those pass) stays in the classification stage, which computes the four tangents it needs anyway.
  // Measured (ms/step, hypothesis 0 / 1, 16384 x 2^18): this 230 / 153; the cheap test on the full prelude 224 / 178; two
  // cheap stages 245 / 165 -- every extra queue ends each chunk with one more partial batch.
  static constexpr int kPreStages = 1;
  static constexpr int kCheapBlock = 3;
  // first 56 constants: the layout of ProcTTdilep (two top sides, conics, resultant, jets b and bbar)
  enum { LE, LX, LY, LZ, I2EL, ELK, IDZ, NLZ, AX, AY, LAX, LAY, MX, MY, SIDE = 14,
         S0 = 0, S1 = 14,
         DX0 = 28, DY0, DZ0, DX1, DY1, DZ1,
         CA0 = 34, CB0, CC0, CA1, CB1, CC1,
         U2 = 40, V1, W3, IR4,
         J0 = 44, J1 = 49,                                  // b, bbar: E rlo, E dr, n_x, n_y, n_z
         IEJ0 = 54, IEJ1,
         J2 = 56, J3 = 61,                                  // b1, b2: E_jet rlo, E_jet rhi, n_x, n_y, n_z
         IEJ2 = 66, IEJ3,                                   // 1 / E_jet
         K2I,                                               // 2 / K12, K12 = 1 - n_b1.n_b2
         FLO, FDR,                                          // f = FLO + FDR u7
         SLO,                                               // hypothesis 1: lower edge of the k^2 window
         C0, PTX, PTY, VISE, _N };

  __device__ static void prepare(const DevConst& c, const double* ev, int64_t n, int64_t e, int k, double* ec) {
    for (int j = 0; j < NC; ++j) ec[j] = 0.0;
    int sig[4];
    tth_assignment(c.n_perm, k, sig);
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
    ec[PTX] = ptx; ec[PTY] = pty; ec[VISE] = lE[0] + lE[1];
    const double a1 = ec[CA0], b1 = ec[CB0], c1 = ec[CC0], a2 = ec[CA1], b2 = ec[CB1], c2 = ec[CC1];
    ec[U2] = c1 * a2 - c2 * a1; ec[V1] = c1 * b2 - c2 * b1; ec[W3] = b1 * a2 - b2 * a1;
    ec[IR4] = 1.0 / (ec[U2] * ec[U2] - ec[V1] * ec[W3]);
    // Higgs candidates
    double Eh[2], etah[2], phih[2];
    for (int j = 0; j < 2; ++j) {
      Eh[j] = ev[(6 + 3 * sig[2 + j]) * n + e]; etah[j] = ev[(7 + 3 * sig[2 + j]) * n + e]; phih[j] = ev[(8 + 3 * sig[2 + j]) * n + e];
      double* o = ec + J2 + 5 * j;
      const double st = 1.0 / cosh(etah[j]);
      o[0] = Eh[j] * c.rlo; o[1] = Eh[j] * c.rhi;
      o[2] = st * cos(phih[j]); o[3] = st * sin(phih[j]); o[4] = tanh(etah[j]);
      ec[IEJ2 + j] = 1.0 / Eh[j];
      sth *= st / (2.0 * kTwoPi3);
    }
    const double K12 = one_minus_cos(etah[0], phih[0], etah[1], phih[1]);
    ec[K2I] = 2.0 / K12;
    ec[FLO] = (Eh[0] + Eh[1]) * c.rlo; ec[FDR] = (Eh[0] + Eh[1]) * c.dr;
    ec[SLO] = 2.0 * K12 * Eh[0] * Eh[1] * c.rlo * c.rlo;
    vol *= (Eh[0] + Eh[1]) * c.dr;
    // vol: jets b, bbar, f; dt_W^2 dt_t^2; the k^2 map and everything constant of the radiated system (c.tth_c);
    // four jets' sin(theta)/(2 (2pi)^3) [their E is inside E T(E_jet; E)]; leptons 1/(2 E_l (2pi)^3); (2pi)^4 (2/S);
    // prod_k ds_k/dt_k D_k = 1/(m_W Gam_W)^2 1/(m_t Gam_t)^2; neutrinos 1/((2pi)^6 4) and
    // J/(E_nu E_nubar) = 1/(16 E_l+ E_l- E_b E_bbar |..|) [1/(E_b E_bbar |..|) stays in the point];
    // flux 4/(x1 x2 S) [1/(x1 x2) stays]; g_s^4; decays (1/2)(4 g^4 V_tb^2) each; Eq. 9: 1/(2 K12) [1/|E1 - E2| stays]
    ec[C0] = vol * c.tW_dt * c.tW_dt * c.tT_dt * c.tT_dt * c.tth_c * sth /
             (2.0 * lE[0] * kTwoPi3) / (2.0 * lE[1] * kTwoPi3) * kTwoPi4 * (2.0 * c.inv_S) /
             (c.mWGW * c.mWGW * c.mtGt * c.mtGt) / (kTwoPi3 * kTwoPi3 * 4.0) / (16.0 * lE[0] * lE[1]) * (4.0 * c.inv_S) *
             c.gs4 * (2.0 * c.g4w * c.V_tb2) * (2.0 * c.g4w * c.V_tb2) / (2.0 * K12);
  }

  __device__ static double cheap_test(const DevConst& c, const double* ec, double u6, double u7) {
    const double sH = c.tth_hyp ? ec[SLO] * exp_tab(c.lnr * u6) : fma(c.mHGH, tan_bw(fma(c.tH_dt, u6, c.tH_lo)), c.mH2);
    const double f = fma(ec[FDR], u7, ec[FLO]);
    const double disc = fma(f, f, -sH * ec[K2I]);
    if (!(disc > 0.0)) return 0.0;
    const double rt = sqrt(disc);
    const double Ehi = 0.5 * (f + rt), Elo = 0.5 * (f - rt);
    const bool in0 = Ehi >= ec[J2] && Ehi <= ec[J2 + 1] && Elo >= ec[J3] && Elo <= ec[J3 + 1];
    const bool in1 = Elo >= ec[J2] && Elo <= ec[J2 + 1] && Ehi >= ec[J3] && Ehi <= ec[J3 + 1];
    return (in0 || in1) ? 1.0 : 0.0;
  }

  template <bool PERM, bool GRIDPDF, bool TAB_UNUSED>
  __device__ static double weight_t(const DevConst& c, const double* ec, const double (&u)[D]) {
    if (!PERM) return weight_rt<GRIDPDF, true>(c, ec, u, kModeFull);
    double w = 0.0;
#pragma unroll 1
    for (int k = 0; k < c.n_perm; ++k) w += weight_rt<GRIDPDF, true>(c, ec + k * NC, u, kModeFull);
    return w;
  }

  __device__ static double weight(const DevConst& c, const double* ec, const double (&u)[D]) {
    return weight_rt<false, true>(c, ec, u, kModeFull);
  }

  // mode (a warp-uniform run-time selector, one copy of the code as in config 4): kModeFull the weight (both Eq. 9
  // orderings); kModeCheap 1 if the point passes the cheap tests (b.nu > 0 on both sides, Eq. 9 has a root and at
  // least one ordering lies inside both energy windows); kModeClassify the point's class (0 = no real root).
  template <bool GRIDPDF, bool TAB>
  __device__ static double weight_rt(const DevConst& c, const double* ec, const double (&u)[D], int mode) {
    // ---- S2: jets b, bbar
    const double xb0 = fma(c.dr, u[0], c.rlo), xb1 = fma(c.dr, u[1], c.rlo);
    const double ixb0 = rcp_fast(xb0), ixb1 = rcp_fast(xb1);
    const double Eb0 = fma(ec[J0 + 1], u[0], ec[J0]), Eb1 = fma(ec[J1 + 1], u[1], ec[J1]);
    const double iEb0 = ixb0 * ec[IEJ0], iEb1 = ixb1 * ec[IEJ1];
    // ---- S2: the mapped invariants, s_k - m_k^2 = m Gam tan t_k (O6); the fifth is the Higgs (hypothesis 0)
    const double tk[5] = {fma(c.tW_dt, u[2], c.tW_lo), fma(c.tT_dt, u[3], c.tT_lo), fma(c.tW_dt, u[4], c.tW_lo),
                          fma(c.tT_dt, u[5], c.tT_lo), fma(c.tH_dt, u[6], c.tH_lo)};
    double tn[5];
    tan_bw_n<5>(tk, tn);
    const double smW0 = c.mWGW * tn[0], smT0 = c.mtGt * tn[1], smW1 = c.mWGW * tn[2], smT1 = c.mtGt * tn[3];
    const double sW0 = c.mW2 + smW0, sW1 = c.mW2 + smW1;
    const double dm2 = c.mt2 - c.mW2;
    const double hD0 = fma(0.5 * (dm2 + (smT0 - smW0)), iEb0, -ec[S0 + ELK]);
    const double hD1 = fma(0.5 * (dm2 + (smT1 - smW1)), iEb1, -ec[S1 + ELK]);
    if (!(hD0 > 0.0 && hD1 > 0.0)) return 0.0;
    // ---- Eq. 9: k^2 and f -> the two orderings (E1, E2) = ((f +- rt)/2, (f -+ rt)/2)
    const double sH = c.tth_hyp ? ec[SLO] * exp_tab(c.lnr * u[6]) : fma(c.mHGH, tn[4], c.mH2);
    const double f = fma(ec[FDR], u[7], ec[FLO]);
    const double disc = fma(f, f, -sH * ec[K2I]);
    if (!(disc > 0.0)) return 0.0;
    const double rt = sqrt(disc);
    const double Ehi = 0.5 * (f + rt), Elo = 0.5 * (f - rt);
    // an ordering counts only inside both parton-energy windows: the chart then covers exactly the box of O5
    const bool in0 = Ehi >= ec[J2] && Ehi <= ec[J2 + 1] && Elo >= ec[J3] && Elo <= ec[J3 + 1];     // (E1, E2) = (Ehi, Elo)
    const bool in1 = Elo >= ec[J2] && Elo <= ec[J2 + 1] && Ehi >= ec[J3] && Ehi <= ec[J3 + 1];     // (E1, E2) = (Elo, Ehi)
    if (!(in0 || in1)) return 0.0;
    if (mode == kModeCheap) return 1.0;
    // ---- everything of the point that does not depend on the ordering or the solution, folded into one factor now
    // (the full pass only: its points have real roots), so that a dozen values need not stay live -- or be spilled --
    // across the two loops: S5 decays (p_t.p_l)(p_b.p_nu) per side, S6 transfer functions of b and bbar, 1/(E_b E_bbar)
    // of the Jacobian, Eq. 9's 1/|E1 - E2|, and k^2 of sum |M(H -> b bbar)|^2 (hypothesis 1: (1/k^4) k^2 (dk^2/du ~ k^2) = const)
    double pre = 0.0;
    if (mode == kModeFull) {
      TfAcc<double> tfa{0.0, 1.0};
      tf_accum<TAB>(c, ixb0, tfa);
      tf_accum<TAB>(c, ixb1, tfa);
      const double tf = tfa.fac * (TAB ? exp_tab<true>(-tfa.esum) : exp(-tfa.esum));
      const double dec = fma(Eb0, ec[S0 + ELK], 0.5 * sW0) * (Eb0 * hD0) * fma(Eb1, ec[S1 + ELK], 0.5 * sW1) * (Eb1 * hD1);
      pre = ec[C0] * tf * dec * (iEb0 * iEb1) * (c.tth_hyp ? 1.0 : sH) * rcp_fast(rt);
    }
    // ---- S2: offsets of nu_z and E_nu on each side, conic linear/constant parts (independent of the ordering)
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
    const double uu2 = ec[U2], vv1 = ec[V1], ir4 = ec[IR4];
    // visible momentum without the Higgs candidates
    const double vx0 = ec[PTX] + Eb0 * ec[J0 + 2] + Eb1 * ec[J1 + 2], vy0 = ec[PTY] + Eb0 * ec[J0 + 3] + Eb1 * ec[J1 + 3];
    // (the visible momenta of the two tops are rebuilt from E_b, E_bbar inside the solution loop: eight values fewer to
    // keep live across the loops)
    const double s_t = c.mt2 + smT0, s_tb = c.mt2 + smT1;
    double total = 0.0;
    int nr0 = 0, nr1 = 0;
#pragma unroll 1
    for (int r = 0; r < 2; ++r) {
      if (!(r ? in1 : in0)) continue;
      const double E1 = r ? Elo : Ehi, E2 = r ? Ehi : Elo;
      const double kx = fma(E1, ec[J2 + 2], E2 * ec[J3 + 2]), ky = fma(E1, ec[J2 + 3], E2 * ec[J3 + 3]);
      const double kz = fma(E1, ec[J2 + 4], E2 * ec[J3 + 4]);
      // Eq. 11: the neutrino pair balances the visible system of this point
      const double Sx = -(vx0 + kx), Sy = -(vy0 + ky);
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
      const double R3 = fma(2.0 * uu2, U1, -fma(vv1, W2, V0 * ec[W3]));
      const double R2 = fma(U1, U1, fma(2.0 * uu2, U0, -fma(vv1, W1, V0 * W2)));
      const double R1 = fma(2.0 * U1, U0, -fma(vv1, W0, V0 * W1));
      const double R0 = fma(U0, U0, -V0 * W0);
      double xr[4];
      const int nr = quartic_real_roots(R3 * ir4, R2 * ir4, R1 * ir4, R0 * ir4, xr);
      if (mode == kModeClassify) { if (r) nr1 = nr; else nr0 = nr; continue; }
      if (nr == 0) continue;
      // S6: transfer functions of the two Higgs candidates for this ordering
      TfAcc<double> th{0.0, 1.0};
      tf_accum<TAB>(c, rcp_fast(E1 * ec[IEJ2]), th);
      tf_accum<TAB>(c, rcp_fast(E2 * ec[IEJ3]), th);
      const double tf12 = th.fac * (TAB ? exp_tab<true>(-th.esum) : exp(-th.esum));
      double sum = 0.0;
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
          // rare: the Ferrari root was a poor start (the resultant's coefficients lose 6-8 digits to cancellation
          // next to a tangency of the conics); polish until the point stops moving, as the oracle does
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
        // ---- S3: the two tops; P_T = 0 by Eq. 11, so x1, x2 come straight from P_E, P_z
        const double tE = ec[S0 + LE] + Eb0 + En, tz = fma(Eb0, ec[J0 + 4], ec[S0 + LZ]) + nz;
        const double aE = ec[S1 + LE] + Eb1 + Enb, az = fma(Eb1, ec[J1 + 4], ec[S1 + LZ]) + nbz;
        const double tx = fma(Eb0, ec[J0 + 2], ec[S0 + LX]) + x, ty = fma(Eb0, ec[J0 + 3], ec[S0 + LY]) + y;
        const double ax = fma(Eb1, ec[J1 + 2], ec[S1 + LX]) + xb, ay = fma(Eb1, ec[J1 + 3], ec[S1 + LY]) + yb;
        const double PE = (tE + aE) + f, Pz = (tz + az) + kz;
        const double x1 = (PE + Pz) * c.inv_sqrt_s, x2 = (PE - Pz) * c.inv_sqrt_s;
        if (!(x1 > 0.0 && x1 < 1.0 && x2 > 0.0 && x2 < 1.0)) continue;
        // ---- S5: production next to the radiated system (reading A20): normalised tau, rho from (p_t + p_tbar)^2
        const double ptpb = fma(tE, aE, -fma(tx, ax, fma(ty, ay, tz * az)));
        const double stt = s_t + s_tb + 2.0 * ptpb;
        if (!(4.0 * c.mt2 < stt)) continue;
        const double n1 = fma(x1, tE - tz, x2 * (aE + az)), n2 = fma(x2, tE + tz, x1 * (aE - az));
        const double in12 = rcp_fast(n1 + n2);
        const double tau1 = n1 * in12, tau2 = n2 * in12;
        const double rho = 4.0 * c.mt2 * rcp_fast(stt);
        const double iT = rcp_fast(tau1 * tau2);
        const double tt = fma(tau1, tau1, tau2 * tau2);
        const double Mgg = fma(iT, 1.0 / 6.0, -0.375) * (tt + rho - 0.25 * rho * rho * iT);
        const double Mqq = tt + 0.5 * rho;
        // ---- radiation of k = p_b1 + p_b2 off the top pair
        const double tk_ = fma(tE, f, -fma(tx, kx, fma(ty, ky, tz * kz)));
        const double ak_ = fma(aE, f, -fma(ax, kx, fma(ay, ky, az * kz)));
        double rad;
        if (c.tth_hyp) {
          const double itk = rcp_fast(tk_), iak = rcp_fast(ak_);
          rad = fma(2.0 * ptpb * itk, iak, -fma(s_t * itk, itk, s_tb * iak * iak));
        } else {
          const double Xt = fma(2.0, tk_, sH), Xa = fma(2.0, ak_, sH);
          const double q = (Xt + Xa) * rcp_fast(Xt * Xa);
          rad = q * q;
        }
        const TtLumi<double> lum = tt_lumi<GRIDPDF>(c, x1, x2);
        const double ws = fma(lum.gg, Mgg, lum.qq * Mqq) * rad * rcp_fast(x1 * x2 * xz);
        if (isfinite(ws)) sum += ws;
      }
      total = fma(tf12, sum, total);
    }
    if (mode == kModeClassify) {
      if (nr0 == 0 || nr1 == 0) return (double)((nr0 + nr1) >> 1);        // 0, 1 (two roots) or 2 (four)
      return (double)(3 + (nr0 >> 2) * 2 + (nr1 >> 2));                     // (2,2) 3, (2,4) 4, (4,2) 5, (4,4) 6
    }
    const double w = pre * total;
    return isfinite(w) ? w : 0.0;
  }
};

// ---------------------------------------------------------------------------------------
// Post-processing (PAPER.md:45 Eq. 1 "1/sigma"; :143 Eq. 10; reading A22).
// normalisation_kernel: one block; sigma = (1/n) sum_e p_e / g_e in a fixed order (thread-strided ->
// warp shuffle -> warps), g = the density the events were drawn from.
// discriminant_kernel: D_e = log10((p_sig,e / sigma_sig) / (p_bkg,e / sigma_bkg)).
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) normalisation_kernel(const double* __restrict__ p, const double* __restrict__ g,
                                                                 int64_t n, double* __restrict__ out_sigma) {
  __shared__ double sh[2 * kWarps];
  double s = 0.0, dummy = 0.0;
  for (int64_t e = threadIdx.x; e < n; e += kThreads) s += p[e] / g[e];
  block_sum2(s, dummy, sh);
  if (threadIdx.x == 0) out_sigma[0] = s / (double)n;
}

__global__ void discriminant_kernel(const double* __restrict__ p_sig, const double* __restrict__ p_bkg, int64_t n,
                                    const double* __restrict__ sigma_sig, const double* __restrict__ sigma_bkg,
                                    double* __restrict__ out_D) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n) return;
  out_D[e] = log10((p_sig[e] / sigma_sig[0]) / (p_bkg[e] / sigma_bkg[0]));
}

}  // namespace memb200
