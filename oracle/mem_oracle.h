/* oracle/mem_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU oracle for the per-event Monte Carlo
 * estimate of the matrix-element-method likelihood of arXiv 1407.7595
 * (PAPER.md:45 Eq. 1, :49 Eq. 2, :56 Eq. 3, :76-81 Eq. 5-6, :103-118 Eq. 7-8).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may use it.  It shares no code, header, table or
 * constant with the CUDA path under paper_1407_7595_b200/csrc/ (its parameter
 * struct below is its own, deliberately laid out differently from mem_params).
 *
 * All momenta are (E, px, py, pz), natural units, GeV, metric (+,-,-,-).
 */
#ifndef MEM_ORACLE_H
#define MEM_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_W_ENU = 1, ORC_Z_BB = 2, ORC_TT_LJETS = 3, ORC_TT_DILEP = 4, ORC_TTH_DILEP = 5 };

/* DESIGN.md "Readings" O8/A13: the paper gives no constants; BASELINE.json
 * configs give sqrt_s, m_W, Gam_W, m_t, Gam_t, the toy PDF and the TF numbers. */
typedef struct orc_params {
  /* physics constants */
  double sqrt_s, G_F, alpha_s, sin2_thw;
  double m_W, Gam_W, m_Z, Gam_Z, m_t, Gam_t;
  double V_ud, V_tb;
  /* toy PDF f(x) = A x^pow_x (1-x)^pow_1mx (BASELINE.json:configs[0]) */
  double pdf_A_q, pdf_A_g, pdf_pow_x, pdf_pow_1mx;
  /* double-Gaussian jet TF, as fractions of the parton energy (configs[1]) */
  double tf_w_tail, tf_mu1, tf_sig1, tf_mu2, tf_sig2;
  /* integration windows */
  double jetE_rlo, jetE_rhi, bw_nwidths, nu_pz_max, nu_eta_max, met_sigma, met_nsigma;
  /* VEGAS (configs[4]) */
  double vegas_alpha;
  int64_t vegas_points;
  int32_t vegas_iters, vegas_bins;
  int32_t n_flav;
  /* NEXT-1, Eq. 7 "sum over all permutations of assigning measured jets to partons":
   * 0 or 1 = the record order only; ORC_TT_LJETS: 4 = b-tags known (the two b jets swapped x the two
   * light jets swapped), 24 = all assignments; ORC_TT_DILEP: 2 = both b assignments. */
  int32_t n_perm;
  /* NEXT-3, grid PDFs (PAPER.md:141, :274-306 Fig. A.5): pdf_mode != 0 replaces the toy PDF by bilinear
   * interpolation of pdf_data[species][iq][ix] (species 0 = g, 1..5 = d,u,s,c,b; NQ x NX samples on a
   * uniform grid in ln x, ln Q) at the fixed scale pdf_Q.  t tbar processes only. */
  int32_t pdf_mode, pdf_nx, pdf_nq, pdf_pad;
  double pdf_lxmin, pdf_lxmax, pdf_lqmin, pdf_lqmax, pdf_Q;
  const double* pdf_data;
  /* NEXT-4, t tbar H(-> b bbar) dilepton (PAPER.md:101-137 Eq. 7-9, :178-180 Eq. 11; readings A18-A21):
   * Higgs mass and width (Breit-Wigner map of Eq. 9's m_H^2), Yukawa couplings of the factorised matrix element,
   * tth_hyp 0 = t tbar H signal, 1 = non-resonant t tbar b bbar stand-in (the second hypothesis of Eq. 10);
   * tth_chart (oracle only) 0 = Eq. 9 chart (f, m_H^2), 1 = flat (E1, E2) chart for the chart-independence pin.
   * ORC_TTH_DILEP: n_perm 12 = all 4!/2 distinct assignments of four b jets to (b, bbar, {b1, b2}). */
  double m_H, Gam_H, yuk_t, yuk_b;
  int32_t tth_hyp, tth_chart;
} orc_params;

int  orc_params_default(int process, orc_params* p);
int  orc_n_fields(int process);   /* 5 / 6 / 17 / 14 / 18 */
int  orc_n_dims(int process);     /* 1 / 2 / 6 / 8 / 8 */

/* --- random numbers (O2) --- */
void   orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_u52(uint32_t a, uint32_t b);
void   orc_uniforms(uint64_t seed, uint64_t event, uint64_t point, uint32_t iteration,
                    int n_dims, double* u);

/* --- building blocks, exposed so that the tests can pin each one --- */
double orc_pdf_shape(const orc_params* p, double x);
double orc_tf_jet(const orc_params* p, double E_jet, double E_parton);
double orc_pdf_grid(const orc_params* p, int species, double x, double Q);   /* NEXT-3 */
/* Breit-Wigner map: t-window of [s_lo, s_hi]; at t: s - m^2, ds/dt, D(s). */
void   orc_bw_window(double m, double Gam, double s_lo, double s_hi, double* t_lo, double* t_hi);
void   orc_bw_point(double m, double Gam, double t, double* s_minus_m2, double* dsdt, double* D);
/* spin/colour averaged (initial), summed (final) LO matrix elements */
double orc_me_w(const orc_params* p, const double qa[4], const double qb[4],
                const double lep[4], const double nu[4]);           /* u(qa) dbar(qb) -> e+ nu */
double orc_me_z(const orc_params* p, int up_type, const double qa[4], const double qb[4],
                const double p1[4], const double p2[4]);            /* q(qa) qbar(qb) -> b(p1) bbar(p2) */
double orc_me_tt_qq(const orc_params* p, const double q1[4], const double q2[4],
                    const double pt[4], const double ptb[4]);
double orc_me_tt_gg(const orc_params* p, const double q1[4], const double q2[4],
                    const double pt[4], const double ptb[4]);
/* sum over ALL spins of |M(t -> b f fbar')|^2, colour factor n_c (1 leptonic, 3 hadronic) */
double orc_me_top_decay(const orc_params* p, double n_c, const double pt[4], const double pb[4],
                        const double pf_down[4], const double pf_up[4]);
void   orc_boost_transverse(const double P[4], int n, double* mom /* n x 4, in place */);

/* config 4: real roots of q[0] + q[1] x + ... + q[4] x^4 (Ferrari); all
 * solutions of the dilepton system PAPER.md:113-118 Eq. 8, sol[k] = {nu(E,x,y,z), nubar(E,x,y,z)},
 * jac[k] = |d(nu,nubar)/d(s_W+, s_t, s_W-, s_tbar, S_x, S_y)|.  Both return the count. */
int    orc_quartic_real_roots(const double q[5], double x[4]);
int    orc_dilep_solve(const double lp[4], const double b[4], const double lm[4], const double bb[4],
                       double sWp, double st, double sWm, double stb, double Sx, double Sy,
                       double* sol, double* jac);

/* NEXT-4 building blocks.  Eq. 9 inverted for massless b quarks: both orderings
 * (E1[r], E2[r]) with E1 + E2 = f, 2 E1 E2 K12 = sH, *jac = |d(E1,E2)/d(f,sH)|; returns 0 or 2.
 * Factorised matrix-element pieces (reading A20): radiation factor of k = p_b1 + p_b2 off the top pair and
 * the decay factor of the radiated system, both for p->tth_hyp; normalised (tau1, tau2, rho) of the t tbar
 * subsystem (returns 0 when rho >= 1); the production MEs as functions of (tau1, tau2, rho); the flavour sum
 * incl. the PDFs. */
int    orc_eq9_roots(double K12, double f, double sH, double E1[2], double E2[2], double* jac);
double orc_tth_radiator(const orc_params* p, const double pt[4], const double ptb[4], const double k[4]);
double orc_tth_decay(const orc_params* p, double sH);
int    orc_tth_tt_invariants(const orc_params* p, const double q1[4], const double q2[4], const double pt[4],
                             const double ptb[4], double* t1, double* t2, double* rho);
double orc_me_tt_gg_inv(const orc_params* p, double t1, double t2, double rho);
double orc_me_tt_qq_inv(const orc_params* p, double t1, double t2, double rho);
double orc_tt_flavour_sum(const orc_params* p, double x1, double x2, double me_gg, double me_qq);
double orc_me_top_decay_D(const orc_params* p, double n_c, const double pt[4], const double pb[4],
                          const double pf_down[4], const double pf_up[4], double D_W);
/* 1/sigma and the discriminant (Eq. 10; reading A22) */
double orc_normalisation(const double* p, const double* g, int64_t n);
void   orc_discriminant(const double* p_sig, const double* p_bkg, int64_t n, double sigma_sig, double sigma_bkg,
                        double* out_D);

/* --- the integrand: one event record (n_fields doubles), one unit-cube point --- */
/* dbg (may be NULL): [0]=n_sol, [1..]= per solution: x1, x2, then the boosted final momenta
 * (2 / 6 / 8 four-vectors; room for 8 solutions of 8 particles: 273 doubles). */
double orc_weight(int process, const orc_params* p, const double* rec, const double* u, double* dbg);
/* Extended-precision referee: the same templates instantiated in long double (x87, 64-bit
 * mantissa), result rounded to double.  Used by the tests to adjudicate ill-conditioned points. */
double orc_weight_x(int process, const orc_params* p, const double* rec, const double* u);

/* events: SoA, field-major [n_fields][n_events].  grid (may be NULL) = VEGAS edges
 * [n_events][D][bins+1]; then u is warped through it first. */
int orc_eval_points(int process, const orc_params* p, const double* events, int64_t n_events,
                    int64_t event, uint64_t event_offset, int64_t first_point, int64_t n,
                    uint64_t seed, int32_t iteration, const double* grid, double* out_w);
int orc_eval_points_x(int process, const orc_params* p, const double* events, int64_t n_events,
                      int64_t event, uint64_t event_offset, int64_t first_point, int64_t n,
                      uint64_t seed, int32_t iteration, const double* grid, double* out_w);
int orc_integrate(int process, const orc_params* p, const double* events, int64_t n_events,
                  uint64_t event_offset, int64_t n_points, uint64_t seed,
                  double* out_p, double* out_err);

/* --- NEXT-2, parton-level mode (Table 2): delta transfer functions, no integration.
 * mom: SoA field-major [24][n_events] = (E,px,py,pz) of l, nu, b_had, b_lep, q, qbar'.
 * out_w[e] = sum over the n_perm jet assignments of f f / (|q1||q2|) |M|^2.  extended != 0: the
 * long-double referee. */
int orc_parton_weights(int process, const orc_params* p, const double* mom, int64_t n_events, int extended,
                       double* out_w);

/* --- VEGAS (DESIGN.md config 5, reading A14) --- */
void orc_vegas_map(const double* edges /* [D][bins+1] */, int bins, int n_dims, const double* u,
                   double* z, int* k, double* jac);
void orc_vegas_refine(const double* hist /* [bins] */, double* edges /* [bins+1], in place */,
                      int bins, double alpha);
/* runs p->vegas_iters adaptation passes of p->vegas_points, then a final pass of n_points;
 * grid_out (may be NULL): final edges [n_events][D][bins+1]. */
int orc_vegas_integrate(int process, const orc_params* p, const double* events, int64_t n_events,
                        uint64_t event_offset, int64_t n_points, uint64_t seed,
                        double* out_p, double* out_err, double* grid_out);

#ifdef __cplusplus
}
#endif
#endif
