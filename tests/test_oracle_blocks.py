"""Pins of the oracle's building blocks against things other than itself (CPU only).

Philox known-answer vectors; exactness of the 52-bit uniform; Breit-Wigner and
double-Gaussian normalisation (BASELINE.json:north_star); every matrix element against an
explicit Dirac-trace evaluation and/or the textbook closed-form cross-section or width.
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate as si

import oracle
from helpers import (G, PL, PR, lorentz_contract, massless, mdot, random_massless, slash,
                     two_body_decay)

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- O2
def test_philox_known_answer_vectors():
    rows = [l.split() for l in open(os.path.join(GOLD, "philox4x32_10_kat.txt")) if not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert oracle.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_u52_exact_and_open_interval():
    assert oracle.u52(0, 0) == 2.0 ** -53
    assert oracle.u52(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    # bit layout: a supplies the high 26 bits, b the low 26; the low 6 bits of each are dropped
    assert oracle.u52(1 << 6, 0) == (2.0 ** 26 + 0.5) * 2.0 ** -52
    assert oracle.u52(0, 1 << 6) == 1.5 * 2.0 ** -52
    assert oracle.u52(63, 63) == 2.0 ** -53


def test_uniform_counter_layout():
    """counter = (point lo, point hi, event, iteration*256 + j); dims 2j, 2j+1 from words (0,1), (2,3)."""
    seed, ev, pt, it = 0x123456789ABCDEF0, 77, (5 << 32) | 9, 3
    u = oracle.uniforms(seed, ev, pt, it, 6)
    for j in range(3):
        r = oracle.philox4x32_10([9, 5, 77, it * 256 + j], [0x9ABCDEF0, 0x12345678])
        assert u[2 * j] == oracle.u52(r[0], r[1])
        assert u[2 * j + 1] == oracle.u52(r[2], r[3])
    # odd dimension count takes only words (0,1) of the last block
    assert np.array_equal(oracle.uniforms(seed, ev, pt, it, 5), u[:5])


def test_uniform_moments():
    u = np.array([oracle.uniforms(1, 0, i, 0, 2) for i in range(20000)])
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / u.size)
    assert abs((u ** 2).mean() - 1 / 3) < 0.01
    assert abs(np.corrcoef(u[:, 0], u[:, 1])[0, 1]) < 0.03


# ----------------------------------------------------------------------------- O6
@pytest.mark.parametrize("m,gam", [(80.4, 2.09), (173.0, 1.4), (91.1876, 2.4952)])
def test_breit_wigner_map(m, gam):
    s_lo, s_hi = (m - 15 * gam) ** 2, (m + 15 * gam) ** 2
    t_lo, t_hi = oracle.bw_window(m, gam, s_lo, s_hi)
    # int D(s) ds over the window = (t_hi - t_lo)/(m Gam): independent quadrature of the plain Lorentzian
    q, _ = si.quad(lambda s: 1.0 / ((s - m * m) ** 2 + (m * gam) ** 2), s_lo, s_hi,
                   points=[m * m], epsabs=0, epsrel=1e-12, limit=400)
    assert math.isclose(q, (t_hi - t_lo) / (m * gam), rel_tol=1e-10)
    # the mapped estimator of the bare propagator has zero variance: (ds/dt) D = 1/(m Gam);
    # and s(t) hits the window ends
    for t in np.linspace(t_lo, t_hi, 17):
        smm, dsdt, D = oracle.bw_point(m, gam, t)
        assert math.isclose(dsdt * D, 1.0 / (m * gam), rel_tol=1e-14)
        assert math.isclose(D, 1.0 / (smm ** 2 + (m * gam) ** 2), rel_tol=1e-14)
    assert math.isclose(m * m + oracle.bw_point(m, gam, t_lo)[0], s_lo, rel_tol=1e-12)
    assert math.isclose(m * m + oracle.bw_point(m, gam, t_hi)[0], s_hi, rel_tol=1e-12)
    # ds/dt is the derivative of s(t)
    t, h = 0.3, 1e-6
    num = (oracle.bw_point(m, gam, t + h)[0] - oracle.bw_point(m, gam, t - h)[0]) / (2 * h)
    assert math.isclose(num, oracle.bw_point(m, gam, t)[1], rel_tol=1e-8)


# ----------------------------------------------------------------------------- O5
@pytest.mark.parametrize("E", [20.0, 75.0, 400.0])
def test_jet_tf_normalised_and_shaped(E):
    p = oracle.params_default(oracle.Z_BB)
    q, _ = si.quad(lambda ej: oracle.tf_jet(p, ej, E), E * (1 - 3.0), E * (1 + 3.0),
                   points=[E, 0.9 * E], epsabs=0, epsrel=1e-11, limit=400)
    assert math.isclose(q, 1.0, rel_tol=1e-9)          # "double-Gaussian normalisation"
    # mean and variance of the mixture: mean = E(1 + w mu2), core mu = 0
    mean, _ = si.quad(lambda ej: ej * oracle.tf_jet(p, ej, E), -2 * E, 4 * E, points=[E], epsrel=1e-11, limit=400)
    assert math.isclose(mean, E * (1 + 0.3 * (-0.1)), rel_tol=1e-8)
    var, _ = si.quad(lambda ej: (ej - mean) ** 2 * oracle.tf_jet(p, ej, E), -2 * E, 4 * E, points=[E],
                     epsrel=1e-11, limit=400)
    expect = 0.7 * (0.15 ** 2 + 0.03 ** 2) + 0.3 * (0.35 ** 2 + 0.07 ** 2)
    assert math.isclose(var, expect * E * E, rel_tol=1e-7)
    # pure core when the tail weight is zero: value at the peak is 1/(sigma sqrt(2 pi))
    p.tf_w_tail = 0.0
    assert math.isclose(oracle.tf_jet(p, E, E), 1 / (0.15 * E * math.sqrt(2 * math.pi)), rel_tol=1e-14)


def test_pdf_shape():
    p = oracle.params_default(oracle.W_ENU)
    for x in (1e-4, 0.03, 0.5, 0.999):
        assert math.isclose(oracle.pdf_shape(p, x), (1 - x) ** 3 / math.sqrt(x), rel_tol=1e-14)


# ----------------------------------------------------------------------------- matrix elements
def _cm(shat, cth, phi=0.3, m=0.0):
    E = math.sqrt(shat) / 2
    q1, q2 = np.array([E, 0, 0, E]), np.array([E, 0, 0, -E])
    k = math.sqrt(E * E - m * m)
    sth = math.sqrt(1 - cth * cth)
    p1 = np.array([E, k * sth * math.cos(phi), k * sth * math.sin(phi), k * cth])
    p2 = np.array([E, -p1[1], -p1[2], -p1[3]])
    return q1, q2, p1, p2


def _chiral_trace(pa, pb, Pa, Pb):
    """T^{mu nu} = Tr[ pa-slash gamma^mu Pa pb-slash gamma^nu Pb ]"""
    return [[np.trace(slash(pa) @ G[mu] @ Pa @ slash(pb) @ G[nu] @ Pb) for nu in range(4)] for mu in range(4)]


def test_me_w_against_dirac_trace():
    p = oracle.params_default(oracle.W_ENU)
    g2 = 4 * math.sqrt(2) * p.G_F * p.m_W ** 2
    rng = np.random.default_rng(5)
    for _ in range(5):
        shat = (60 + 50 * rng.random()) ** 2
        qa, qb, lep, nu = _cm(shat, 2 * rng.random() - 1, 6.28 * rng.random())
        # M = (g^2/2) V [vbar(qb) g^mu PL u(qa)] [ubar(nu) g_mu PL v(lep)] / (s - m^2 + i m Gam)
        Lq = _chiral_trace(qb, qa, PL, PL)
        Ll = _chiral_trace(nu, lep, PL, PL)
        tr = lorentz_contract(Lq, Ll).real
        D = 1 / ((shat - p.m_W ** 2) ** 2 + (p.m_W * p.Gam_W) ** 2)
        expect = (g2 / 2) ** 2 * tr * D / 12.0          # 1/4 spins, 1/3 colour
        assert math.isclose(oracle.me_w(p, qa, qb, lep, nu), expect, rel_tol=1e-12)


def test_me_w_angular_shape_and_total():
    p = oracle.params_default(oracle.W_ENU)
    shat = 85.0 ** 2
    # d sigma / d cos(theta) ~ (1 - cos)^2, theta between the u quark and the e+
    vals = [oracle.me_w(p, *_cm(shat, c)) for c in (-0.7, 0.1, 0.6)]
    assert math.isclose(vals[0] / vals[1], (1.7 / 0.9) ** 2, rel_tol=1e-12)
    assert math.isclose(vals[2] / vals[1], (0.4 / 0.9) ** 2, rel_tol=1e-12)
    # sigma-hat = 1/(2 s) int |M|^2 dPhi_2, dPhi_2 = dcos/(16 pi); textbook: G_F^2 m_W^4 s D/(18 pi)
    q, _ = si.quad(lambda c: oracle.me_w(p, *_cm(shat, c)) / (16 * math.pi), -1, 1, epsrel=1e-12)
    sig = q / (2 * shat)
    D = 1 / ((shat - p.m_W ** 2) ** 2 + (p.m_W * p.Gam_W) ** 2)
    assert math.isclose(sig, p.G_F ** 2 * p.m_W ** 4 * shat * D / (18 * math.pi), rel_tol=1e-11)
    assert math.isclose(sig, 1.19630629e-06, rel_tol=1e-7)     # SURVEY.md 8(c) probe value
    # resonance-peak identity: sigma(m^2) = 4 pi/(3 m^2) Gam(W->ud) Gam(W->e nu)/Gam_W^2 with the
    # textbook widths Gam(W->e nu) = G_F m^3/(6 sqrt2 pi), Gam(W->ud) = 3 |V|^2 Gam(W->e nu)
    m = p.m_W
    q, _ = si.quad(lambda c: oracle.me_w(p, *_cm(m * m, c)) / (16 * math.pi), -1, 1, epsrel=1e-12)
    gl = p.G_F * m ** 3 / (6 * math.sqrt(2) * math.pi)
    assert math.isclose(q / (2 * m * m), 4 * math.pi / (3 * m * m) * 3 * gl * gl / p.Gam_W ** 2, rel_tol=1e-11)


@pytest.mark.parametrize("up", [0, 1])
def test_me_z_against_dirac_trace_and_peak(up):
    p = oracle.params_default(oracle.Z_BB)
    gz2 = 4 * math.sqrt(2) * p.G_F * p.m_Z ** 2
    s2 = p.sin2_thw
    Lq, Rq = ((0.5 - 2 / 3 * s2), (-2 / 3 * s2)) if up else ((-0.5 + s2 / 3), (s2 / 3))
    Lb, Rb = (-0.5 + s2 / 3), (s2 / 3)
    rng = np.random.default_rng(6)
    for _ in range(4):
        shat = (70 + 50 * rng.random()) ** 2
        qa, qb, p1, p2 = _cm(shat, 2 * rng.random() - 1, 6.28 * rng.random())
        tot = 0.0
        for (cq, Pq) in ((Lq, PL), (Rq, PR)):
            for (cb, Pb) in ((Lb, PL), (Rb, PR)):
                # [vbar(qb) g^mu Pq u(qa)] [ubar(p1) g_mu Pb v(p2)]
                A = _chiral_trace(qb, qa, Pq, Pq)
                B = _chiral_trace(p1, p2, Pb, Pb)
                tot += (cq * cb) ** 2 * lorentz_contract(A, B).real
        D = 1 / ((shat - p.m_Z ** 2) ** 2 + (p.m_Z * p.Gam_Z) ** 2)
        expect = gz2 ** 2 * tot * D / 4.0                 # 1/4 spins; colour 3*3/9 = 1
        assert math.isclose(oracle.me_z(p, up, qa, qb, p1, p2), expect, rel_tol=1e-12)
    # peak identity with textbook widths Gam(Z->ff) = N_c G_F m^3 (L^2+R^2)/(3 sqrt2 pi)
    m = p.m_Z
    q, _ = si.quad(lambda c: oracle.me_z(p, up, *_cm(m * m, c)) / (16 * math.pi), -1, 1, epsrel=1e-12)
    gam = lambda L, R: 3 * p.G_F * m ** 3 * (L * L + R * R) / (3 * math.sqrt(2) * math.pi)
    assert math.isclose(q / (2 * m * m), 4 * math.pi / (3 * m * m) * gam(Lq, Rq) * gam(Lb, Rb) / p.Gam_Z ** 2,
                        rel_tol=1e-11)
    # SURVEY.md 8(c) probe values at sqrt(s-hat) = 92
    q, _ = si.quad(lambda c: oracle.me_z(p, up, *_cm(92.0 ** 2, c)) / (16 * math.pi), -1, 1, epsrel=1e-12)
    assert math.isclose(q / (2 * 92.0 ** 2), 6.05646189e-06 if up else 7.80652503e-06, rel_tol=1e-7)


def test_me_tt_production_closed_forms():
    """ESW / PDG total partonic cross-sections for q qbar -> t tbar and g g -> t tbar."""
    p = oracle.params_default(oracle.TT_LJETS)
    for rs in (360.0, 500.0, 1500.0):
        shat, m = rs * rs, p.m_t
        rho = 4 * m * m / shat
        beta = math.sqrt(1 - rho)
        a_s = p.alpha_s
        for fn, closed in (
            (oracle.me_tt_qq, 8 * math.pi * a_s ** 2 / (27 * shat) * beta * (1 + rho / 2)),
            (oracle.me_tt_gg, math.pi * a_s ** 2 / (3 * shat) * (
                (1 + rho + rho * rho / 16) * math.log((1 + beta) / (1 - beta)) - beta * (7 / 4 + 31 * rho / 16))),
        ):
            q, _ = si.quad(lambda c: fn(p, *_cm(shat, c, m=m)) * beta / (16 * math.pi), -1, 1, epsrel=1e-12)
            assert math.isclose(q / (2 * shat), closed, rel_tol=1e-10)
    # SURVEY.md 8(c) probe values: sqrt(s)=500, g_s = 1  (alpha_s = 1/(4 pi))
    p.alpha_s = 1 / (4 * math.pi)
    shat = 500.0 ** 2
    beta = math.sqrt(1 - 4 * 173.0 ** 2 / shat)
    for fn, val in ((oracle.me_tt_qq, 2.10967036e-08), (oracle.me_tt_gg, 2.09364896e-08)):
        q, _ = si.quad(lambda c: fn(p, *_cm(shat, c, m=173.0)) * beta / (16 * math.pi), -1, 1, epsrel=1e-12)
        assert math.isclose(q / (2 * shat), val, rel_tol=1e-7)


def test_me_tt_symmetry_and_offshell_reading():
    """A9: tau1 + tau2 = 1 for any (off-shell) top momenta that conserve momentum; gg is t<->u symmetric."""
    p = oracle.params_default(oracle.TT_LJETS)
    q1, q2 = np.array([400., 0, 0, 400.]), np.array([300., 0, 0, -300.])
    pt = np.array([380., 30., -20., 150.])
    ptb = q1 + q2 - pt
    assert math.isclose(oracle.me_tt_gg(p, q1, q2, pt, ptb), oracle.me_tt_gg(p, q1, q2, ptb, pt), rel_tol=1e-13)
    assert math.isclose(oracle.me_tt_qq(p, q1, q2, pt, ptb), oracle.me_tt_qq(p, q2, q1, pt, ptb), rel_tol=1e-13)


def test_me_top_decay_against_dirac_trace():
    p = oracle.params_default(oracle.TT_LJETS)
    g2 = 4 * math.sqrt(2) * p.G_F * p.m_W ** 2
    rng = np.random.default_rng(8)
    for _ in range(5):
        b, l, nu = (random_massless(rng) for _ in range(3))
        t = b + l + nu
        mt = math.sqrt(mdot(t, t))
        # M = (g^2/2) V_tb [ubar(b) g^mu PL u(t)] [ubar(nu) g_mu PL v(l)] / (sW - mW^2 + i mW GW)
        A = [[np.trace(slash(b) @ G[mu] @ PL @ (slash(t) + mt * np.eye(4)) @ G[nu_] @ PL) for nu_ in range(4)]
             for mu in range(4)]
        B = _chiral_trace(nu, l, PL, PL)
        sW = mdot(l + nu, l + nu)
        D = 1 / ((sW - p.m_W ** 2) ** 2 + (p.m_W * p.Gam_W) ** 2)
        expect = (g2 / 2) ** 2 * lorentz_contract(A, B).real * D
        assert math.isclose(oracle.me_top_decay(p, 1.0, t, b, l, nu), expect, rel_tol=1e-11)
        assert math.isclose(oracle.me_top_decay(p, 3.0, t, b, l, nu), 3 * expect, rel_tol=1e-11)


def test_top_width_from_decay_me():
    """Gamma(t -> b l nu) = 1/(2 m_t) 1/2 int sum|M|^2 dPhi_3, by explicit 3-body quadrature, against
    the narrow-width textbook value Gamma(t->bW) Gamma(W->l nu)/Gamma_W (within O(Gam_W/m_W))."""
    p = oracle.params_default(oracle.TT_LJETS)
    mt, mW, GW = p.m_t, p.m_W, p.Gam_W
    T = np.array([mt, 0, 0, 0.0])
    xs, ws = np.polynomial.legendre.leggauss(8)
    phis = (np.arange(8) + 0.5) * 2 * math.pi / 8

    def inner(s):
        # dPhi_3 = ds/(2 pi) dPhi_2(t -> b W*) dPhi_2(W* -> l nu); W* along +z (isotropy of the top)
        W, b = two_body_decay(T, math.sqrt(s), 0.0, 1.0, 0.0)
        acc = 0.0
        for c, wc in zip(xs, ws):
            for ph in phis:
                l, nu = two_body_decay(W, 0.0, 0.0, c, ph)
                acc += wc * oracle.me_top_decay(p, 1.0, T, b, l, nu) / 16.0   # dcos/2 dphi/(2pi) average
        ps_tb = (1 - s / mt ** 2) / (8 * math.pi)
        ps_w = 1 / (8 * math.pi)
        return acc * ps_tb * ps_w / (2 * math.pi)

    t_lo, t_hi = math.atan((0 - mW ** 2) / (mW * GW)), math.atan((mt ** 2 - mW ** 2) / (mW * GW))
    ts, wt = np.polynomial.legendre.leggauss(96)
    tot = 0.0
    for x, w in zip(ts, wt):
        t = 0.5 * (t_hi + t_lo) + 0.5 * (t_hi - t_lo) * x
        s = mW ** 2 + mW * GW * math.tan(t)
        dsdt = ((s - mW ** 2) ** 2 + (mW * GW) ** 2) / (mW * GW)
        tot += 0.5 * (t_hi - t_lo) * w * dsdt * inner(s)
    width = tot * 0.5 / (2 * mt)
    assert math.isclose(width, 0.160206, rel_tol=2e-5)            # SURVEY.md 8(c) probe value
    x2 = (mW / mt) ** 2
    g_tbw = p.G_F * mt ** 3 / (8 * math.pi * math.sqrt(2)) * (1 - x2) ** 2 * (1 + 2 * x2)
    g_wlnu = p.G_F * mW ** 3 / (6 * math.pi * math.sqrt(2))
    assert math.isclose(width, g_tbw * g_wlnu / GW, rel_tol=3 * GW / mW)


def test_transverse_boost():
    rng = np.random.default_rng(9)
    mom = np.array([random_massless(rng) for _ in range(5)])
    P = mom.sum(axis=0)
    out = oracle.boost_transverse(P, mom)
    Pn = out.sum(axis=0)
    assert abs(Pn[1]) < 1e-11 and abs(Pn[2]) < 1e-11
    assert math.isclose(Pn[3], P[3], rel_tol=1e-14)
    assert math.isclose(Pn[0], math.sqrt(P[0] ** 2 - P[1] ** 2 - P[2] ** 2), rel_tol=1e-13)
    for a in range(5):                                       # Lorentz invariants survive
        assert abs(mdot(out[a], out[a])) < 1e-9
        for b in range(a):
            assert math.isclose(mdot(out[a], out[b]), mdot(mom[a], mom[b]), rel_tol=1e-11)
    # beta = 0 -> identity
    bal = np.array([[50., 30, 40, 0], [50., -30, -40, 0]])
    assert np.allclose(oracle.boost_transverse(bal.sum(axis=0), bal), bal, rtol=0, atol=1e-13)
