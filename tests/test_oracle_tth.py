"""Pins of the oracle's NEXT-4 process: t tbar H(-> b bbar) dilepton with four b jets
(PAPER.md:101-109 Eq. 7, :111-118 Eq. 8, :120-137 Eq. 9, :143 Eq. 10, :178-180 Eq. 11;
DESIGN.md readings A18-A22).  What the paper and the mathematics fix is checked here; the factorised
matrix element itself is a stated reading (A20) and stays "ME parity unpinned"."""
import itertools

import numpy as np
import pytest

import oracle
from helpers import mdot, slash, two_body_decay
from paper_1407_7595_b200 import workloads as wl

PROC = oracle.TTH_DILEP


def _dir(eta, phi):
    return np.array([1.0, np.cos(phi) / np.cosh(eta), np.sin(phi) / np.cosh(eta), np.tanh(eta)])


def _from_pt(pt, eta, phi):
    return pt * np.array([np.cosh(eta), np.cos(phi), np.sin(phi), np.sinh(eta)])


# ----------------------------------------------------------------------------------------------
# Eq. 9
# ----------------------------------------------------------------------------------------------
def _eq9_forward(E1, E2, n1, n2):
    """PAPER.md:131-133 Eq. 9 typed out for massless quarks: f = E1 + E2,
    m_H^2 = (E1 + E2)^2 - |p1|^2 - |p2|^2 - 2 |p1||p2| cos(Delta theta)"""
    p1, p2 = E1 * n1[1:], E2 * n2[1:]
    cosd = (p1 @ p2) / (np.linalg.norm(p1) * np.linalg.norm(p2))
    return E1 + E2, (E1 + E2) ** 2 - p1 @ p1 - p2 @ p2 - 2 * np.linalg.norm(p1) * np.linalg.norm(p2) * cosd


def test_eq9_round_trip_both_orderings_and_jacobian():
    rng = np.random.default_rng(9)
    for _ in range(200):
        n1, n2 = _dir(rng.uniform(-2.5, 2.5), rng.uniform(0, 6.28)), _dir(rng.uniform(-2.5, 2.5), rng.uniform(0, 6.28))
        K12 = 1.0 - n1[1:] @ n2[1:]
        E1, E2 = rng.uniform(20, 300, 2)
        if abs(E1 - E2) < 1.0:
            continue
        f, m2 = _eq9_forward(E1, E2, n1, n2)
        r1, r2, jac = oracle.eq9_roots(K12, f, m2)
        assert len(r1) == 2
        # both orderings come back; one of them is the point we started from
        got = sorted(zip(r1, r2))
        want = sorted([(E1, E2), (E2, E1)])
        assert np.allclose(got, want, rtol=1e-10)
        assert np.allclose(r1 + r2, f, rtol=1e-14)
        # |d(E1,E2)/d(f,m^2)| = 1 / |det d(f,m^2)/d(E1,E2)| by central differences of the forward map (bilinear in
        # the energies, so a large step is exact up to rounding)
        h = 1.0
        J = np.empty((2, 2))
        for k, (d1, d2) in enumerate(((h, 0.0), (0.0, h))):
            fp, mp = _eq9_forward(E1 + d1, E2 + d2, n1, n2)
            fm, mm = _eq9_forward(E1 - d1, E2 - d2, n1, n2)
            J[:, k] = [(fp - fm) / (2 * h), (mp - mm) / (2 * h)]
        assert jac == pytest.approx(1.0 / abs(np.linalg.det(J)), rel=1e-7)


def test_eq9_no_root_beyond_the_kinematic_limit():
    # E1 E2 <= f^2/4, so m^2 > K12 f^2 / 2 has no solution
    K12, f = 0.7, 200.0
    assert len(oracle.eq9_roots(K12, f, 0.5 * K12 * f * f * 1.0001)[0]) == 0
    assert len(oracle.eq9_roots(K12, f, 0.5 * K12 * f * f * 0.9999)[0]) == 2


def test_higgs_breit_wigner_window_integral():
    # int D_H ds over the window = Delta t / (m Gamma) by independent quadrature (narrow and wide width)
    for mH, GH in ((125.0, 0.00407), (125.0, 5.0)):
        lo, hi = (mH - 15 * GH) ** 2, (mH + 15 * GH) ** 2
        t_lo, t_hi = oracle.bw_window(mH, GH, lo, hi)
        x, w = np.polynomial.legendre.leggauss(400)
        # substitute s = m^2 + m G tan t by hand to resolve the peak
        t = 0.5 * (t_hi + t_lo) + 0.5 * (t_hi - t_lo) * x
        s = mH * mH + mH * GH * np.tan(t)
        D = 1.0 / ((s - mH * mH) ** 2 + (mH * GH) ** 2)
        dsdt = mH * GH / np.cos(t) ** 2
        quad = 0.5 * (t_hi - t_lo) * np.sum(w * D * dsdt)
        assert quad == pytest.approx((t_hi - t_lo) / (mH * GH), rel=1e-12)
        assert np.tan(t_lo) == pytest.approx((lo - mH * mH) / (mH * GH), rel=1e-9)


# ----------------------------------------------------------------------------------------------
# factorised matrix-element pieces (reading A20): what is checkable
# ----------------------------------------------------------------------------------------------
def test_higgs_decay_factor_is_the_dirac_trace():
    # sum over spins and colours |ubar(p1) v(p2)|^2 y_b^2 = 3 y_b^2 Tr[p1-slash p2-slash] = 3 y_b^2 4 p1.p2
    p = oracle.params_default(PROC)
    rng = np.random.default_rng(2)
    for _ in range(5):
        n1, n2 = _dir(rng.uniform(-2, 2), rng.uniform(0, 6.28)), _dir(rng.uniform(-2, 2), rng.uniform(0, 6.28))
        p1, p2 = rng.uniform(30, 200) * n1, rng.uniform(30, 200) * n2
        tr = np.trace(slash(p1) @ slash(p2)).real
        sH = mdot(p1 + p2, p1 + p2)
        assert oracle.tth_decay(p, sH) == pytest.approx(3 * p.yuk_b ** 2 * tr, rel=1e-12)
    p.tth_hyp = 1
    assert oracle.tth_decay(p, 1000.0) == pytest.approx(4 * np.pi * p.alpha_s * 1000.0, rel=1e-14)


def _massive(rng, m):
    k = rng.uniform(10, 400) * np.array([np.sin(a := rng.uniform(0, np.pi)) * np.cos(b := rng.uniform(0, 6.28)),
                                         np.sin(a) * np.sin(b), np.cos(a)])
    return np.concatenate([[np.sqrt(m * m + k @ k)], k])


def test_radiators_against_their_definitions():
    rng = np.random.default_rng(3)
    p0, p1 = oracle.params_default(PROC), oracle.params_default(PROC)
    p1.tth_hyp = 1
    for _ in range(50):
        pt, ptb, k = _massive(rng, 173.0 + rng.normal()), _massive(rng, 173.0 + rng.normal()), _massive(rng, rng.uniform(20, 200))
        # hyp 0: soft scalar emission off either top: y_t^2 |2 m_t / ((p_t + k)^2 - p_t^2) + (t -> tbar)|^2
        amp = 2 * p0.m_t / (mdot(pt + k, pt + k) - mdot(pt, pt)) + 2 * p0.m_t / (mdot(ptb + k, ptb + k) - mdot(ptb, ptb))
        assert oracle.tth_radiator(p0, pt, ptb, k) == pytest.approx(p0.yuk_t ** 2 * amp ** 2, rel=1e-12)
        # hyp 1: eikonal current J = p_t/(p_t.k) - p_tbar/(p_tbar.k); -J^2 >= 0 because J.k = 0 and k is timelike
        J = pt / mdot(pt, k) - ptb / mdot(ptb, k)
        assert abs(mdot(J, k)) < 1e-15
        val = oracle.tth_radiator(p1, pt, ptb, k)
        assert val == pytest.approx(-4 * np.pi * p1.alpha_s * mdot(J, J), rel=1e-9)
        assert val >= 0


def test_tt_invariants_next_to_a_third_body():
    p = oracle.params_default(PROC)
    rng = np.random.default_rng(4)
    for _ in range(50):
        pt, ptb, k = _massive(rng, 173.0), _massive(rng, 173.0), _massive(rng, 125.0)
        P = pt + ptb + k
        x1, x2 = (P[0] + P[3]) / p.sqrt_s, (P[0] - P[3]) / p.sqrt_s
        q1, q2 = x1 * 7000 * np.array([1, 0, 0, 1.0]), x2 * 7000 * np.array([1, 0, 0, -1.0])
        ok, t1, t2, rho = oracle.tth_tt_invariants(p, q1, q2, pt, ptb)
        assert ok and t1 + t2 == pytest.approx(1.0, abs=1e-15)
        assert rho == pytest.approx(4 * 173.0 ** 2 / mdot(pt + ptb, pt + ptb), rel=1e-14)
        # physical region of the 2 -> 2 matrix elements: tau1 tau2 >= rho/4 for on-shell tops
        assert t1 * t2 >= rho / 4 * (1 - 1e-12)
        assert oracle.me_tt_gg_inv(p, t1, t2, rho) > 0 and oracle.me_tt_qq_inv(p, t1, t2, rho) > 0
    # without a third body it is the t tbar production of configs 3-5 (pinned by quadrature in test_oracle_blocks)
    P = np.array([600.0, 0, 0, 100.0])
    pt, ptb = two_body_decay(P, 173.0, 173.0, 0.3, 1.0)
    x1, x2 = (P[0] + P[3]) / p.sqrt_s, (P[0] - P[3]) / p.sqrt_s
    q1, q2 = x1 * 7000 * np.array([1, 0, 0, 1.0]), x2 * 7000 * np.array([1, 0, 0, -1.0])
    ok, t1, t2, rho = oracle.tth_tt_invariants(p, q1, q2, pt, ptb)
    assert oracle.me_tt_gg_inv(p, t1, t2, rho) == pytest.approx(oracle.me_tt_gg(p, q1, q2, pt, ptb), rel=1e-12)
    assert oracle.me_tt_qq_inv(p, t1, t2, rho) == pytest.approx(oracle.me_tt_qq(p, q1, q2, pt, ptb), rel=1e-12)


# ----------------------------------------------------------------------------------------------
# the assembled weight
# ----------------------------------------------------------------------------------------------
def _live_points(p, rec, n, seed=5, event=0):
    out = []
    i = 0
    while len(out) < n and i < 400000:
        u = oracle.uniforms(seed, event, i, 0, 8)
        w, dbg = oracle.weight(PROC, p, rec, u, debug=True)
        if w != 0.0:
            out.append((u, w, dbg))
        i += 1
    return out


@pytest.fixture(scope="module")
def closure_events():
    return wl.make_tth_events(6, smear=True)


def test_every_configuration_conserves_momentum_and_balances_eq11(closure_events):
    p = oracle.params_default(PROC)
    for e in range(3):
        rec = closure_events[:, e]
        for u, w, dbg in _live_points(p, rec, 12, event=e):
            nsol = int(dbg[0])
            assert 1 <= nsol <= 8
            # the sampled invariants, from the pinned Breit-Wigner map
            s_k = []
            for k, (m, G) in enumerate(((p.m_W, p.Gam_W), (p.m_t, p.Gam_t), (p.m_W, p.Gam_W), (p.m_t, p.Gam_t))):
                lo, hi = oracle.bw_window(m, G, (m - 15 * G) ** 2, (m + 15 * G) ** 2)
                s_k.append(m * m + oracle.bw_point(m, G, lo + (hi - lo) * u[2 + k])[0])
            lo, hi = oracle.bw_window(p.m_H, p.Gam_H, (p.m_H - 15 * p.Gam_H) ** 2, (p.m_H + 15 * p.Gam_H) ** 2)
            sH = p.m_H ** 2 + oracle.bw_point(p.m_H, p.Gam_H, lo + (hi - lo) * u[6])[0]
            f = (rec[12] + rec[15]) * (p.jetE_rlo + (p.jetE_rhi - p.jetE_rlo) * u[7])
            for s in range(nsol):
                d = dbg[1 + s * 34: 1 + (s + 1) * 34]
                x1, x2, mom = d[0], d[1], d[2:].reshape(8, 4)
                lp, nu, b, lm, nub, bb, b1, b2 = mom
                P = mom.sum(axis=0)
                rs = np.sqrt(x1 * x2) * p.sqrt_s
                # Eq. 11: the neutrinos balance the visible system of the point; q1 + q2 = sum of final momenta
                assert abs(P[1]) <= 1e-9 * rs and abs(P[2]) <= 1e-9 * rs
                q = np.array([(x1 + x2) * 7000.0, 0, 0, (x1 - x2) * 7000.0])
                assert np.all(np.abs(q - P) <= 1e-9 * rs)
                # Eq. 8: the four propagator invariants are the sampled ones; Eq. 9: so are f and m_H^2
                assert mdot(lp + nu, lp + nu) == pytest.approx(s_k[0], rel=1e-9)
                assert mdot(lp + nu + b, lp + nu + b) == pytest.approx(s_k[1], rel=1e-9)
                assert mdot(lm + nub, lm + nub) == pytest.approx(s_k[2], rel=1e-9)
                assert mdot(lm + nub + bb, lm + nub + bb) == pytest.approx(s_k[3], rel=1e-9)
                assert mdot(b1 + b2, b1 + b2) == pytest.approx(sH, rel=1e-9)
                assert b1[0] + b2[0] == pytest.approx(f, rel=1e-12)
                for v in mom:
                    assert abs(mdot(v, v)) <= 1e-9 * v[0] ** 2 and v[0] > 0
                # directions are the measured ones (delta TFs in theta, phi)
                for j, v in zip(range(4), (b, bb, b1, b2)):
                    assert np.allclose(v / v[0], _dir(rec[7 + 3 * j], rec[8 + 3 * j]), atol=1e-12)


def _rebuild_weight(p, rec, u):
    """The weight of Eq. 7 assembled in the test from independently pinned parts: oracle.dilep_solve
    (solutions + Jacobian, pinned in test_oracle_dilep), the transfer function and Breit-Wigner blocks, the
    matrix-element blocks, and the measure typed out here from PAPER.md:49 Eq. 2 and :105 Eq. 7."""
    rlo, dr = p.jetE_rlo, p.jetE_rhi - p.jetE_rlo
    twopi = 2 * np.pi
    lp, lm = _from_pt(*rec[0:3]), _from_pt(*rec[3:6])
    Ej = rec[6::3]
    n = [_dir(rec[7 + 3 * j], rec[8 + 3 * j]) for j in range(4)]
    sin_th = [1 / np.cosh(rec[7 + 3 * j]) for j in range(4)]
    E = [Ej[0] * (rlo + dr * u[0]), Ej[1] * (rlo + dr * u[1])]
    vol = Ej[0] * dr * Ej[1] * dr
    s_k, bw = [], 1.0
    for k, (m, G) in enumerate(((p.m_W, p.Gam_W), (p.m_t, p.Gam_t), (p.m_W, p.Gam_W), (p.m_t, p.Gam_t))):
        lo, hi = oracle.bw_window(m, G, (m - 15 * G) ** 2, (m + 15 * G) ** 2)
        smm, dsdt, D = oracle.bw_point(m, G, lo + (hi - lo) * u[2 + k])
        s_k.append((m * m + smm, D))
        vol *= (hi - lo) * dsdt
    K12 = 1 - n[2][1:] @ n[3][1:]
    if p.tth_hyp == 0:
        lo, hi = oracle.bw_window(p.m_H, p.Gam_H, (p.m_H - 15 * p.Gam_H) ** 2, (p.m_H + 15 * p.Gam_H) ** 2)
        smm, dsdt, propH = oracle.bw_point(p.m_H, p.Gam_H, lo + (hi - lo) * u[6])
        sH = p.m_H ** 2 + smm
        vol *= (hi - lo) * dsdt
    else:
        s_lo, s_hi = 2 * K12 * Ej[2] * Ej[3] * rlo ** 2, 2 * K12 * Ej[2] * Ej[3] * p.jetE_rhi ** 2
        sH = s_lo * (s_hi / s_lo) ** u[6]
        propH = 1 / sH ** 2
        vol *= sH * np.log(s_hi / s_lo)                      # ds = s ln(s_hi/s_lo) du
    f = (Ej[2] + Ej[3]) * (rlo + dr * u[7])
    vol *= (Ej[2] + Ej[3]) * dr
    disc = f * f - 2 * sH / K12
    if disc <= 0:
        return 0.0
    total = 0.0
    for sgn in (+1, -1):
        E1, E2 = 0.5 * (f + sgn * np.sqrt(disc)), 0.5 * (f - sgn * np.sqrt(disc))
        if not (rlo * Ej[2] <= E1 <= p.jetE_rhi * Ej[2] and rlo * Ej[3] <= E2 <= p.jetE_rhi * Ej[3]):
            continue
        jac9 = 1 / (2 * K12 * abs(E1 - E2))
        Es = E + [E1, E2]
        mom = [Es[j] * n[j] for j in range(4)]
        b, bb, b1, b2 = mom
        vis = lp + lm + b + bb + b1 + b2
        sols, jacs = oracle.dilep_solve(lp, b, lm, bb, s_k[0][0], s_k[1][0], s_k[2][0], s_k[3][0], -vis[1], -vis[2])
        # transfer functions and d^3p/((2 pi)^3 2E) -> E sin(theta) dE / (2 (2 pi)^3) per jet (Eq. 7)
        fac = jac9
        for j in range(4):
            fac *= oracle.tf_jet(p, Ej[j], Es[j]) * Es[j] * sin_th[j] / (2 * twopi ** 3)
        fac *= 1 / (2 * lp[0] * twopi ** 3) / (2 * lm[0] * twopi ** 3)              # leptons, delta TFs
        for (nu, nub), J in zip(sols, jacs):
            P = vis + nu + nub
            x1, x2 = (P[0] + P[3]) / p.sqrt_s, (P[0] - P[3]) / p.sqrt_s
            if not (0 < x1 < 1 and 0 < x2 < 1):
                continue
            q1, q2 = x1 * p.sqrt_s / 2 * np.array([1, 0, 0, 1.0]), x2 * p.sqrt_s / 2 * np.array([1, 0, 0, -1.0])
            pt, ptb = lp + nu + b, lm + nub + bb
            ok, t1, t2, rho = oracle.tth_tt_invariants(p, q1, q2, pt, ptb)
            if not ok:
                continue
            prod = oracle.tt_flavour_sum(p, x1, x2, oracle.me_tt_gg_inv(p, t1, t2, rho), oracle.me_tt_qq_inv(p, t1, t2, rho))
            me = (prod * oracle.tth_radiator(p, pt, ptb, b1 + b2) * propH * oracle.tth_decay(p, sH)
                  * s_k[1][1] * s_k[3][1]
                  * 0.5 * oracle.me_top_decay_D(p, 1.0, pt, b, lp, nu, s_k[0][1])
                  * 0.5 * oracle.me_top_decay_D(p, 1.0, ptb, bb, lm, nub, s_k[2][1]))
            flux = x1 * x2 * p.sqrt_s ** 2 / 4                                       # |q1||q2|, Eq. 1
            nu_meas = J / (twopi ** 3 * 2 * nu[0]) / (twopi ** 3 * 2 * nub[0])        # d^3nu d^3nubar -> d(s_k, S_T)
            total += fac * nu_meas * me / flux
    return vol * twopi ** 4 * (2 / p.sqrt_s ** 2) * total


@pytest.mark.parametrize("hyp", [0, 1])
def test_weight_equals_its_parts_assembled_in_the_test(closure_events, hyp):
    p = oracle.params_default(PROC)
    p.tth_hyp = hyp
    n = 0
    for e in range(3):
        rec = closure_events[:, e]
        for u, w, _ in _live_points(p, rec, 8, event=e):
            assert _rebuild_weight(p, rec, u) == pytest.approx(w, rel=1e-9)
            n += 1
    assert n >= 12


@pytest.mark.parametrize("hyp", [0, 1])
def test_chart_independence_eq9_against_flat_energies(closure_events, hyp):
    # The Eq. 9 chart (f, m_H^2) with both orderings and the window test covers exactly the (E1, E2) box:
    # the same integral in the flat chart agrees within Monte Carlo errors.  A wide Higgs makes the flat
    # chart usable (with 4 MeV it would never hit the window).
    p = oracle.params_default(PROC)
    p.tth_hyp, p.Gam_H = hyp, 4.0
    ev = closure_events[:, :2]
    n = 150000
    pa, ea = oracle.integrate(PROC, p, ev, n, 11)
    p.tth_chart = 1
    pb, eb = oracle.integrate(PROC, p, ev, n, 12)
    assert np.all(pa > 0) and np.all(pb > 0)
    pull = (pa - pb) / np.hypot(ea, eb)
    assert np.all(np.abs(pull) < 4.0), (pa, pb, pull)
    assert np.all(np.hypot(ea, eb) / pa < 0.35)            # the comparison has resolving power


def test_symmetric_in_the_two_higgs_candidates_per_point(closure_events):
    # both Eq. 9 orderings are summed, so exchanging the measured jets b1 <-> b2 changes nothing, point by point
    p = oracle.params_default(PROC)
    rec = closure_events[:, 0].copy()
    swapped = rec.copy()
    swapped[12:15], swapped[15:18] = rec[15:18], rec[12:15]
    for u, w, _ in _live_points(p, rec, 10):
        assert oracle.weight(PROC, p, swapped, u) == pytest.approx(w, rel=1e-11)


def test_assignment_sum_is_its_definition(closure_events):
    # PAPER.md:103-109 Eq. 7 "sum over all permutations of assigning measured jets to partons": 4!/2 = 12
    # distinct assignments of four b jets to (b, bbar, {b1, b2})
    p1, p12 = oracle.params_default(PROC), oracle.params_default(PROC)
    p12.n_perm = 12
    rec = closure_events[:, 1]
    jets = rec[6:].reshape(4, 3)
    rng = np.random.default_rng(7)
    done = 0
    for i in range(4000):
        u = oracle.uniforms(3, 0, i, 0, 8)
        w12 = oracle.weight(PROC, p12, rec, u)
        if w12 == 0.0:
            continue
        tot, seen = 0.0, set()
        for sig in itertools.permutations(range(4)):
            key = (sig[0], sig[1], frozenset(sig[2:]))
            if key in seen:
                continue
            seen.add(key)
            r2 = np.concatenate([rec[:6], jets[list(sig)].ravel()])
            tot += oracle.weight(PROC, p1, r2, u)
        assert len(seen) == 12
        assert w12 == pytest.approx(tot, rel=1e-10)
        # with all 12 the result cannot depend on the order of the jets in the record
        sh = rng.permutation(4)
        r3 = np.concatenate([rec[:6], jets[sh].ravel()])
        assert oracle.weight(PROC, p12, r3, u) == pytest.approx(w12, rel=1e-10)
        done += 1
        if done >= 6:
            break
    assert done >= 3


def test_fp64_oracle_against_the_long_double_referee(closure_events):
    p = oracle.params_default(PROC)
    bad = 0
    tot = 0
    for e in range(3):
        rec = closure_events[:, e]
        for u, w, _ in _live_points(p, rec, 40, event=e):
            ref = oracle.weight_x(PROC, p, rec, u)
            tot += 1
            bad += abs(w - ref) > 1e-10 * abs(ref)
    assert tot >= 60 and bad <= 0.05 * tot


# ----------------------------------------------------------------------------------------------
# 1/sigma and the discriminant (Eq. 10; reading A22)
# ----------------------------------------------------------------------------------------------
def test_normalisation_and_discriminant_definitions():
    rng = np.random.default_rng(0)
    ps, pb = 10.0 ** rng.uniform(-40, -36, 50), 10.0 ** rng.uniform(-42, -38, 50)
    g = 10.0 ** rng.uniform(-20, -15, 50)
    ss, sb = oracle.normalisation(ps, g), oracle.normalisation(pb, g)
    assert ss == pytest.approx(np.mean(ps / g), rel=1e-13)
    D = oracle.discriminant(ps, pb, ss, sb)
    assert np.allclose(D, np.log10(ps / ss) - np.log10(pb / sb), rtol=0, atol=1e-12)
    # D is invariant under a common rescaling of either hypothesis (that is what 1/sigma is for)
    assert np.allclose(oracle.discriminant(7 * ps, pb, 7 * ss, sb), D, atol=1e-12)


def test_importance_sampled_normalisation_recovers_a_known_integral():
    # sigma = int p(X) dX estimated as <p/g> over X ~ g: with p = c g h(X) and a known <h> it is exact in expectation
    ev = wl.make_events(wl.TTH_DILEP, 20000, seed=3)
    g = wl.event_density(wl.TTH_DILEP, ev)
    assert np.all(g > 0)
    # h = indicator(lepton 1 pT < 60): P = 1 - exp(-1)
    h = (ev[0] < 60.0).astype(float)
    est = oracle.normalisation(2.5 * g * h, g)
    assert est == pytest.approx(2.5 * (1 - np.exp(-1.0)), rel=0.02)


def test_discriminant_separates_resonant_from_non_resonant_events():
    # the point of Eq. 10: events with m_bb = m_H score higher under the signal hypothesis than events with a
    # non-resonant b bbar pair.  Unsmeared jets would make the narrow Higgs a delta function, so smear.
    sig = wl.make_tth_events(8, seed=21, resonant=True)
    bkg = wl.make_tth_events(8, seed=22, resonant=False)
    ps, pb = oracle.params_default(PROC), oracle.params_default(PROC)
    pb.tth_hyp = 1
    n = 30000
    D = []
    for ev in (sig, bkg):
        a, _ = oracle.integrate(PROC, ps, ev, n, 5)
        b, _ = oracle.integrate(PROC, pb, ev, n, 5)
        ok = b > 0                                          # a = 0 (m_H outside the reach of the TF windows): D = -inf
        with np.errstate(divide="ignore"):
            D.append(np.log10(a[ok] / b[ok]))
    assert len(D[0]) >= 5 and len(D[1]) >= 3
    assert np.median(D[0]) > np.median(D[1]) + 0.3
