"""Pins of the oracle's config 4 (8-D t tbar dilepton; Eq. 7-8).

The absolute value of the config-4 integral has no closed form ("parity unpinned" beyond the
factor-wise pins); what is pinned here:
  * the Ferrari quartic solver against numpy's companion-matrix roots (a library routine);
  * the neutrino solver: a constructed true (nu, nubar) is recovered among the solutions, every
    solution satisfies the six equations of Eq. 8, and the Jacobian equals the 6x6 determinant
    computed with numpy;
  * every evaluated configuration conserves four-momentum and reproduces the sampled masses;
  * the factor structure of the weight (couplings, PDF split, Gaussian MET transfer function).
"""
import math

import numpy as np
import pytest

import oracle
from helpers import massless, mdot
from paper_1407_7595_b200 import workloads as wl

SEED = 20140729


def setup_module(module):
    oracle.build()


# ------------------------------------------------------------------ quartic
@pytest.mark.parametrize("n_real", [0, 2, 4])
def test_quartic_real_roots_against_numpy(n_real):
    rng = np.random.default_rng(100 + n_real)
    for _ in range(300):
        roots = []
        for _ in range(n_real):
            roots.append(complex(rng.normal(0, 50), 0))
        for _ in range((4 - n_real) // 2):
            z = complex(rng.normal(0, 50), abs(rng.normal(0, 30)) + 0.5)
            roots += [z, z.conjugate()]
        lead = rng.normal() * 3 + 0.1
        c_hi = np.real(np.poly(roots)) * lead                 # highest power first
        got = np.sort(oracle.quartic_real_roots(c_hi[::-1]))
        ref = np.roots(c_hi)
        ref = np.sort(ref[np.abs(ref.imag) < 1e-7 * (1 + np.abs(ref.real))].real)
        if n_real and np.min(np.diff(np.sort([r.real for r in roots[:n_real]]))) < 1e-3:
            continue                                          # nearly double roots: ill-conditioned by nature
        assert len(got) == n_real == len(ref)
        if n_real:
            assert np.allclose(got, ref, rtol=1e-8, atol=1e-8)
            # and they are roots: residual small against the sum of the term magnitudes
            for x in got:
                terms = np.abs(c_hi * np.array([x ** 4, x ** 3, x ** 2, x, 1.0]))
                assert abs(np.polyval(c_hi, x)) <= 1e-9 * terms.sum()


def test_quartic_biquadratic_and_degenerate():
    # (x^2 - 4)(x^2 - 9): q = 0 exactly, the resolvent has the root z0 = (2+3)^2 - ... handled without division by s = 0
    assert np.allclose(np.sort(oracle.quartic_real_roots([36.0, 0.0, -13.0, 0.0, 1.0])), [-3, -2, 2, 3])
    # (x^2 + 1)(x^2 + 4): no real roots
    assert len(oracle.quartic_real_roots([4.0, 0.0, 5.0, 0.0, 1.0])) == 0
    # (x^2 - 1)(x^2 + 4): two real roots
    assert np.allclose(np.sort(oracle.quartic_real_roots([-4.0, 0.0, 3.0, 0.0, 1.0])), [-1, 1])
    # leading coefficient zero: not a quartic, no solutions reported
    assert len(oracle.quartic_real_roots([1.0, 2.0, 3.0, 4.0, 0.0])) == 0


# ------------------------------------------------------------------ neutrino solver
def _random_truth(rng):
    lp, lm = massless(20 + 80 * rng.random(), 2 * rng.random() - 1, 6.28 * rng.random()), \
        massless(20 + 80 * rng.random(), 2 * rng.random() - 1, 6.28 * rng.random())
    b, bb = massless(30 + 100 * rng.random(), 2 * rng.random() - 1, 6.28 * rng.random()), \
        massless(30 + 100 * rng.random(), 2 * rng.random() - 1, 6.28 * rng.random())
    nu, nub = massless(10 + 90 * rng.random(), 2 * rng.random() - 1, 6.28 * rng.random()), \
        massless(10 + 90 * rng.random(), 2 * rng.random() - 1, 6.28 * rng.random())
    return lp, b, lm, bb, nu, nub


def _masses(lp, b, lm, bb, nu, nub):
    return (mdot(lp + nu, lp + nu), mdot(lp + nu + b, lp + nu + b), mdot(lm + nub, lm + nub),
            mdot(lm + nub + bb, lm + nub + bb), nu[1] + nub[1], nu[2] + nub[2])


def _numeric_jacobian(lp, b, lm, bb, nu, nub):
    """6x6 matrix d(s_W+, s_t, s_W-, s_tbar, S_x, S_y)/d(nu_xyz, nubar_xyz), analytic rows, numpy det"""
    def rows(l, bq, v):
        h = v[1:] / v[0]
        return 2 * (l[0] * h - l[1:]), 2 * ((l[0] + bq[0]) * h - (l[1:] + bq[1:]))
    A, B = rows(lp, b, nu)
    Cc, Dd = rows(lm, bb, nub)
    M = np.zeros((6, 6))
    M[0, :3], M[1, :3], M[2, 3:], M[3, 3:] = A, B, Cc, Dd
    M[4, 0] = M[4, 3] = 1.0
    M[5, 1] = M[5, 4] = 1.0
    return M


def test_solver_recovers_truth_and_jacobian_is_the_6x6_determinant():
    rng = np.random.default_rng(8)
    n_sol_seen = set()
    for _ in range(400):
        lp, b, lm, bb, nu, nub = _random_truth(rng)
        sWp, st, sWm, stb, Sx, Sy = _masses(lp, b, lm, bb, nu, nub)
        sol, jac = oracle.dilep_solve(lp, b, lm, bb, sWp, st, sWm, stb, Sx, Sy)
        n_sol_seen.add(len(sol))
        assert len(sol) in (2, 4)                              # real solutions come in pairs, truth is one
        truth = np.stack([nu, nub])
        dist = [np.abs(s - truth).max() for s in sol]
        assert min(dist) <= 1e-7 * 100.0, min(dist)
        for s, J in zip(sol, jac):
            got = _masses(lp, b, lm, bb, s[0], s[1])
            for g, want, scale in zip(got, (sWp, st, sWm, stb, Sx, Sy), (sWp, st, sWm, stb, 100.0, 100.0)):
                assert abs(g - want) <= 1e-8 * abs(scale)
            assert abs(mdot(s[0], s[0])) <= 1e-9 * s[0][0] ** 2 and s[0][0] > 0 and s[1][0] > 0
            det = abs(np.linalg.det(_numeric_jacobian(lp, b, lm, bb, s[0], s[1])))
            assert math.isclose(J * det, 1.0, rel_tol=1e-9)
    assert n_sol_seen == {2, 4}


def test_jacobian_against_finite_differences():
    """independent of the analytic gradient rows: move (nu, nubar) by finite steps"""
    rng = np.random.default_rng(9)
    for _ in range(20):
        lp, b, lm, bb, nu, nub = _random_truth(rng)
        base = np.concatenate([nu[1:], nub[1:]])

        def f(v):
            a = np.concatenate([[np.linalg.norm(v[:3])], v[:3]])
            c = np.concatenate([[np.linalg.norm(v[3:])], v[3:]])
            return np.array(_masses(lp, b, lm, bb, a, c))
        M = np.zeros((6, 6))
        h = 1e-4
        for k in range(6):
            d = np.zeros(6)
            d[k] = h
            M[:, k] = (f(base + d) - f(base - d)) / (2 * h)
        sWp, st, sWm, stb, Sx, Sy = f(base)
        sol, jac = oracle.dilep_solve(lp, b, lm, bb, sWp, st, sWm, stb, Sx, Sy)
        k = int(np.argmin([np.abs(s - np.stack([nu, nub])).max() for s in sol]))
        assert math.isclose(jac[k] * abs(np.linalg.det(M)), 1.0, rel_tol=1e-6)


# ------------------------------------------------------------------ the weight
def test_momentum_conservation_and_sampled_masses():
    p = oracle.params_default(4)
    ev = wl.make_events(4, 40, seed=11)
    S = p.sqrt_s
    n = p.bw_nwidths
    tW = oracle.bw_window(p.m_W, p.Gam_W, (p.m_W - n * p.Gam_W) ** 2, (p.m_W + n * p.Gam_W) ** 2)
    tT = oracle.bw_window(p.m_t, p.Gam_t, (p.m_t - n * p.Gam_t) ** 2, (p.m_t + n * p.Gam_t) ** 2)
    checked, multi = 0, 0
    for e in range(40):
        rec = ev[:, e]
        for i in range(300):
            u = oracle.uniforms(SEED, e, i, 0, 8)
            w, dbg = oracle.weight(4, p, rec, u, debug=True)
            nsol = int(dbg[0])
            if nsol == 0:
                assert w == 0.0
                continue
            assert w > 0.0
            multi += nsol > 1
            want = []
            for k, (m, G, (lo, hi)) in enumerate([(p.m_W, p.Gam_W, tW), (p.m_t, p.Gam_t, tT),
                                                  (p.m_W, p.Gam_W, tW), (p.m_t, p.Gam_t, tT)]):
                smm, _, _ = oracle.bw_point(m, G, lo + (hi - lo) * u[2 + k])
                want.append(m * m + smm)
            for s in range(nsol):
                d = dbg[1 + s * 26:]
                x1, x2 = d[0], d[1]
                mom = d[2:26].reshape(6, 4)                   # l+, nu, b, l-, nubar, bbar (boosted)
                q = np.array([(x1 + x2) * S / 2, 0, 0, (x1 - x2) * S / 2])
                rs = math.sqrt(x1 * x2) * S
                assert np.all(np.abs(mom.sum(axis=0) - q) <= 1e-9 * rs)
                assert 0 < x1 < 1 and 0 < x2 < 1 and rs > 2 * p.m_t
                for k in range(6):
                    assert abs(mdot(mom[k], mom[k])) <= 1e-9 * mom[k][0] ** 2 + 1e-9
                got = [mdot(mom[0] + mom[1], mom[0] + mom[1]), mdot(mom[0] + mom[1] + mom[2], mom[0] + mom[1] + mom[2]),
                       mdot(mom[3] + mom[4], mom[3] + mom[4]), mdot(mom[3] + mom[4] + mom[5], mom[3] + mom[4] + mom[5])]
                for g, wv in zip(got, want):
                    assert math.isclose(g, wv, rel_tol=1e-8)
                checked += 1
    assert checked > 300 and multi > 10


def _first_live_point(p, ev, n_try=4000):
    for e in range(ev.shape[1]):
        for i in range(n_try):
            u = oracle.uniforms(SEED, e, i, 0, 8)
            if oracle.weight(4, p, ev[:, e], u) > 0:
                return ev[:, e].copy(), np.array(u)
    raise AssertionError("no live point found")


def test_factor_structure():
    p = oracle.params_default(4)
    ev = wl.make_events(4, 8, seed=5)
    rec, u = _first_live_point(p, ev)
    w0 = oracle.weight(4, p, rec, u)
    q = oracle.params_default(4)
    q.pdf_A_g, q.pdf_A_q = 0.0, 1.0
    wq = oracle.weight(4, q, rec, u)
    q.pdf_A_g, q.pdf_A_q = 1.0, 0.0
    wg = oracle.weight(4, q, rec, u)
    assert wq > 0 and wg > 0 and math.isclose(wq + wg, w0, rel_tol=1e-13)
    q = oracle.params_default(4)
    q.alpha_s = 2 * p.alpha_s
    assert math.isclose(oracle.weight(4, q, rec, u), 4 * w0, rel_tol=1e-13)
    q = oracle.params_default(4)
    q.V_tb = 0.5                                               # |V_tb|^2 in each decay
    assert math.isclose(oracle.weight(4, q, rec, u), w0 / 16, rel_tol=1e-13)
    q = oracle.params_default(4)
    q.sqrt_s = 300.0
    assert oracle.weight(4, q, rec, u) == 0.0
    # Gaussian MET TF: shift the measured MET by d and the sampled offset back, so that the total
    # neutrino pT (hence the whole kinematics) is unchanged; only exp(-|met - S|^2/(2 sigma^2)) moves
    sig, ns = p.met_sigma, p.met_nsigma
    off = sig * ns * (2 * u[6] - 1)
    d = 3.0 if off > -30.0 else -3.0
    rec2 = rec.copy()
    rec2[12] += d
    u2 = u.copy()
    u2[6] = ((off - d) / (sig * ns) + 1) / 2
    assert 0 < u2[6] < 1
    offy = sig * ns * (2 * u[7] - 1)
    ratio = math.exp(-((off - d) ** 2 + offy ** 2) / (2 * sig ** 2)) / math.exp(-(off ** 2 + offy ** 2) / (2 * sig ** 2))
    assert math.isclose(oracle.weight(4, p, rec2, u2), w0 * ratio, rel_tol=1e-9)
    # jet TF: w is proportional to T(E_jet; E) at fixed parton energy -- change E_jet and u0 together
    Ej, E = rec[6], rec[6] * (p.jetE_rlo + (p.jetE_rhi - p.jetE_rlo) * u[0])
    Ej2 = 1.1 * Ej
    u3 = u.copy()
    u3[0] = (E / Ej2 - p.jetE_rlo) / (p.jetE_rhi - p.jetE_rlo)
    rec3 = rec.copy()
    rec3[6] = Ej2
    want = w0 * (Ej2 / Ej) * oracle.tf_jet(p, Ej2, E) / oracle.tf_jet(p, Ej, E)     # volume factor E_jet dr
    assert math.isclose(oracle.weight(4, p, rec3, u3), want, rel_tol=1e-9)


def test_fp64_oracle_agrees_with_its_long_double_referee():
    p = oracle.params_default(4)
    ev = wl.make_events(4, 12, seed=7)
    live = 0
    for e in range(12):
        wo = oracle.eval_points(4, p, ev, e, 0, 1500, SEED)
        wx = oracle.eval_points_x(4, p, ev, e, 0, 1500, SEED)
        assert np.array_equal(wo == 0, wx == 0)
        m = wo != 0
        live += m.sum()
        if m.any():
            assert np.max(np.abs(wo[m] - wx[m]) / np.abs(wx[m])) < 1e-8
    assert live > 200
