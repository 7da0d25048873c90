"""Pins of the oracle's parton-level mode (NEXT-2; Table 2) -- and, through it,
of the complete t tbar -> b l nu bbar q qbar' matrix element used by configs 3-5 (production x top
propagators x decays x spin-average factors), whose absolute normalisation has no other pin.

Narrow-width closure: integrating |M|^2 over the six-body phase space at fixed partonic s-hat must
give  sigma-hat(gg -> t tbar) x Gamma(t -> b l nu)/Gamma_t x Gamma(t -> b q qbar')/Gamma_t  up to
O(Gamma_t/m_t), with the textbook sigma-hat and the partial width pinned in test_oracle_blocks.py.
The phase space is built here from two-body decays (tests/helpers.py), independently of the oracle.
"""
import itertools
import math

import numpy as np
import pytest

import oracle
from helpers import mdot, two_body_decay
from paper_1407_7595_b200 import workloads as wl


def setup_module(module):
    oracle.build()


def _bw(rng, m, G, s_lo, s_hi):
    t_lo, t_hi = math.atan((s_lo - m * m) / (m * G)), math.atan((s_hi - m * m) / (m * G))
    t = t_lo + (t_hi - t_lo) * rng.random()
    s = m * m + m * G * math.tan(t)
    dsdt = ((s - m * m) ** 2 + (m * G) ** 2) / (m * G)
    return s, (t_hi - t_lo) * dsdt / (2 * math.pi)           # ds/(2 pi) per unit of the uniform variate


def _k(M2, a2, b2):
    return math.sqrt(max(0.0, (M2 - a2 - b2) ** 2 - 4 * a2 * b2)) / (2 * math.sqrt(M2))


def _phi2(M2, a2, b2):
    return _k(M2, a2, b2) / (4 * math.pi * math.sqrt(M2))    # two-body phase-space volume


def _decay(rng, P, m1, m2):
    return two_body_decay(P, m1, m2, 2 * rng.random() - 1, 2 * math.pi * rng.random())


def test_narrow_width_closure_of_the_full_matrix_element():
    p = oracle.params_default(3)
    p.pdf_A_q, p.pdf_A_g = 0.0, 1.0                          # g g initial state only
    p.Gam_t = 0.2                                            # narrow: off-shell corrections ~ Gamma_t/m_t
    mt, Gt, mW, GW, S = p.m_t, p.Gam_t, p.m_W, p.Gam_W, p.sqrt_s ** 2
    rs, y = 600.0, 0.3
    shat = rs * rs
    x1, x2 = rs / p.sqrt_s * math.exp(y), rs / p.sqrt_s * math.exp(-y)
    P = np.array([(x1 + x2) * p.sqrt_s / 2, 0.0, 0.0, (x1 - x2) * p.sqrt_s / 2])
    rng = np.random.default_rng(17)
    n = 24000
    mom = np.empty((24, n))
    wps = np.empty(n)
    nw = 40.0
    for i in range(n):
        st, j1 = _bw(rng, mt, Gt, (mt - nw * Gt) ** 2, (mt + nw * Gt) ** 2)
        stb, j2 = _bw(rng, mt, Gt, (mt - nw * Gt) ** 2, (mt + nw * Gt) ** 2)
        sw1, j3 = _bw(rng, mW, GW, 0.0, st)                  # full W range: the partial width integrates it all
        sw2, j4 = _bw(rng, mW, GW, 0.0, stb)
        t, tb = _decay(rng, P, math.sqrt(st), math.sqrt(stb))
        W1, b_lep = _decay(rng, t, math.sqrt(sw1), 0.0)
        lep, nu = _decay(rng, W1, 0.0, 0.0)
        W2, b_had = _decay(rng, tb, math.sqrt(sw2), 0.0)
        q, qb = _decay(rng, W2, 0.0, 0.0)
        mom[:, i] = np.concatenate([lep, nu, b_had, b_lep, q, qb])
        wps[i] = (j1 * j2 * j3 * j4 * _phi2(shat, st, stb) * _phi2(st, sw1, 0) * _phi2(sw1, 0, 0) *
                  _phi2(stb, sw2, 0) * _phi2(sw2, 0, 0))
    w = oracle.parton_weights(3, p, mom)
    me2 = w * (x1 * x2 * S / 4) / (oracle.pdf_shape(p, x1) * oracle.pdf_shape(p, x2))
    vals = wps * me2 / (2 * shat)
    sig_mc, err = vals.mean(), vals.std(ddof=1) / math.sqrt(n)
    rho = 4 * mt * mt / shat
    beta = math.sqrt(1 - rho)
    sig_gg = math.pi * p.alpha_s ** 2 / (3 * shat) * ((1 + rho + rho * rho / 16) * math.log((1 + beta) / (1 - beta))
                                                      - beta * (7 / 4 + 31 * rho / 16))
    gam_lnu = 0.160206                                       # Gamma(t -> b l nu), pinned in test_oracle_blocks.py
    window = (2 * math.atan(((mt + nw * Gt) ** 2 - mt * mt) / (mt * Gt)) / math.pi) ** 2   # ~ fraction of both BWs sampled
    expect = sig_gg * (gam_lnu / Gt) * (3 * gam_lnu / Gt) * window
    assert err < 0.015 * expect
    assert abs(sig_mc - expect) < 4 * err + 0.01 * expect, (sig_mc, expect, err)


def test_parton_weight_assignments_and_symmetries():
    ev = wl.make_parton_events(12, seed=5)
    base = oracle.params_default(3)
    w1 = oracle.parton_weights(3, base, ev)
    assert np.all(w1 > 0)
    # the definition written out: permute the four jets of the record, sum the single-assignment weights
    full = oracle.params_default(3)
    full.n_perm = 24
    w24 = oracle.parton_weights(3, full, ev)
    for e in range(4):
        rec = ev[:, e].reshape(6, 4)
        terms = []
        for sig in itertools.permutations(range(4)):
            r = rec.copy()
            for role, j in enumerate(sig):
                r[2 + role] = rec[2 + j]
            terms.append(oracle.parton_weights(3, base, r.reshape(24, 1))[0])
        assert math.isclose(w24[e], math.fsum(terms), rel_tol=1e-12)
        assert w24[e] >= w1[e]
    # generated with the right assignment: together with its q <-> qbar' twin (same top and W masses)
    # it dominates the sum for on-shell events
    assert np.median(w1 / w24) > 0.25
    # couplings: g_s^4 and the two decays' |V_tb|^2
    q = oracle.params_default(3)
    q.alpha_s, q.V_tb = 2 * base.alpha_s, 0.5
    assert np.allclose(oracle.parton_weights(3, q, ev), w1 * 4 / 16, rtol=1e-12)
    # the long-double referee agrees
    wx = oracle.parton_weights(3, base, ev, extended=True)
    assert np.max(np.abs(w1 - wx) / wx) < 1e-10
    # a transverse kick of the whole event is undone by O7 up to the recoil's effect on x1 x2: the weight
    # of the boosted configuration equals that of the original one
    kick = ev.copy().reshape(6, 4, -1)
    bx = 0.2
    g = 1 / math.sqrt(1 - bx * bx)
    E, px = kick[:, 0].copy(), kick[:, 1].copy()
    kick[:, 0], kick[:, 1] = g * (E + bx * px), g * (px + bx * E)
    wk = oracle.parton_weights(3, base, kick.reshape(24, -1))
    assert np.allclose(wk, w1, rtol=1e-10)


def test_parton_events_are_physical():
    ev = wl.make_parton_events(200, seed=1).reshape(6, 4, -1)
    tot = ev.sum(axis=0)
    assert np.all(np.abs(tot[1]) < 1e-9) and np.all(np.abs(tot[2]) < 1e-9)
    for i in range(6):
        m2 = ev[i, 0] ** 2 - ev[i, 1] ** 2 - ev[i, 2] ** 2 - ev[i, 3] ** 2
        assert np.all(np.abs(m2) < 1e-6 * ev[i, 0] ** 2 + 1e-6)
    t = ev[0] + ev[1] + ev[3]
    mt = np.sqrt(t[0] ** 2 - t[1] ** 2 - t[2] ** 2 - t[3] ** 2)
    assert np.all(np.abs(mt - 173.0) < 15 * 1.4 + 1e-6)


def _record_from_partons(ev, e, swap=None):
    """config-3 record [lep (pT, eta, phi), (E, eta, phi) x {b_had, b_lep, q, qbar'}, met, met_phi] from a parton
    configuration with perfect jets (E_jet = E_parton); swap = (i, j) exchanges two jets of the record"""
    m = ev[:, e].reshape(6, 4)

    def pt_eta_phi(p):
        pt = math.hypot(p[1], p[2])
        return pt, math.asinh(p[3] / pt), math.atan2(p[2], p[1]) % (2 * math.pi)
    lep, nu = m[0], m[1]
    jets = [m[2], m[3], m[4], m[5]]
    if swap:
        jets[swap[0]], jets[swap[1]] = jets[swap[1]], jets[swap[0]]
    rec = list(pt_eta_phi(lep))
    for j in jets:
        _, eta, phi = pt_eta_phi(j)
        rec += [j[0], eta, phi]
    npt, _, nphi = pt_eta_phi(nu)
    return np.array(rec + [npt, nphi])


def test_closure_the_integrand_peaks_on_physical_events():
    """SURVEY.md 8(d) closure check: records built from on-shell t tbar configurations (perfect jets, MET
    azimuth = neutrino azimuth) give likelihoods orders of magnitude above those of records in which a b jet
    and a light jet are exchanged, and the true point (u = 1/3 for every jet: E = E_jet) is live."""
    ev = wl.make_parton_events(12, seed=31)
    p = oracle.params_default(3)
    ratios = []
    for e in range(12):
        good = _record_from_partons(ev, e)
        bad = _record_from_partons(ev, e, swap=(0, 2))          # b_had <-> q: wrong top and W masses
        pg, _ = oracle.integrate(3, p, good.reshape(17, 1), 6000, 5)
        pb, _ = oracle.integrate(3, p, bad.reshape(17, 1), 6000, 5)
        assert pg[0] > 0
        ratios.append(pg[0] / max(pb[0], 1e-300))
    assert np.median(ratios) > 30.0
    assert np.mean(np.array(ratios) > 1.0) >= 0.9
