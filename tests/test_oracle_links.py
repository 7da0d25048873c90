"""Absolute-normalisation pins of the assembled config-3 and config-4 weights ("parity unpinned: the
constant factors of weight_tt_ljets and weight_tt_dilep").

The complete t tbar matrix element with PDFs and flux is pinned on its own by the narrow-width closure of
oracle.parton_weights (tests/test_oracle_parton.py: sigma-hat(gg -> t tbar) x Gamma x Gamma).  Here each assembled
weight is rebuilt in the test from that pinned function, the pinned building blocks (Breit-Wigner map, jet TF,
dilep_solve with its Jacobian) and the measure typed out from PAPER.md:49 Eq. 2 and :105 Eq. 7:
every final particle d^3y/((2 pi)^3 2E), overall (2 pi)^4, delta(E) delta(p_z) -> 2/s; a jet with delta TFs in
direction contributes E sin(theta) dE / (2 (2 pi)^3).  A dropped 1/2, a (2 pi)^3 -> (2 pi)^2, a missing sin(theta)
or colour factor in the oracle's own copy of these constants fails here.
"""
import numpy as np
import pytest

import oracle
from paper_1407_7595_b200 import workloads as wl

TWOPI = 2.0 * np.pi


def _dir(eta, phi):
    return np.array([1.0, np.cos(phi) / np.cosh(eta), np.sin(phi) / np.cosh(eta), np.tanh(eta)])


def _from_pt(pt, eta, phi):
    return pt * np.array([np.cosh(eta), np.cos(phi), np.sin(phi), np.sinh(eta)])


def _live(proc, p, ev, n, seed=17):
    out = []
    for e in range(ev.shape[1]):
        got = 0
        for i in range(4000):
            u = oracle.uniforms(seed, e, i, 0, oracle.n_dims(proc))
            w = oracle.weight(proc, p, ev[:, e], u)
            if w != 0.0:
                out.append((ev[:, e], u, w))
                got += 1
                if got >= n:
                    break
    return out


def _bw(p, m, G, u):
    lo, hi = oracle.bw_window(m, G, (m - p.bw_nwidths * G) ** 2, (m + p.bw_nwidths * G) ** 2)
    smm, dsdt, D = oracle.bw_point(m, G, lo + (hi - lo) * u)
    return m * m + smm, (hi - lo) * dsdt, D


def test_config3_weight_is_measure_times_the_closure_pinned_parton_weight():
    proc = oracle.TT_LJETS
    p = oracle.params_default(proc)
    ev = wl.make_events(proc, 8, seed=5)
    pts = _live(proc, p, ev, 3)
    assert len(pts) >= 18
    for rec, u, w in pts:
        rlo, dr, H = p.jetE_rlo, p.jetE_rhi - p.jetE_rlo, p.nu_eta_max
        lep = _from_pt(*rec[0:3])
        jets, fac = [], 1.0
        for j in range(4):                                   # b_had, b_lep, q, qbar'
            Ej, eta, phi = rec[3 + 3 * j:6 + 3 * j]
            E = Ej * (rlo + dr * u[j])
            fac *= Ej * dr                                    # dE = E_jet dr du
            fac *= oracle.tf_jet(p, Ej, E)                    # T(E_jet; E)
            fac *= E * (1 / np.cosh(eta)) / (2 * TWOPI ** 3)  # E^2 sin(theta) dE / ((2 pi)^3 2E)
            jets.append(E * _dir(eta, phi))
        eta_nu = -H + 2 * H * u[4]
        fac *= 2 * H
        sW, jac_bw, _ = _bw(p, p.m_W, p.Gam_W, u[5])
        fac *= jac_bw
        met_phi = rec[16]
        nuT = sW / (2 * rec[0] * (np.cosh(rec[1] - eta_nu) - np.cos(rec[2] - met_phi)))
        nu = _from_pt(nuT, eta_nu, met_phi)
        assert (lep + nu) @ np.diag([1, -1, -1, -1]) @ (lep + nu) == pytest.approx(sW, rel=1e-12)
        fac *= 1 / (2 * lep[0] * TWOPI ** 3)                  # lepton, delta TF
        fac *= nuT ** 2 / (2 * sW * TWOPI ** 3)               # d^3nu/((2pi)^3 2E) = nu_T^2/(2 s_W (2pi)^3) ds_W d eta d phi
        fac *= TWOPI ** 4 * 2 / p.sqrt_s ** 2                 # (2 pi)^4, delta(E) delta(p_z) dx1 dx2 -> 2/s
        mom = np.concatenate([lep, nu, jets[0], jets[1], jets[2], jets[3]])[:, None]   # l, nu, b_had, b_lep, q, qbar'
        pw = oracle.parton_weights(proc, p, mom)[0]
        assert pw > 0
        # the parton weight takes the leptonic W propagator from the momenta, the config-3 weight from the mapped variable
        assert fac * pw == pytest.approx(w, rel=1e-8)


def test_config4_weight_is_measure_times_the_closure_pinned_parton_weight():
    proc = oracle.TT_DILEP
    p = oracle.params_default(proc)
    ev = wl.make_events(proc, 40, seed=6)
    pts = _live(proc, p, ev, 3)
    assert len(pts) >= 18
    p3 = oracle.params_default(oracle.TT_LJETS)
    for rec, u, w in pts:
        rlo, dr = p.jetE_rlo, p.jetE_rhi - p.jetE_rlo
        lp, lm = _from_pt(*rec[0:3]), _from_pt(*rec[3:6])
        jets, fac = [], 1.0
        for j in range(2):                                   # b, bbar
            Ej, eta, phi = rec[6 + 3 * j:9 + 3 * j]
            E = Ej * (rlo + dr * u[j])
            fac *= Ej * dr * oracle.tf_jet(p, Ej, E) * E * (1 / np.cosh(eta)) / (2 * TWOPI ** 3)
            jets.append(E * _dir(eta, phi))
        s = []
        for k, (m, G) in enumerate(((p.m_W, p.Gam_W), (p.m_t, p.Gam_t), (p.m_W, p.Gam_W), (p.m_t, p.Gam_t))):
            sk, jac_bw, _ = _bw(p, m, G, u[2 + k])
            s.append(sk)
            fac *= jac_bw
        span = p.met_sigma * p.met_nsigma
        Sx, Sy = rec[12] + span * (2 * u[6] - 1), rec[13] + span * (2 * u[7] - 1)
        fac *= (2 * span) ** 2
        fac *= np.exp(-((rec[12] - Sx) ** 2 + (rec[13] - Sy) ** 2) / (2 * p.met_sigma ** 2)) / (TWOPI * p.met_sigma ** 2)
        fac *= 1 / (2 * lp[0] * TWOPI ** 3) / (2 * lm[0] * TWOPI ** 3)
        fac *= TWOPI ** 4 * 2 / p.sqrt_s ** 2
        sols, jacs = oracle.dilep_solve(lp, jets[0], lm, jets[1], s[0], s[1], s[2], s[3], Sx, Sy)
        tot = 0.0
        for (nu, nub), J in zip(sols, jacs):
            # d^3nu d^3nubar / ((2pi)^6 4 E E') = J d(s_W+, s_t, s_W-, s_tbar, S_x, S_y) / ((2pi)^6 4 E E')
            meas = J / (TWOPI ** 6 * 4 * nu[0] * nub[0])
            # l+jets topology with (q, qbar') = (l-, nubar) has the hadronic colour factor 3 and |V_ud|^2 = 1
            mom = np.concatenate([lp, nu, jets[1], jets[0], lm, nub])[:, None]    # l, nu, b_had = bbar, b_lep = b, q, qbar'
            tot += meas * oracle.parton_weights(oracle.TT_LJETS, p3, mom)[0] / 3.0
        # propagators from reconstructed momenta (parton weight) against mapped variables (config 4): a few 1e-9
        assert fac * tot == pytest.approx(w, rel=1e-6)
