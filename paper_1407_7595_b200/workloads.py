"""Seeded synthetic event generators shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no Philox, no matrix element, no
transfer function): it only draws event records with the shapes BASELINE.json's configs
state.  It stands in for the paper's MadGraph+Pythia samples
(PAPER.md:145), which are not available.  It imports neither the CUDA binding nor the
oracle.

Records are float64, SoA, field-major: shape [n_fields, n_events].
Only numpy.random.Generator(PCG64).random() is used (a stable stream); exponential and
normal variates are derived here by inversion / Box-Muller so that numpy version changes
cannot alter the events.
"""
from __future__ import annotations

import numpy as np

DEFAULT_SEED = 20140729

W_ENU, Z_BB, TT_LJETS, TT_DILEP, TTH_DILEP = 1, 2, 3, 4, 5
N_FIELDS = {W_ENU: 5, Z_BB: 6, TT_LJETS: 17, TT_DILEP: 14, TTH_DILEP: 18}
N_DIMS = {W_ENU: 1, Z_BB: 2, TT_LJETS: 6, TT_DILEP: 8, TTH_DILEP: 8}

# BASELINE.json:configs[0..3]: (process, n_events, n_points)
CONFIGS = {
    1: (W_ENU, 64, 1 << 16),
    2: (Z_BB, 1024, 1 << 18),
    3: (TT_LJETS, 4096, 1 << 20),
    4: (TT_DILEP, 16384, 1 << 18),
    # NEXT-4 (not a BASELINE config; sizes follow config 4): the paper's own benchmark shape
    6: (TTH_DILEP, 16384, 1 << 18),
}


def _rng(seed, process):
    return np.random.Generator(np.random.PCG64([int(seed), int(process)]))


def _exp(u, mean):
    return -mean * np.log1p(-u)


def _lepton(r, n):
    """lepton pT ~ Exp(40 GeV) + 20, eta ~ U(-2.5, 2.5), phi ~ U(0, 2 pi)  (configs[0])."""
    return 20.0 + _exp(r.random(n), 40.0), -2.5 + 5.0 * r.random(n), 2.0 * np.pi * r.random(n)


def _jet(r, n):
    """jet E ~ Exp(60) + 30 GeV, |eta| < 2.5, phi ~ U(0, 2 pi)  (configs[2])."""
    return 30.0 + _exp(r.random(n), 60.0), -2.5 + 5.0 * r.random(n), 2.0 * np.pi * r.random(n)


def make_events(process: int, n_events: int, seed: int = DEFAULT_SEED) -> np.ndarray:
    r = _rng(seed, process)
    n = int(n_events)
    if process == W_ENU:
        pt, eta, phi = _lepton(r, n)
        # PAPER.md:180 Eq. 11: MET = -(sum of visible transverse momenta)
        rows = [pt, eta, phi, -pt * np.cos(phi), -pt * np.sin(phi)]
    elif process == Z_BB:
        rows = [*_jet(r, n), *_jet(r, n)]
    elif process == TT_LJETS:
        rows = [*_lepton(r, n)]
        for _ in range(4):                       # b_had, b_lep, q, qbar'
            rows += [*_jet(r, n)]
        rows += [20.0 + _exp(r.random(n), 40.0), 2.0 * np.pi * r.random(n)]   # met, met_phi
    elif process == TT_DILEP:
        lp, lm = _lepton(r, n), _lepton(r, n)
        b, bb = _jet(r, n), _jet(r, n)
        vx = lp[0] * np.cos(lp[2]) + lm[0] * np.cos(lm[2])
        vy = lp[0] * np.sin(lp[2]) + lm[0] * np.sin(lm[2])
        for E, eta, phi in (b, bb):
            vx = vx + E / np.cosh(eta) * np.cos(phi)
            vy = vy + E / np.cosh(eta) * np.sin(phi)
        u1, u2 = r.random(n), r.random(n)
        rad = np.sqrt(-2.0 * np.log1p(-u1))      # Box-Muller
        rows = [*lp, *lm, *b, *bb, -vx + 10.0 * rad * np.cos(2 * np.pi * u2),
                -vy + 10.0 * rad * np.sin(2 * np.pi * u2)]
    elif process == TTH_DILEP:
        # two leptons and four b jets (b, bbar, b1, b2), i.i.d. like configs 3-4; no MET field (Eq. 11)
        rows = [*_lepton(r, n), *_lepton(r, n)]
        for _ in range(4):
            rows += [*_jet(r, n)]
    else:
        raise ValueError("unknown process %r" % (process,))
    ev = np.ascontiguousarray(np.stack(rows, axis=0), dtype=np.float64)
    assert ev.shape == (N_FIELDS[process], n)
    return ev


def event_density(process: int, ev: np.ndarray) -> np.ndarray:
    """Probability density g(X) of make_events' records with respect to the record's own coordinates
    (pT or E, eta, phi per object), for the importance-sampled normalisation sigma = <p/g> (DESIGN.md
    reading A22).  Implemented for the processes whose records are products of independent objects."""
    if process != TTH_DILEP:
        raise ValueError("event_density: process %r has correlated fields" % (process,))
    g = np.ones(ev.shape[1])
    for k in range(2):                                       # leptons: pT = 20 + Exp(40)
        g *= np.exp(-(ev[3 * k] - 20.0) / 40.0) / 40.0 / 5.0 / (2.0 * np.pi)
    for k in range(4):                                       # jets: E = 30 + Exp(60)
        g *= np.exp(-(ev[6 + 3 * k] - 30.0) / 60.0) / 60.0 / 5.0 / (2.0 * np.pi)
    return g


def shard_range(n_events: int, rank: int, world: int):
    """Contiguous event range of `rank`: events are independent units."""
    base, rem = divmod(int(n_events), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


# ------------------------------------------------------------------------------------------
# NEXT-2, parton-level mode (Table 2): fully specified partonic
# t tbar -> b l nu bbar q qbar' configurations.  Pure kinematics: Breit-Wigner distributed top and
# W masses, isotropic two-body decays, a longitudinal boost.  Stands in for the paper's MadGraph
# parton-level samples.
# ------------------------------------------------------------------------------------------
def _boost(p, b):
    """boost four-vectors p [4, n] by velocities b [3, n]"""
    b2 = np.sum(b * b, axis=0)
    g = 1.0 / np.sqrt(1.0 - b2)
    bp = np.sum(b * p[1:], axis=0)
    k = np.where(b2 > 0, (g - 1.0) * bp / np.where(b2 > 0, b2, 1.0), 0.0) + g * p[0]
    return np.concatenate([(g * (p[0] + bp))[None], p[1:] + k * b], axis=0)


def _two_body(r, P, m1, m2):
    """isotropic decay of P [4, n] into masses m1, m2 (arrays or scalars)"""
    n = P.shape[1]
    M2 = P[0] ** 2 - P[1] ** 2 - P[2] ** 2 - P[3] ** 2
    M = np.sqrt(M2)
    k = np.sqrt(np.maximum(0.0, (M2 - (m1 + m2) ** 2) * (M2 - (m1 - m2) ** 2))) / (2.0 * M)
    c = 2.0 * r.random(n) - 1.0
    ph = 2.0 * np.pi * r.random(n)
    s = np.sqrt(1.0 - c * c)
    d = np.stack([s * np.cos(ph), s * np.sin(ph), c])
    p1 = np.concatenate([np.sqrt(k * k + m1 * m1)[None], k * d])
    p2 = np.concatenate([np.sqrt(k * k + m2 * m2)[None], -k * d])
    b = P[1:] / P[0]
    return _boost(p1, b), _boost(p2, b)


def _breit_wigner(r, n, m, G, nwidths):
    lo, hi = np.arctan(((m - nwidths * G) ** 2 - m * m) / (m * G)), np.arctan(((m + nwidths * G) ** 2 - m * m) / (m * G))
    return np.sqrt(m * m + m * G * np.tan(lo + (hi - lo) * r.random(n)))


def make_parton_events(n_events: int, seed: int = DEFAULT_SEED, sqrt_s: float = 14000.0, m_t: float = 173.0,
                       Gam_t: float = 1.4, m_W: float = 80.4, Gam_W: float = 2.09) -> np.ndarray:
    """[24, n_events]: (E, px, py, pz) of l, nu, b_had, b_lep, q, qbar' with t = b_lep + l + nu and
    tbar = b_had + q + qbar'; sqrt(s-hat) = 2 m_t + 30 + Exp(150) GeV, rapidity of the pair U(-1.5, 1.5)."""
    r = np.random.Generator(np.random.PCG64([int(seed), 1407]))
    n = int(n_events)
    mt1, mt2 = _breit_wigner(r, n, m_t, Gam_t, 15.0), _breit_wigner(r, n, m_t, Gam_t, 15.0)
    mw1, mw2 = _breit_wigner(r, n, m_W, Gam_W, 15.0), _breit_wigner(r, n, m_W, Gam_W, 15.0)
    rs = 2.0 * m_t + 30.0 + _exp(r.random(n), 150.0)
    y = -1.5 + 3.0 * r.random(n)
    rs = np.minimum(rs, 0.9 * sqrt_s * np.exp(-np.abs(y)))          # keep x1, x2 below 1
    P = np.stack([rs * np.cosh(y), np.zeros(n), np.zeros(n), rs * np.sinh(y)])
    t, tb = _two_body(r, P, mt1, mt2)
    W1, b_lep = _two_body(r, t, mw1, np.zeros(n))
    lep, nu = _two_body(r, W1, np.zeros(n), np.zeros(n))
    W2, b_had = _two_body(r, tb, mw2, np.zeros(n))
    q, qb = _two_body(r, W2, np.zeros(n), np.zeros(n))
    ev = np.concatenate([lep, nu, b_had, b_lep, q, qb], axis=0)
    return np.ascontiguousarray(ev, dtype=np.float64)


def _smear_jet(r, E, w_tail=0.3, mu1=0.0, sig1=0.15, mu2=-0.1, sig2=0.35):
    """measured jet energy for parton energy E: a draw from the double-Gaussian shape BASELINE.json:configs[1]
    states (mixture of two normals in (E_jet - E)/E); pure sampling, the TF itself lives in the kernels"""
    n = E.shape[0]
    tail = r.random(n) < w_tail
    u1, u2 = r.random(n), r.random(n)
    g = np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)
    return E * (1.0 + np.where(tail, mu2 + sig2 * g, mu1 + sig1 * g))


def _eta_phi(p):
    pt = np.hypot(p[1], p[2])
    return np.arcsinh(p[3] / pt), np.mod(np.arctan2(p[2], p[1]), 2.0 * np.pi)


def make_tth_events(n_events: int, seed: int = DEFAULT_SEED, resonant: bool = True, smear: bool = True,
                    m_H: float = 125.0, m_t: float = 173.0, Gam_t: float = 1.4, m_W: float = 80.4,
                    Gam_W: float = 2.09, sqrt_s: float = 14000.0, return_truth: bool = False):
    """NEXT-4 closure sample, [18, n_events] records of MEM_PROC_TTH_DILEP built from physical
    t tbar (b bbar) kinematics: s-hat -> (t tbar)(bb) -> t, tbar, b1 b2 by isotropic two-body steps,
    Breit-Wigner top and W masses, dileptonic decays, jets smeared with the double Gaussian.
    resonant: m_bb = m_H (signal-like); otherwise m_bb log-uniform in [20, 300] GeV (background-like).
    Stands in for the paper's MadGraph+Pythia t tbar H / t tbar b bbar samples."""
    r = np.random.Generator(np.random.PCG64([int(seed), 1407, 9 if resonant else 10]))
    n = int(n_events)
    mt1, mt2 = _breit_wigner(r, n, m_t, Gam_t, 15.0), _breit_wigner(r, n, m_t, Gam_t, 15.0)
    mw1, mw2 = _breit_wigner(r, n, m_W, Gam_W, 15.0), _breit_wigner(r, n, m_W, Gam_W, 15.0)
    mbb = np.full(n, m_H) if resonant else 20.0 * np.exp(np.log(15.0) * r.random(n))
    mtt = mt1 + mt2 + 20.0 + _exp(r.random(n), 120.0)
    rs = mtt + mbb + 20.0 + _exp(r.random(n), 150.0)
    y = -1.5 + 3.0 * r.random(n)
    rs = np.minimum(rs, 0.9 * sqrt_s * np.exp(-np.abs(y)))
    P = np.stack([rs * np.cosh(y), np.zeros(n), np.zeros(n), rs * np.sinh(y)])
    TT, H = _two_body(r, P, mtt, mbb)
    t, tb = _two_body(r, TT, mt1, mt2)
    W1, b = _two_body(r, t, mw1, np.zeros(n))
    lp, nu = _two_body(r, W1, np.zeros(n), np.zeros(n))
    W2, bb = _two_body(r, tb, mw2, np.zeros(n))
    lm, nub = _two_body(r, W2, np.zeros(n), np.zeros(n))
    b1, b2 = _two_body(r, H, np.zeros(n), np.zeros(n))
    rows = []
    for l in (lp, lm):
        eta, phi = _eta_phi(l)
        rows += [np.hypot(l[1], l[2]), eta, phi]
    for j in (b, bb, b1, b2):
        eta, phi = _eta_phi(j)
        rows += [_smear_jet(r, j[0]) if smear else j[0].copy(), eta, phi]
    ev = np.ascontiguousarray(np.stack(rows, axis=0), dtype=np.float64)
    if return_truth:
        return ev, dict(lp=lp, nu=nu, b=b, lm=lm, nub=nub, bb=bb, b1=b1, b2=b2)
    return ev


# ------------------------------------------------------------------------------------------
# NEXT-3, grid PDFs: the paper fills per-flavour (x, Q) tables by querying
# LHAPDF / CTEQ, which are not available; these tables are synthesised from BASELINE's toy shape
# A x^a (1-x)^b (times a mild, made-up ln Q slope so that the Q interpolation is exercised) and
# stand in for them.  Sample i sits at min + i (max - min) / N, the listing's convention.
# ------------------------------------------------------------------------------------------
PDF_GRID = dict(nx=256, nq=16, lxmin=float(np.log(1e-6)), lxmax=0.0, lqmin=float(np.log(10.0)),
                lqmax=float(np.log(1000.0)))


def make_pdf_table(A_g: float = 1.0, A_q: float = 1.0, pow_x: float = -0.5, pow_1mx: float = 3.0,
                   q_slope: float = 0.0, Q0: float = 173.0, **grid) -> np.ndarray:
    """float64 [6, NQ, NX]: species 0 = gluon, 1..5 = d, u, s, c, b."""
    g = dict(PDF_GRID, **grid)
    lx = g["lxmin"] + (g["lxmax"] - g["lxmin"]) / g["nx"] * np.arange(g["nx"])
    lq = g["lqmin"] + (g["lqmax"] - g["lqmin"]) / g["nq"] * np.arange(g["nq"])
    x = np.exp(lx)
    shape = x ** pow_x * (1.0 - x) ** pow_1mx
    qfac = 1.0 + q_slope * (lq - np.log(Q0))
    tab = np.empty((6, g["nq"], g["nx"]))
    for s in range(6):
        tab[s] = (A_g if s == 0 else A_q) * qfac[:, None] * shape[None, :]
    return tab
