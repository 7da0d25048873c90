"""Test-side helpers: explicit Dirac algebra and 2->2 kinematics (numpy only).

Independent of both the oracle and the CUDA path: used to pin the oracle's matrix
elements against explicit traces and textbook closed forms.
"""
import numpy as np

I2 = np.eye(2, dtype=complex)
Z2 = np.zeros((2, 2), dtype=complex)
SIG = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]], dtype=complex),
       np.array([[1, 0], [0, -1]], dtype=complex)]
G = [np.block([[I2, Z2], [Z2, -I2]])] + [np.block([[Z2, s], [-s, Z2]]) for s in SIG]   # Dirac rep
G5 = 1j * G[0] @ G[1] @ G[2] @ G[3]
PL = 0.5 * (np.eye(4) - G5)
PR = 0.5 * (np.eye(4) + G5)
METRIC = np.diag([1.0, -1.0, -1.0, -1.0])


def slash(p):
    return G[0] * p[0] - G[1] * p[1] - G[2] * p[2] - G[3] * p[3]


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def lorentz_contract(A, B):
    """sum_{mu,nu} A[mu][nu] B_{mu nu} for rank-2 tensors given with upper indices."""
    tot = 0.0
    for mu in range(4):
        for nu in range(4):
            tot += A[mu][nu] * B[mu][nu] * METRIC[mu, mu] * METRIC[nu, nu]
    return tot


def massless(E, cth, phi):
    sth = np.sqrt(max(0.0, 1.0 - cth * cth))
    return np.array([E, E * sth * np.cos(phi), E * sth * np.sin(phi), E * cth])


def random_massless(rng, scale=100.0):
    return massless(scale * (0.2 + rng.random()), 2 * rng.random() - 1, 2 * np.pi * rng.random())


def boost(p, b):
    """boost four-vector p by velocity vector b."""
    b = np.asarray(b, dtype=float)
    b2 = b @ b
    if b2 == 0:
        return np.array(p, dtype=float)
    g = 1.0 / np.sqrt(1.0 - b2)
    bp = b @ p[1:]
    out = np.empty(4)
    out[0] = g * (p[0] + bp)
    out[1:] = p[1:] + ((g - 1.0) * bp / b2 + g * p[0]) * b
    return out


def two_body_decay(P, m1, m2, cth, phi):
    """decay of four-momentum P into masses m1, m2 with rest-frame angles (cth, phi)."""
    M = np.sqrt(mdot(P, P))
    k = np.sqrt(max(0.0, (M * M - (m1 + m2) ** 2) * (M * M - (m1 - m2) ** 2))) / (2 * M)
    sth = np.sqrt(max(0.0, 1 - cth * cth))
    n = np.array([sth * np.cos(phi), sth * np.sin(phi), cth])
    p1 = np.concatenate([[np.sqrt(k * k + m1 * m1)], k * n])
    p2 = np.concatenate([[np.sqrt(k * k + m2 * m2)], -k * n])
    b = P[1:] / P[0]
    return boost(p1, b), boost(p2, b)


# ----------------------------------------------------------------------------------------------
# Parity bars of the processes that solve the two-conic neutrino system (config 4, NEXT-4).
# next to a tangency of the conics two solutions merge; whether they
# exist is decided by the sign of a Ferrari discriminant computed from resultant coefficients that have
# lost 6-8 digits to cancellation ("cancellation of large coefficients"), so about one live
# point in 1e5 is decided differently by ANY two fp64 evaluations (the fp64 oracle against its own
# long-double referee included), and such a point can carry 1e-5 of an event's integral.
# ----------------------------------------------------------------------------------------------
def conic_ill_conditioned(ev, first_jet=6, n_jets=2, threshold=0.02):
    """Per event: True when some lepton-jet pair has |tanh(eta_l) - tanh(eta_b)| below the threshold.  The neutrino's
    z component is eliminated through the plane (n_l - n_b).nu = kappa by dividing by exactly that difference
    (SURVEY.md 8(c) "Config 4"), so for such a record the conics' coefficients are ~1/d_z^2 large, most solutions
    come in nearly coincident pairs and their existence is decided by rounding far more often than elsewhere."""
    ev = np.asarray(ev)
    bad = np.zeros(ev.shape[1], dtype=bool)
    for l in range(2):
        for j in range(n_jets):
            bad |= np.abs(np.tanh(ev[3 * l + 1]) - np.tanh(ev[first_jet + 3 * j + 1])) < threshold
    return bad


def check_points_conic(wg, wo, wx, min_live):
    """per-point bar: wg = CUDA path, wo = fp64 oracle, wx = long-double referee"""
    live = (wo != 0.0) | (wx != 0.0) | (wg != 0.0)
    assert live.sum() >= min_live, live.sum()
    flips = (wg == 0.0) != (wo == 0.0)
    # the zero pattern may differ only at isolated near-tangent points ...
    assert flips.sum() <= max(2, 2e-4 * live.sum()), (flips.sum(), live.sum())
    # ... and there at least one of the two fp64 evaluations sides with the referee
    for i in np.flatnonzero(flips):
        assert (wg[i] == 0.0) == (wx[i] == 0.0) or (wo[i] == 0.0) == (wx[i] == 0.0)
    nz = (wo != 0.0) & (wg != 0.0) & (wx != 0.0)
    ref = np.abs(wx[nz])
    eg = np.abs(wg[nz] - wx[nz]) / ref
    eo = np.abs(wo[nz] - wx[nz]) / ref
    assert np.mean(eg <= 1e-12) >= 0.99, np.mean(eg <= 1e-12)
    assert np.mean(eg > 1e-12 + 4.0 * eo) <= 1e-3
    assert eg.max() <= 1e-8
    assert np.percentile(eg, 99.9) <= 2.0 * np.percentile(eo, 99.9) + 1e-12


def check_events_conic(pg, eg, po, eo, drill, n_points, ill=None):
    """per-event bar: 1e-9 on the mean and on the standard error.  An event that misses it is taken apart:
    drill(e) -> (wg, wo, wx), the per-point weights of the three evaluations; the miss must be carried by a
    few isolated points (at most max(2, 2e-4 of the live ones); 1e-2 for a record flagged by conic_ill_conditioned)
    at each of which one of the two fp64 evaluations sides with the referee, and the sums over all other points
    must agree to 1e-9."""
    assert np.array_equal(pg == 0.0, po == 0.0)
    miss = np.flatnonzero(~(np.abs(pg - po) <= 1e-9 * np.abs(po)) | ~(np.abs(eg - eo) <= 1e-9 * np.abs(eo) + 1e-300))
    assert len(miss) <= max(1, 0.15 * len(pg)), (len(miss), len(pg))
    for e in miss:
        # never beyond a small fraction of the statistical error
        assert abs(pg[e] - po[e]) <= 0.05 * eo[e], (e, pg[e], po[e], eo[e])
        wg, wo, wx = drill(int(e))
        live = (wo != 0.0) | (wg != 0.0)
        # the K points with the largest |w_gpu - w_orc| carry the miss
        K = int(max(2, (1e-2 if (ill is not None and ill[e]) else 2e-4) * live.sum()))
        d = np.abs(wg - wo)
        off = np.zeros(len(d), dtype=bool)
        off[np.argsort(d)[-K:]] = True
        off &= d > 1e-9 * np.abs(wo)
        assert off.sum() >= 1, e
        for i in np.flatnonzero(off):
            # the CUDA path is within the per-point cap of the referee, or it is a root-count flip of the CUDA
            # path at a point where the fp64 oracle sides with the referee
            assert abs(wg[i] - wx[i]) <= 1e-8 * abs(wx[i]) or abs(wo[i] - wx[i]) <= 1e-9 * abs(wx[i]), (e, i, wg[i], wo[i], wx[i])
        sg, so = np.sum(wg[~off]), np.sum(wo[~off])
        assert abs(sg - so) <= 1e-9 * abs(so), (e, sg, so, off.sum())
        # and the CUDA path's integral is the sum of the weights it reports
        assert abs(np.sum(wg) / n_points - pg[e]) <= 1e-9 * abs(pg[e])
