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
# lost 6-8 digits to cancellation ("cancellation of large coefficients").
#
# Round 3: every number below is the round-1 bar again or a measured value (profiles/r03_conic_parity.md, taken on the
# kernels of this round with every call of these helpers instrumented): on all per-point test sets the zero pattern of
# the CUDA path is identical to the oracle's and to the referee's; every config-4 event of every test meets 1e-9; the
# only events that miss it are 2 of 32 NEXT-4 records (both flagged by conic_ill_conditioned) and 1 of 24 config-4
# records under the two-assignment sum.  So the default is strict, and a test that needs an allowance names it.
# ----------------------------------------------------------------------------------------------
def _record(**fields):
    """With MEM_CONIC_STATS=<file> in the environment every call of the two checks below appends what it measured
    (one JSON object per line) before asserting anything: the source of profiles/r03_conic_parity.md."""
    import json
    import os
    path = os.environ.get("MEM_CONIC_STATS")
    if path:
        fields["test"] = os.environ.get("PYTEST_CURRENT_TEST", "").split(" ")[0]
        with open(path, "a") as f:
            f.write(json.dumps(fields) + "\n")


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
    """per-point bar (round 1's, with the cap at the measured level): wg = CUDA path, wo = fp64 oracle,
    wx = long-double referee.
      A  identical zero pattern: the same points have no solution / fail the cuts
      B  |w_gpu - w_ref| <= 1e-12 |w_ref| at >= 99 % of the live points (measured >= 99.7 %; the fp64 oracle itself
         departs from its referee by more than 1e-12 at ~0.3 % of them)
      C  |w_gpu - w_ref| <= 1e-12 |w_ref| + 4 |w_orc - w_ref| except at <= 0.1 % of the live points (measured
         <= 0.09 %), and never beyond 1e-10 (measured 4.4e-11; the oracle's own worst point: 2.9e-10)
      D  the 99.9th percentile of the CUDA path's error is not larger than twice the oracle's"""
    both = (wo != 0.0) & (wg != 0.0) & (wx != 0.0)
    rg, ro = np.abs(wg[both] - wx[both]) / np.abs(wx[both]), np.abs(wo[both] - wx[both]) / np.abs(wx[both])
    _record(kind="points", live=int(((wo != 0.0) | (wg != 0.0) | (wx != 0.0)).sum()),
            flips_gpu_orc=int(((wg == 0.0) != (wo == 0.0)).sum()), flips_gpu_ref=int(((wg == 0.0) != (wx == 0.0)).sum()),
            flips_orc_ref=int(((wo == 0.0) != (wx == 0.0)).sum()),
            gpu_within_1e12=float(np.mean(rg <= 1e-12)), orc_within_1e12=float(np.mean(ro <= 1e-12)),
            gpu_beyond_1e12_plus_4orc=float(np.mean(rg > 1e-12 + 4.0 * ro)), gpu_max=float(rg.max()), orc_max=float(ro.max()),
            gpu_p999=float(np.percentile(rg, 99.9)), orc_p999=float(np.percentile(ro, 99.9)))
    assert np.array_equal(wg == 0.0, wo == 0.0), ("zero pattern differs", int(((wg == 0.0) != (wo == 0.0)).sum()))
    nz = wo != 0.0
    assert nz.sum() >= min_live, nz.sum()
    assert np.all(np.isfinite(wg))
    # a point the referee decides differently from both fp64 evaluations is compared on the others
    nz &= wx != 0.0
    assert (wo != 0.0).sum() - nz.sum() <= max(2, 2e-4 * nz.sum())
    ref = np.abs(wx[nz])
    eg = np.abs(wg[nz] - wx[nz]) / ref
    eo = np.abs(wo[nz] - wx[nz]) / ref
    assert np.mean(eg <= 1e-12) >= 0.99, np.mean(eg <= 1e-12)
    assert np.mean(eg > 1e-12 + 4.0 * eo) <= 1e-3
    assert eg.max() <= 1e-10, eg.max()
    assert np.percentile(eg, 99.9) <= 2.0 * np.percentile(eo, 99.9) + 1e-12


def check_events_conic(pg, eg, po, eo, drill, n_points, ill=None, max_miss=0):
    """per-event bar: 1e-9 on the mean and on the standard error of EVERY event (max_miss = 0, the default).

    max_miss > 0 is for the few tests whose records are known to miss it (the measured count, stated at the call):
    at most that many events may, and each of them is taken apart.  drill(e) -> (wg, wo, wx), the per-point weights
    of the CUDA path, the fp64 oracle and the long-double referee:
      - the miss stays below 2e-3 of the event's statistical error (measured: 7.8e-4 at worst);
      - it is carried by a few isolated points: at most max(2, 2e-4 of the live ones), 1e-2 for a record flagged by
        conic_ill_conditioned (measured: 1 of 14375; 11 of 2998 on a flagged record);
      - at each of them one of the two fp64 evaluations agrees with the referee, the CUDA path's value is finite and
        not negative (every solution's weight is >= 0: a dropped or an extra pair of merging solutions moves w, it
        cannot change its sign), and the CUDA path is wrong against the referee no more often than the oracle + 2;
      - all the other points sum to the same integral within 1e-9, and the CUDA path's integral is the sum of the
        weights it reports."""
    assert np.array_equal(pg == 0.0, po == 0.0)
    miss = np.flatnonzero(~(np.abs(pg - po) <= 1e-9 * np.abs(po)) | ~(np.abs(eg - eo) <= 1e-9 * np.abs(eo) + 1e-300))
    _record(kind="events", n_events=int(len(pg)), n_points=int(n_points), beyond_1e9=int(len(miss)), max_miss=int(max_miss))
    assert len(miss) <= max_miss, (len(miss), len(pg), [(int(e), pg[e], po[e]) for e in miss])
    for e in miss:
        wg, wo, wx = drill(int(e))
        live = (wo != 0.0) | (wg != 0.0)
        K = int(max(2, (1e-2 if (ill is not None and ill[e]) else 2e-4) * live.sum()))
        off = np.abs(wg - wo) > 1e-9 * np.abs(wo)
        _record(kind="miss", event=int(e), flagged=bool(ill is not None and ill[e]), rel=float(abs(pg[e] - po[e]) / abs(po[e])),
                over_sigma=float(abs(pg[e] - po[e]) / eo[e]), live=int(live.sum()), off=int(off.sum()),
                off_zero_flips=int(((wg[off] == 0.0) != (wo[off] == 0.0)).sum()),
                off_gpu_within_1e8_of_ref=int((np.abs(wg[off] - wx[off]) <= 1e-8 * np.abs(wx[off])).sum()),
                off_orc_within_1e9_of_ref=int((np.abs(wo[off] - wx[off]) <= 1e-9 * np.abs(wx[off])).sum()))
        assert abs(pg[e] - po[e]) <= 2e-3 * eo[e], (e, pg[e], po[e], eo[e])
        assert 1 <= off.sum() <= K, (e, off.sum(), K)
        gpu_bad = orc_bad = 0
        for i in np.flatnonzero(off):
            g_ok = abs(wg[i] - wx[i]) <= 1e-8 * abs(wx[i])
            o_ok = abs(wo[i] - wx[i]) <= 1e-9 * abs(wx[i])
            assert g_ok or o_ok, (e, i, wg[i], wo[i], wx[i])
            assert np.isfinite(wg[i]) and wg[i] >= 0.0, (e, i, wg[i])
            gpu_bad += not g_ok
            orc_bad += not o_ok
        assert gpu_bad <= orc_bad + 2, (e, gpu_bad, orc_bad)
        sg, so = np.sum(wg[~off]), np.sum(wo[~off])
        assert abs(sg - so) <= 1e-9 * abs(so), (e, sg, so, off.sum())
        assert abs(np.sum(wg) / n_points - pg[e]) <= 1e-9 * abs(pg[e])
