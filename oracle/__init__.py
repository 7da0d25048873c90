"""ctypes front end of the CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports paper_1407_7595_b200.
All arithmetic lives in mem_oracle.cpp; this file only marshals arguments.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mem_oracle.cpp")
_HDR = os.path.join(_HERE, "mem_oracle.h")
_LIB = os.path.join(_HERE, "libmem_oracle.so")

W_ENU, Z_BB, TT_LJETS, TT_DILEP, TTH_DILEP = 1, 2, 3, 4, 5


def build(force: bool = False) -> str:
    """g++ -O2, no FMA contraction, platform libm (reading A16)."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(s) > os.path.getmtime(_LIB) for s in (_SRC, _HDR))
    if force or stale:
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Params(C.Structure):
    _fields_ = [(n, C.c_double) for n in (
        "sqrt_s", "G_F", "alpha_s", "sin2_thw", "m_W", "Gam_W", "m_Z", "Gam_Z", "m_t", "Gam_t",
        "V_ud", "V_tb", "pdf_A_q", "pdf_A_g", "pdf_pow_x", "pdf_pow_1mx",
        "tf_w_tail", "tf_mu1", "tf_sig1", "tf_mu2", "tf_sig2",
        "jetE_rlo", "jetE_rhi", "bw_nwidths", "nu_pz_max", "nu_eta_max", "met_sigma", "met_nsigma",
        "vegas_alpha")] + [("vegas_points", C.c_int64), ("vegas_iters", C.c_int32),
                           ("vegas_bins", C.c_int32), ("n_flav", C.c_int32), ("n_perm", C.c_int32),
                           ("pdf_mode", C.c_int32), ("pdf_nx", C.c_int32), ("pdf_nq", C.c_int32), ("pdf_pad", C.c_int32),
                           ("pdf_lxmin", C.c_double), ("pdf_lxmax", C.c_double), ("pdf_lqmin", C.c_double),
                           ("pdf_lqmax", C.c_double), ("pdf_Q", C.c_double), ("pdf_data", C.c_void_p),
                           ("m_H", C.c_double), ("Gam_H", C.c_double), ("yuk_t", C.c_double), ("yuk_b", C.c_double),
                           ("tth_hyp", C.c_int32), ("tth_chart", C.c_int32)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_params_default.argtypes = [C.c_int, C.POINTER(Params)]
        L.orc_n_fields.argtypes = [C.c_int]
        L.orc_n_dims.argtypes = [C.c_int]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.orc_philox4x32_10.restype = None
        L.orc_u52.argtypes = [C.c_uint32, C.c_uint32]
        L.orc_u52.restype = C.c_double
        L.orc_uniforms.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint32, C.c_int, _dp]
        L.orc_uniforms.restype = None
        L.orc_pdf_shape.argtypes = [C.POINTER(Params), C.c_double]
        L.orc_pdf_shape.restype = C.c_double
        L.orc_tf_jet.argtypes = [C.POINTER(Params), C.c_double, C.c_double]
        L.orc_tf_jet.restype = C.c_double
        L.orc_pdf_grid.argtypes = [C.POINTER(Params), C.c_int, C.c_double, C.c_double]
        L.orc_pdf_grid.restype = C.c_double
        L.orc_bw_window.argtypes = [C.c_double] * 4 + [_dp, _dp]
        L.orc_bw_window.restype = None
        L.orc_bw_point.argtypes = [C.c_double] * 3 + [_dp, _dp, _dp]
        L.orc_bw_point.restype = None
        L.orc_me_w.argtypes = [C.POINTER(Params)] + [_dp] * 4
        L.orc_me_w.restype = C.c_double
        L.orc_me_z.argtypes = [C.POINTER(Params), C.c_int] + [_dp] * 4
        L.orc_me_z.restype = C.c_double
        for f in (L.orc_me_tt_qq, L.orc_me_tt_gg):
            f.argtypes = [C.POINTER(Params)] + [_dp] * 4
            f.restype = C.c_double
        L.orc_me_top_decay.argtypes = [C.POINTER(Params), C.c_double] + [_dp] * 4
        L.orc_me_top_decay.restype = C.c_double
        L.orc_boost_transverse.argtypes = [_dp, C.c_int, _dp]
        L.orc_boost_transverse.restype = None
        L.orc_quartic_real_roots.argtypes = [_dp, _dp]
        L.orc_dilep_solve.argtypes = [_dp] * 4 + [C.c_double] * 6 + [_dp, _dp]
        L.orc_eq9_roots.argtypes = [C.c_double] * 3 + [_dp, _dp, _dp]
        L.orc_tth_radiator.argtypes = [C.POINTER(Params)] + [_dp] * 3
        L.orc_tth_radiator.restype = C.c_double
        L.orc_tth_decay.argtypes = [C.POINTER(Params), C.c_double]
        L.orc_tth_decay.restype = C.c_double
        L.orc_tth_tt_invariants.argtypes = [C.POINTER(Params)] + [_dp] * 4 + [C.POINTER(C.c_double)] * 3
        for f in (L.orc_me_tt_gg_inv, L.orc_me_tt_qq_inv):
            f.argtypes = [C.POINTER(Params)] + [C.c_double] * 3
            f.restype = C.c_double
        L.orc_tt_flavour_sum.argtypes = [C.POINTER(Params)] + [C.c_double] * 4
        L.orc_tt_flavour_sum.restype = C.c_double
        L.orc_me_top_decay_D.argtypes = [C.POINTER(Params), C.c_double] + [_dp] * 4 + [C.c_double]
        L.orc_me_top_decay_D.restype = C.c_double
        L.orc_normalisation.argtypes = [_dp, _dp, C.c_int64]
        L.orc_normalisation.restype = C.c_double
        L.orc_discriminant.argtypes = [_dp, _dp, C.c_int64, C.c_double, C.c_double, _dp]
        L.orc_discriminant.restype = None
        L.orc_parton_weights.argtypes = [C.c_int, C.POINTER(Params), _dp, C.c_int64, C.c_int, _dp]
        L.orc_weight.argtypes = [C.c_int, C.POINTER(Params), _dp, _dp, _dp]
        L.orc_weight.restype = C.c_double
        L.orc_eval_points.argtypes = [C.c_int, C.POINTER(Params), _dp, C.c_int64, C.c_int64, C.c_uint64,
                                      C.c_int64, C.c_int64, C.c_uint64, C.c_int32, _dp, _dp]
        L.orc_weight_x.argtypes = [C.c_int, C.POINTER(Params), _dp, _dp]
        L.orc_weight_x.restype = C.c_double
        L.orc_eval_points_x.argtypes = [C.c_int, C.POINTER(Params), _dp, C.c_int64, C.c_int64, C.c_uint64,
                                        C.c_int64, C.c_int64, C.c_uint64, C.c_int32, _dp, _dp]
        L.orc_integrate.argtypes = [C.c_int, C.POINTER(Params), _dp, C.c_int64, C.c_uint64, C.c_int64,
                                    C.c_uint64, _dp, _dp]
        L.orc_vegas_map.argtypes = [_dp, C.c_int, C.c_int, _dp, _dp, C.POINTER(C.c_int), _dp]
        L.orc_vegas_map.restype = None
        L.orc_vegas_refine.argtypes = [_dp, _dp, C.c_int, C.c_double]
        L.orc_vegas_refine.restype = None
        L.orc_vegas_integrate.argtypes = [C.c_int, C.POINTER(Params), _dp, C.c_int64, C.c_uint64, C.c_int64,
                                          C.c_uint64, _dp, _dp, _dp]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def params_default(process: int) -> Params:
    p = Params()
    if lib().orc_params_default(process, C.byref(p)) != 0:
        raise ValueError("unknown process %r" % process)
    return p


def set_pdf_grid(p: Params, table, lxmin, lxmax, lqmin, lqmax, Q):
    """NEXT-3: switch p to grid PDFs.  table = float64 [6, NQ, NX]; the array is kept alive on p."""
    t = np.ascontiguousarray(table, dtype=np.float64)
    assert t.ndim == 3 and t.shape[0] == 6
    p._pdf_keepalive = t
    p.pdf_mode, p.pdf_nq, p.pdf_nx = 1, t.shape[1], t.shape[2]
    p.pdf_lxmin, p.pdf_lxmax, p.pdf_lqmin, p.pdf_lqmax, p.pdf_Q = lxmin, lxmax, lqmin, lqmax, Q
    p.pdf_data = t.ctypes.data
    return p


def pdf_grid(p, species, x, Q):
    return lib().orc_pdf_grid(C.byref(p), int(species), float(x), float(Q))


def n_fields(process):
    return lib().orc_n_fields(process)


def n_dims(process):
    return lib().orc_n_dims(process)


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def u52(a, b):
    return lib().orc_u52(a, b)


def uniforms(seed, event, point, iteration, n):
    u = np.empty(n, dtype=np.float64)
    lib().orc_uniforms(seed, event, point, iteration, n, _p(u))
    return u


def pdf_shape(p, x):
    return lib().orc_pdf_shape(C.byref(p), x)


def tf_jet(p, e_jet, e_parton):
    return lib().orc_tf_jet(C.byref(p), e_jet, e_parton)


def bw_window(m, gam, s_lo, s_hi):
    a, b = C.c_double(), C.c_double()
    lib().orc_bw_window(m, gam, s_lo, s_hi, C.byref(a), C.byref(b))
    return a.value, b.value


def bw_point(m, gam, t):
    a, b, c = C.c_double(), C.c_double(), C.c_double()
    lib().orc_bw_point(m, gam, t, C.byref(a), C.byref(b), C.byref(c))
    return a.value, b.value, c.value


def _v4(*vs):
    return [_f64(v) for v in vs]


def me_w(p, qa, qb, lep, nu):
    a = _v4(qa, qb, lep, nu)
    return lib().orc_me_w(C.byref(p), *[_p(x) for x in a])


def me_z(p, up_type, qa, qb, p1, p2):
    a = _v4(qa, qb, p1, p2)
    return lib().orc_me_z(C.byref(p), int(up_type), *[_p(x) for x in a])


def me_tt_qq(p, q1, q2, pt, ptb):
    a = _v4(q1, q2, pt, ptb)
    return lib().orc_me_tt_qq(C.byref(p), *[_p(x) for x in a])


def me_tt_gg(p, q1, q2, pt, ptb):
    a = _v4(q1, q2, pt, ptb)
    return lib().orc_me_tt_gg(C.byref(p), *[_p(x) for x in a])


def me_top_decay(p, n_c, pt, pb, pf_down, pf_up):
    a = _v4(pt, pb, pf_down, pf_up)
    return lib().orc_me_top_decay(C.byref(p), float(n_c), *[_p(x) for x in a])


def boost_transverse(P, mom):
    P = _f64(P)
    m = _f64(mom).copy()
    lib().orc_boost_transverse(_p(P), m.shape[0], _p(m))
    return m


def quartic_real_roots(coeffs_low_to_high):
    """real roots of q[0] + q[1] x + ... + q[4] x^4 (the oracle's Ferrari solver)"""
    q = _f64(coeffs_low_to_high)
    x = np.empty(4)
    n = lib().orc_quartic_real_roots(_p(q), _p(x))
    return x[:n].copy()


def dilep_solve(lp, b, lm, bb, sWp, st, sWm, stb, Sx, Sy):
    """all (nu, nubar) solutions of PAPER.md Eq. 8: returns (sol [n, 2, 4], jac [n])"""
    a = [_f64(v) for v in (lp, b, lm, bb)]
    sol, jac = np.empty(32), np.empty(4)
    n = lib().orc_dilep_solve(_p(a[0]), _p(a[1]), _p(a[2]), _p(a[3]), sWp, st, sWm, stb, Sx, Sy, _p(sol), _p(jac))
    return sol[:8 * n].reshape(n, 2, 4).copy(), jac[:n].copy()


def eq9_roots(K12, f, sH):
    """NEXT-4, Eq. 9 inverted: returns (E1 [n], E2 [n], jac) with n = 0 or 2"""
    e1, e2, j = np.empty(2), np.empty(2), C.c_double()
    n = lib().orc_eq9_roots(K12, f, sH, _p(e1), _p(e2), C.byref(j))
    return e1[:n].copy(), e2[:n].copy(), j.value


def tth_radiator(p, pt, ptb, k):
    a = _v4(pt, ptb, k)
    return lib().orc_tth_radiator(C.byref(p), *[_p(x) for x in a])


def tth_decay(p, sH):
    return lib().orc_tth_decay(C.byref(p), float(sH))


def tth_tt_invariants(p, q1, q2, pt, ptb):
    """(ok, tau1, tau2, rho) of the t tbar subsystem (reading A20)"""
    a = _v4(q1, q2, pt, ptb)
    t1, t2, rho = C.c_double(), C.c_double(), C.c_double()
    ok = lib().orc_tth_tt_invariants(C.byref(p), *[_p(x) for x in a], C.byref(t1), C.byref(t2), C.byref(rho))
    return bool(ok), t1.value, t2.value, rho.value


def me_tt_gg_inv(p, t1, t2, rho):
    return lib().orc_me_tt_gg_inv(C.byref(p), t1, t2, rho)


def me_tt_qq_inv(p, t1, t2, rho):
    return lib().orc_me_tt_qq_inv(C.byref(p), t1, t2, rho)


def tt_flavour_sum(p, x1, x2, me_gg, me_qq):
    return lib().orc_tt_flavour_sum(C.byref(p), x1, x2, me_gg, me_qq)


def me_top_decay_D(p, n_c, pt, pb, pf_down, pf_up, D_W):
    a = _v4(pt, pb, pf_down, pf_up)
    return lib().orc_me_top_decay_D(C.byref(p), float(n_c), *[_p(x) for x in a], float(D_W))


def normalisation(p_evt, g_evt):
    """reading A22: sigma = (1/n) sum_e p_e / g_e over events drawn from the density g"""
    a, b = _f64(p_evt), _f64(g_evt)
    return lib().orc_normalisation(_p(a), _p(b), a.shape[0])


def discriminant(p_sig, p_bkg, sigma_sig, sigma_bkg):
    """PAPER.md:143 Eq. 10 with the 1/sigma of Eq. 1"""
    a, b = _f64(p_sig), _f64(p_bkg)
    out = np.empty(a.shape[0])
    lib().orc_discriminant(_p(a), _p(b), a.shape[0], sigma_sig, sigma_bkg, _p(out))
    return out


def parton_weights(process, p, mom, extended=False):
    """NEXT-2: parton-level weights; mom = [24, n_events] (l, nu, b_had, b_lep, q, qbar')"""
    m = _f64(mom)
    out = np.empty(m.shape[1])
    if lib().orc_parton_weights(process, C.byref(p), _p(m), m.shape[1], int(extended), _p(out)) != 0:
        raise ValueError("orc_parton_weights failed")
    return out


def weight(process, p, rec, u, debug=False):
    rec, u = _f64(rec), _f64(u)
    if debug:
        dbg = np.zeros(1 + 8 * (2 + 4 * 8), dtype=np.float64)
        w = lib().orc_weight(process, C.byref(p), _p(rec), _p(u), _p(dbg))
        return w, dbg
    return lib().orc_weight(process, C.byref(p), _p(rec), _p(u), None)


def eval_points(process, p, events, event, first_point, n, seed, iteration=0, grid=None, event_offset=0):
    ev = _f64(events)
    out = np.empty(n, dtype=np.float64)
    g = None if grid is None else _f64(grid)
    rc = lib().orc_eval_points(process, C.byref(p), _p(ev), ev.shape[1], event, event_offset, first_point, n,
                               seed, iteration, None if g is None else _p(g), _p(out))
    if rc != 0:
        raise ValueError("orc_eval_points failed")
    return out


def weight_x(process, p, rec, u):
    """Extended-precision (long double) referee evaluation of the same algorithm."""
    rec, u = _f64(rec), _f64(u)
    return lib().orc_weight_x(process, C.byref(p), _p(rec), _p(u))


def eval_points_x(process, p, events, event, first_point, n, seed, iteration=0, event_offset=0, grid=None):
    ev = _f64(events)
    out = np.empty(n, dtype=np.float64)
    g = None if grid is None else _f64(grid)
    rc = lib().orc_eval_points_x(process, C.byref(p), _p(ev), ev.shape[1], event, event_offset, first_point, n,
                                 seed, iteration, None if g is None else _p(g), _p(out))
    if rc != 0:
        raise ValueError("orc_eval_points_x failed")
    return out


def integrate(process, p, events, n_points, seed, event_offset=0):
    ev = _f64(events)
    ne = ev.shape[1]
    op, oe = np.empty(ne), np.empty(ne)
    rc = lib().orc_integrate(process, C.byref(p), _p(ev), ne, event_offset, n_points, seed, _p(op), _p(oe))
    if rc != 0:
        raise ValueError("orc_integrate failed")
    return op, oe


def vegas_map(edges, u):
    e = _f64(edges)
    D, B1 = e.shape
    u = _f64(u)
    z = np.empty(D)
    k = (C.c_int * D)()
    jac = C.c_double()
    lib().orc_vegas_map(_p(e), B1 - 1, D, _p(u), _p(z), k, C.byref(jac))
    return z, np.array(list(k)), jac.value


def vegas_refine(hist, edges, alpha):
    h = _f64(hist)
    e = _f64(edges).copy()
    lib().orc_vegas_refine(_p(h), _p(e), h.shape[0], alpha)
    return e


def vegas_integrate(process, p, events, n_points, seed, event_offset=0, return_grid=False):
    ev = _f64(events)
    ne = ev.shape[1]
    D = n_dims(process)
    op, oe = np.empty(ne), np.empty(ne)
    grid = np.empty((ne, D, p.vegas_bins + 1))
    rc = lib().orc_vegas_integrate(process, C.byref(p), _p(ev), ne, event_offset, n_points, seed,
                                   _p(op), _p(oe), _p(grid))
    if rc != 0:
        raise ValueError("orc_vegas_integrate failed")
    return (op, oe, grid) if return_grid else (op, oe)
