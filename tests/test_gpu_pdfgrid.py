"""GPU parity of the grid PDFs (NEXT-3) against the CPU oracle."""
import numpy as np
import pytest

import oracle
from paper_1407_7595_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SEED = 20140729
G = wl.PDF_GRID


@pytest.fixture(scope="module")
def mem():
    import torch
    assert torch.cuda.is_available()
    import paper_1407_7595_b200 as m
    m.lib()
    return m


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _oracle_params(proc, table, Q, **kw):
    p = oracle.params_default(proc)
    for k, v in kw.items():
        setattr(p, k, v)
    return oracle.set_pdf_grid(p, table, G["lxmin"], G["lxmax"], G["lqmin"], G["lqmax"], Q)


def _table():
    # species-dependent normalisations and a ln Q slope: every table entry matters
    t = wl.make_pdf_table(A_g=1.3, A_q=0.8, q_slope=0.15)
    for s in range(1, 6):
        t[s] *= 1.0 + 0.1 * s
    return t


@pytest.mark.parametrize("proc,Q,n_flav", [(3, 173.0, 5), (3, 61.7, 3), (4, 400.0, 5)])
def test_per_point_with_grid_pdfs(mem, proc, Q, n_flav):
    """the cell index and the interpolation weights come from ln x on both sides; 1e-12 against the long-double
    referee at well-conditioned points (config-4 bar as in test_gpu_dilep.py)"""
    ne, n = 12, 2048 + 37
    ev = wl.make_events(proc, ne, seed=7)
    dev = _dev(ev)
    tab = _table()
    p = _oracle_params(proc, tab, Q, n_flav=n_flav)
    G_, O_, X_ = [], [], []
    with mem.Integrator(proc, n_flav=n_flav) as it:
        it.set_pdf_grid(tab, G["lxmin"], G["lxmax"], G["lqmin"], G["lqmax"], Q)
        for e in range(ne):
            G_.append(it.eval_points(dev, e, 3, n, SEED).cpu().numpy())
            O_.append(oracle.eval_points(proc, p, ev, e, 3, n, SEED))
            X_.append(oracle.eval_points_x(proc, p, ev, e, 3, n, SEED))
    wg, wo, wx = np.concatenate(G_), np.concatenate(O_), np.concatenate(X_)
    assert np.array_equal(wg == 0, wo == 0)
    nz = wo != 0
    assert nz.sum() > 1000
    eg = np.abs(wg[nz] - wx[nz]) / np.abs(wx[nz])
    eo = np.abs(wo[nz] - wx[nz]) / np.abs(wx[nz])
    if proc == 3:
        assert eg.max() <= 1e-12
    else:
        assert np.mean(eg <= 1e-12) >= 0.99 and eg.max() <= 1e-8 and np.mean(eg > 1e-12 + 4.0 * eo) <= 1e-3


def test_per_event_parton_and_toggle(mem):
    import torch
    proc, ne, n_points = 3, 6, (1 << 14) + 301
    ev = wl.make_events(proc, ne, seed=11)
    tab = _table()
    p = _oracle_params(proc, tab, 173.0)
    po, eo = oracle.integrate(proc, p, ev, n_points, SEED)
    toy = oracle.params_default(proc)
    pt, _ = oracle.integrate(proc, toy, ev, n_points, SEED)
    pe = wl.make_parton_events(2000, seed=4)
    wo = oracle.parton_weights(3, p, pe)
    with mem.Integrator(proc) as it:
        it.set_pdf_grid(tab, G["lxmin"], G["lxmax"], G["lqmin"], G["lqmax"], 173.0)
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        assert np.all(np.abs(pg.cpu().numpy() - po) <= 1e-9 * np.abs(po))
        assert np.all(np.abs(eg.cpu().numpy() - eo) <= 1e-9 * np.abs(eo))
        wg = it.eval_parton(_dev(pe)).cpu().numpy()
        assert np.max(np.abs(wg - wo) / wo) <= 1e-10
        it.set_pdf_grid(None)                                # back to the toy PDF
        pg2, _ = it.integrate(_dev(ev), n_points, SEED)
        assert np.all(np.abs(pg2.cpu().numpy() - pt) <= 1e-9 * np.abs(pt))
    # VEGAS and the assignment sum take the grid PDFs like any other integrand
    p.n_perm, p.vegas_iters, p.vegas_points = 4, 2, 6000
    po, _ = oracle.vegas_integrate(proc, p, ev[:, :3], 9000, SEED)
    with mem.Integrator(proc, n_perm=4, vegas_iters=2, vegas_points=6000) as it:
        it.set_pdf_grid(tab, G["lxmin"], G["lxmax"], G["lqmin"], G["lqmax"], 173.0)
        pg, _ = it.integrate(_dev(ev[:, :3]), 9000, SEED)
    assert np.all(np.abs(pg.cpu().numpy() - po) <= 1e-9 * np.abs(po))


def test_unsupported_and_invalid(mem):
    tab = _table()
    for proc in (1, 2):
        with mem.Integrator(proc) as it:
            with pytest.raises(mem.MemError) as ei:
                it.set_pdf_grid(tab, G["lxmin"], G["lxmax"], G["lqmin"], G["lqmax"], 100.0)
            assert ei.value.status == mem.MEM_ERR_UNSUPPORTED
    with mem.Integrator(3, precision=32) as it:
        with pytest.raises(mem.MemError):
            it.set_pdf_grid(tab, G["lxmin"], G["lxmax"], G["lqmin"], G["lqmax"], 100.0)
    with mem.Integrator(3) as it:
        for bad in (dict(lxmin=0.0, lxmax=-1.0), dict(Q=0.0)):
            kw = dict(lxmin=G["lxmin"], lxmax=G["lxmax"], lqmin=G["lqmin"], lqmax=G["lqmax"], Q=100.0)
            kw.update(bad)
            with pytest.raises(mem.MemError) as ei:
                it.set_pdf_grid(tab, **kw)
            assert ei.value.status == mem.MEM_ERR_INVALID_ARG
