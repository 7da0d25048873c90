"""GPU parity of the jet-permutation sum (NEXT-1; Eq. 7) against the CPU oracle."""
import numpy as np
import pytest

import oracle
from helpers import check_events_conic, conic_ill_conditioned
from paper_1407_7595_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SEED = 20140729


@pytest.fixture(scope="module")
def mem():
    import torch
    assert torch.cuda.is_available()
    import paper_1407_7595_b200 as m
    m.lib()
    return m


def _dev(ev):
    import torch
    return torch.from_numpy(np.ascontiguousarray(ev)).cuda()


@pytest.mark.parametrize("n_perm", [1, 4, 24])
def test_config3_per_point(mem, n_perm):
    """same bar as the single-assignment kernel: 1e-12 against the long-double referee, 1e-12 plus the
    fp64 oracle's own rounding error against the oracle, identical zero pattern"""
    proc, ne, n = 3, 10, 2048 + 37
    ev = wl.make_events(proc, ne, seed=7)
    dev = _dev(ev)
    p = oracle.params_default(proc)
    p.n_perm = n_perm
    worst = 0.0
    with mem.Integrator(proc, n_perm=n_perm) as it:
        for e in range(ne):
            wg = it.eval_points(dev, e, 5, n, SEED).cpu().numpy()
            wo = oracle.eval_points(proc, p, ev, e, 5, n, SEED)
            wx = oracle.eval_points_x(proc, p, ev, e, 5, n, SEED)
            assert np.array_equal(wg == 0.0, wo == 0.0)
            nz = wo != 0.0
            rel = np.abs(wg[nz] - wx[nz]) / np.abs(wx[nz])
            worst = max(worst, rel.max())
            excess = np.abs(wg[nz] - wo[nz]) - (1e-12 * np.abs(wo[nz]) + 2.0 * np.abs(wo[nz] - wx[nz]))
            assert excess.max() <= 0.0
    assert worst <= 1e-12


@pytest.mark.parametrize("proc,n_perm,ne,n_points", [(3, 24, 6, 2 * (1 << 14) + 301), (3, 4, 6, (1 << 14) + 1),
                                                     (4, 2, 24, (1 << 14) + 301)])
def test_per_event(mem, proc, n_perm, ne, n_points):
    ev = wl.make_events(proc, ne, seed=11)
    p = oracle.params_default(proc)
    p.n_perm = n_perm
    po, eo = oracle.integrate(proc, p, ev, n_points, SEED)
    with mem.Integrator(proc, n_perm=n_perm) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    if proc == 4:
        # conic-solver process: an event that misses 1e-9 is taken apart point by point
        def drill(e):
            with mem.Integrator(proc, n_perm=n_perm) as it2:
                wg = it2.eval_points(_dev(ev), e, 0, n_points, SEED).cpu().numpy()
            return (wg, oracle.eval_points(proc, p, ev, e, 0, n_points, SEED),
                    oracle.eval_points_x(proc, p, ev, e, 0, n_points, SEED))
        # measured (profiles/r03_conic_parity.md): 1 of the 24 records misses 1e-9, by 1.7e-9 (4e-8 of its statistical
        # error), through one point of 14375 at which the oracle sides with the referee
        check_events_conic(pg, eg, po, eo, drill, n_points, ill=conic_ill_conditioned(ev), max_miss=1)
    else:
        assert np.array_equal(pg == 0, po == 0)
        assert np.all(np.abs(pg - po) <= 1e-9 * np.abs(po))
        assert np.all(np.abs(eg - eo) <= 1e-9 * np.abs(eo) + 1e-300)
    assert (po > 0).sum() >= ne // 4


def test_config4_per_point(mem):
    proc, ne, n = 4, 24, 2048 + 37
    ev = wl.make_events(proc, ne, seed=7)
    dev = _dev(ev)
    p = oracle.params_default(proc)
    p.n_perm = 2
    G, O, X = [], [], []
    with mem.Integrator(proc, n_perm=2) as it:
        for e in range(ne):
            G.append(it.eval_points(dev, e, 0, n, SEED).cpu().numpy())
            O.append(oracle.eval_points(proc, p, ev, e, 0, n, SEED))
            X.append(oracle.eval_points_x(proc, p, ev, e, 0, n, SEED))
    wg, wo, wx = np.concatenate(G), np.concatenate(O), np.concatenate(X)
    assert np.array_equal(wg == 0, wo == 0)
    nz = wo != 0
    assert nz.sum() > 2000
    eg = np.abs(wg[nz] - wx[nz]) / np.abs(wx[nz])
    eo = np.abs(wo[nz] - wx[nz]) / np.abs(wx[nz])
    assert np.mean(eg <= 1e-12) >= 0.99 and eg.max() <= 1e-8
    assert np.mean(eg > 1e-12 + 4.0 * eo) <= 1e-3


def test_record_order_invariance_and_vegas(mem):
    """with all 24 assignments the result does not depend on how the record lists its jets; the
    VEGAS path and the fp32 core take the summed integrand like any other"""
    import torch
    proc, ne, n_points = 3, 4, 20000
    ev = wl.make_events(proc, ne, seed=3)
    ev2 = ev.copy()
    ev2[3:6], ev2[9:12] = ev[9:12], ev[3:6]                      # swap jets 0 and 2 in the record
    with mem.Integrator(proc, n_perm=24) as it:
        a, _ = it.integrate(_dev(ev), n_points, SEED)
        b, _ = it.integrate(_dev(ev2), n_points, SEED)
        assert torch.allclose(a, b, rtol=1e-11, atol=0)
    p = oracle.params_default(proc)
    p.n_perm, p.vegas_iters, p.vegas_points = 24, 2, 9000
    po, eo = oracle.vegas_integrate(proc, p, ev, n_points, SEED)
    with mem.Integrator(proc, n_perm=24, vegas_iters=2, vegas_points=9000) as it:
        pg, _ = it.integrate(_dev(ev), n_points, SEED)
    assert np.all(np.abs(pg.cpu().numpy() - po) <= 1e-9 * np.abs(po))
    p = oracle.params_default(proc)
    p.n_perm = 24
    po, _ = oracle.integrate(proc, p, ev, n_points, SEED)
    with mem.Integrator(proc, n_perm=24, precision=32) as it:
        pg, _ = it.integrate(_dev(ev), n_points, SEED)
    assert np.all(np.abs(pg.cpu().numpy() - po) <= 1e-4 * np.abs(po))


def test_invalid_assignment_counts(mem):
    for proc, bad in ((1, 2), (2, 24), (3, 2), (3, 12), (4, 4), (4, 24)):
        with pytest.raises(mem.MemError) as ei:
            mem.Integrator(proc, n_perm=bad)
        assert ei.value.status == mem.MEM_ERR_INVALID_ARG
