"""GPU parity of config 4 (8-D t tbar dilepton) against the CPU oracle, through the C ABI.

Per-point bar (config-4 paragraph).  Config 4 solves two conics
for the neutrino momenta; next to a tangency of the conics the solution and its Jacobian are
ill-conditioned in fp64 on either side ("double precision is required due to
cancellation of large coefficients"), so the fp64 oracle itself departs from its long-double
referee by more than 1e-12 at ~0.3 % of the live points.  The bar is therefore:
  A  identical zero pattern (same points have no solution / fail the cuts)
  B  |w_gpu - w_ref| <= 1e-12 |w_ref| at >= 99 % of the live points
  C  at every live point |w_gpu - w_ref| <= 1e-12 |w_ref| + 4 |w_orc - w_ref|, except at most 0.1 % of
     them, and never beyond 1e-10
  D  the 99.9th percentile of the GPU's error is not larger than twice the fp64 oracle's
Per-event bar: |p_gpu - p_orc| <= 1e-9 |p_orc| on every event, same for the standard error -- no allowance
(tests/helpers.py: check_points_conic, check_events_conic with max_miss = 0).  These are round 1's bars; the round-2
relaxations (zero-pattern flips, 15 % of the events) are gone: measured on this round's kernel, no config-4 test
needs them (profiles/r03_conic_parity.md).
"""
import numpy as np
import pytest

import oracle
from helpers import check_events_conic, check_points_conic
from paper_1407_7595_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SEED = 20140729
PROC = 4


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


def _collect(mem, ev, first, n, p, over=None, offset=0):
    dev = _dev(ev)
    G, O, X = [], [], []
    with mem.Integrator(PROC, **(over or {})) as it:
        it.set_event_offset(offset)
        for e in range(ev.shape[1]):
            G.append(it.eval_points(dev, e, first, n, SEED).cpu().numpy())
            O.append(oracle.eval_points(PROC, p, ev, e, first, n, SEED, event_offset=offset))
            X.append(oracle.eval_points_x(PROC, p, ev, e, first, n, SEED, event_offset=offset))
    return np.concatenate(G), np.concatenate(O), np.concatenate(X)


_check = check_points_conic


def _drill(mem, ev, n_points, offset=0):
    def f(e):
        p = oracle.params_default(PROC)
        with mem.Integrator(PROC) as it:
            it.set_event_offset(offset)
            wg = it.eval_points(_dev(ev), e, 0, n_points, SEED).cpu().numpy()
        return (wg, oracle.eval_points(PROC, p, ev, e, 0, n_points, SEED, event_offset=offset),
                oracle.eval_points_x(PROC, p, ev, e, 0, n_points, SEED, event_offset=offset))
    return f


def test_per_point_parity(mem):
    """4133 points (several tiles and a ragged tail) of 48 events, first point 5"""
    ev = wl.make_events(PROC, 48, seed=7)
    p = oracle.params_default(PROC)
    _check(*_collect(mem, ev, 5, 4096 + 37, p), min_live=5000)


def test_per_point_parity_high_point_index_and_offset(mem):
    ev = wl.make_events(PROC, 16, seed=3)
    p = oracle.params_default(PROC)
    _check(*_collect(mem, ev, (1 << 32) + 11, 1200, p, offset=1000), min_live=500)


def test_per_point_parity_other_parameters(mem):
    """wider resonances and MET resolution, generic PDF exponents, other TF parameters"""
    ev = wl.make_events(PROC, 16, seed=5)
    over = dict(pdf_pow_x=-0.4, pdf_pow_1mx=4.5, pdf_A_q=0.7, pdf_A_g=1.9, tf_w_tail=0.2, tf_mu2=-0.05,
                tf_sig1=0.12, jetE_rlo=0.6, jetE_rhi=1.8, bw_nwidths=10.0, n_flav=4, Gam_t=2.5, Gam_W=3.0,
                met_sigma=15.0, met_nsigma=3.0)
    p = oracle.params_default(PROC)
    for k, v in over.items():
        setattr(p, k, v)
    _check(*_collect(mem, ev, 0, 1500, p, over=over), min_live=500)


@pytest.mark.parametrize("ne,n_points", [(24, 2), (24, 255), (16, 1 << 14), (16, (1 << 14) + 1),
                                         (32, 2 * (1 << 14) + 301)])
def test_per_event_parity(mem, ne, n_points):
    ev = wl.make_events(PROC, ne, seed=11)
    p = oracle.params_default(PROC)
    po, eo = oracle.integrate(PROC, p, ev, n_points, SEED)
    with mem.Integrator(PROC) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    check_events_conic(pg, eg, po, eo, _drill(mem, ev, n_points), n_points)
    if n_points > 1000:
        assert (po > 0).sum() >= ne // 4


def test_reproducible_partition_invariant_and_host_entry(mem):
    import torch
    ne, n_points = 12, (1 << 15) + 5
    ev = wl.make_events(PROC, ne, seed=4)
    with mem.Integrator(PROC) as it:
        p1, e1 = it.integrate(_dev(ev), n_points, SEED)
        p2, e2 = it.integrate(_dev(ev), n_points, SEED)
        assert torch.equal(p1, p2) and torch.equal(e1, e2)
        ph, eh = it.integrate_host(torch.from_numpy(ev), n_points, SEED)
        assert torch.equal(p1.cpu(), ph) and torch.equal(e1.cpu(), eh)
        parts = []
        for rank in range(3):
            lo, hi = wl.shard_range(ne, rank, 3)
            it.set_event_offset(lo)
            parts.append(it.integrate(_dev(ev[:, lo:hi]), n_points, SEED)[0])
        assert torch.equal(torch.cat(parts), p1)


def test_vegas_on_config4(mem):
    """the VEGAS path is process-generic: 2 adaptation passes on the 8-D integrand"""
    ne = 6
    ev = wl.make_events(PROC, 64, seed=11)
    p = oracle.params_default(PROC)
    # keep events that have live points
    po, _ = oracle.integrate(PROC, p, ev, 2000, SEED)
    ev = np.ascontiguousarray(ev[:, po > 0][:, :ne])
    assert ev.shape[1] == ne
    p.vegas_iters, p.vegas_points = 2, 12000
    po, eo, go = oracle.vegas_integrate(PROC, p, ev, 20000, SEED, return_grid=True)
    with mem.Integrator(PROC, vegas_iters=2, vegas_points=12000) as it:
        pg, eg = it.integrate(_dev(ev), 20000, SEED)
        gg = it.grid(ne).cpu().numpy()
    assert np.max(np.abs(gg - go)) <= 1e-10
    assert np.all(np.abs(pg.cpu().numpy() - po) <= 1e-9 * np.abs(po))


def test_full_size_sampled_outputs(mem):
    """BASELINE config 4 at full size (16384 events x 2^18 points) in the launch configuration
    bench.py times; the oracle recomputes a sample of the per-event outputs one by one"""
    proc, ne, n_points = wl.CONFIGS[4]
    ev = wl.make_events(proc, ne)
    p = oracle.params_default(proc)
    with mem.Integrator(proc) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    assert np.all(np.isfinite(pg)) and np.all(np.isfinite(eg)) and np.all(pg >= 0) and np.all(eg >= 0)
    assert 0.3 < np.mean(pg > 0) < 0.7
    live = np.flatnonzero(pg > 0)
    dead = np.flatnonzero(pg == 0)
    rng = np.random.default_rng(4)
    for e in list(rng.choice(live, 3, replace=False)) + list(rng.choice(dead, 1)):
        one = np.ascontiguousarray(ev[:, e:e + 1])
        po, eo = oracle.integrate(proc, p, one, n_points, SEED, event_offset=int(e))
        check_events_conic(pg[e:e + 1], eg[e:e + 1], po, eo, _drill(mem, one, n_points, offset=int(e)), n_points)
