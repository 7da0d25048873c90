"""GPU parity of NEXT-4 (t tbar H(-> b bbar) dilepton, four b jets, Eq. 9 chart, Eq. 11 balance) against the
CPU oracle, through the C ABI; then 1/sigma and the discriminant D (Eq. 10).

The neutrino system is the one of config 4 (two conics, Ferrari quartic, Newton polish), so the per-point
bar is config 4's: identical zero pattern; <= 1e-12 against the long-double
referee at >= 99 % of the live points; <= 1e-12 + 4 |w_orc - w_ref| everywhere except <= 0.1 % of them and
never beyond 1e-10; the GPU's 99.9th-percentile error not larger than twice the fp64 oracle's.
Eq. 9 adds one more integrable 1/sqrt edge (E1 = E2) with the same character.
Per event: |p_gpu - p_orc| <= 1e-9 |p_orc|, same for the standard error, on every event; the one test with records
that miss it states how many (two ill-conditioned ones of 32) and has each taken apart (tests/helpers.py).
"""
import numpy as np
import pytest

import oracle
from helpers import check_events_conic, check_points_conic, conic_ill_conditioned
from paper_1407_7595_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SEED = 20140729
PROC = 5


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


def _params(over):
    p = oracle.params_default(PROC)
    for k, v in (over or {}).items():
        setattr(p, k, v)
    return p


def _collect(mem, ev, first, n, over=None, offset=0):
    dev = _dev(ev)
    p = _params(over)
    G, O, X = [], [], []
    with mem.Integrator(PROC, **(over or {})) as it:
        it.set_event_offset(offset)
        for e in range(ev.shape[1]):
            G.append(it.eval_points(dev, e, first, n, SEED).cpu().numpy())
            O.append(oracle.eval_points(PROC, p, ev, e, first, n, SEED, event_offset=offset))
            X.append(oracle.eval_points_x(PROC, p, ev, e, first, n, SEED, event_offset=offset))
    return np.concatenate(G), np.concatenate(O), np.concatenate(X)


_check = check_points_conic


def _drill(mem, ev, n_points, over=None, offset=0):
    def f(e):
        p = _params(over)
        with mem.Integrator(PROC, **(over or {})) as it:
            it.set_event_offset(offset)
            wg = it.eval_points(_dev(ev), e, 0, n_points, SEED).cpu().numpy()
        return (wg, oracle.eval_points(PROC, p, ev, e, 0, n_points, SEED, event_offset=offset),
                oracle.eval_points_x(PROC, p, ev, e, 0, n_points, SEED, event_offset=offset))
    return f


@pytest.mark.parametrize("hyp", [0, 1])
def test_per_point_parity_closure_events(mem, hyp):
    """4133 points (several tiles and a ragged tail) of 24 physical t tbar H records, first point 5"""
    ev = wl.make_tth_events(24, seed=7)
    _check(*_collect(mem, ev, 5, 4096 + 37, over=dict(tth_hyp=hyp)), min_live=3000)


def test_per_point_parity_iid_events_high_point_index_and_offset(mem):
    ev = wl.make_events(PROC, 32, seed=3)
    _check(*_collect(mem, ev, (1 << 32) + 11, 1500, offset=1000), min_live=100)


@pytest.mark.parametrize("hyp", [0, 1])
def test_per_point_parity_other_parameters(mem, hyp):
    """wider resonances (also the Higgs), generic PDF exponents, other TF parameters and windows, other couplings"""
    ev = wl.make_tth_events(12, seed=5)
    over = dict(pdf_pow_x=-0.4, pdf_pow_1mx=4.5, pdf_A_q=0.7, pdf_A_g=1.9, tf_w_tail=0.2, tf_mu2=-0.05,
                tf_sig1=0.12, jetE_rlo=0.6, jetE_rhi=1.8, bw_nwidths=10.0, n_flav=4, Gam_t=2.5, Gam_W=3.0,
                m_H=120.0, Gam_H=3.0, yuk_t=0.8, yuk_b=0.03, tth_hyp=hyp)
    _check(*_collect(mem, ev, 0, 2500, over=over), min_live=500)


def test_per_point_parity_assignment_sum(mem):
    """PAPER.md:103-109 Eq. 7: all 4!/2 = 12 assignments of the four b jets per point"""
    ev = wl.make_tth_events(8, seed=9)
    _check(*_collect(mem, ev, 3, 700, over=dict(n_perm=12)), min_live=1000)


def test_per_point_parity_grid_pdfs(mem):
    ev = wl.make_tth_events(6, seed=13)
    tab = wl.make_pdf_table(A_g=1.3, A_q=0.8, q_slope=0.05)
    g = wl.PDF_GRID
    p = oracle.params_default(PROC)
    oracle.set_pdf_grid(p, tab, g["lxmin"], g["lxmax"], g["lqmin"], g["lqmax"], 173.0)
    dev = _dev(ev)
    G, O, X = [], [], []
    with mem.Integrator(PROC) as it:
        it.set_pdf_grid(tab, g["lxmin"], g["lxmax"], g["lqmin"], g["lqmax"], 173.0)
        for e in range(ev.shape[1]):
            G.append(it.eval_points(dev, e, 0, 1500, SEED).cpu().numpy())
            O.append(oracle.eval_points(PROC, p, ev, e, 0, 1500, SEED))
            X.append(oracle.eval_points_x(PROC, p, ev, e, 0, 1500, SEED))
    _check(np.concatenate(G), np.concatenate(O), np.concatenate(X), min_live=200)


# max_miss: events allowed to miss 1e-9, the measured count (profiles/r03_conic_parity.md).  Only the 32-record case
# has any: two records, both flagged by conic_ill_conditioned, miss by 8.5e-7 and 5.6e-5 (3e-6 and 7.8e-4 of their
# statistical error) through 1 of 707 and 11 of 2998 live points; each is taken apart by check_events_conic.
@pytest.mark.parametrize("ne,n_points,hyp,max_miss", [(24, 2, 0, 0), (24, 255, 0, 0), (16, 1 << 14, 0, 0),
                                                      (16, (1 << 14) + 1, 1, 0), (32, 2 * (1 << 14) + 301, 0, 2),
                                                      (12, 2 * (1 << 14) + 301, 1, 0)])
def test_per_event_parity(mem, ne, n_points, hyp, max_miss):
    ev = wl.make_tth_events(ne, seed=11)
    p = _params(dict(tth_hyp=hyp))
    po, eo = oracle.integrate(PROC, p, ev, n_points, SEED)
    with mem.Integrator(PROC, tth_hyp=hyp) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    check_events_conic(pg, eg, po, eo, _drill(mem, ev, n_points, dict(tth_hyp=hyp)), n_points,
                       ill=conic_ill_conditioned(ev, n_jets=4), max_miss=max_miss)
    if n_points > 1000:
        assert (po > 0).sum() >= ne // 2


def test_per_event_parity_assignment_sum_and_iid_events(mem):
    ev = wl.make_events(PROC, 24, seed=2)
    p = _params(dict(n_perm=12))
    n_points = 9000
    po, eo = oracle.integrate(PROC, p, ev, n_points, SEED)
    with mem.Integrator(PROC, n_perm=12) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
    check_events_conic(pg.cpu().numpy(), eg.cpu().numpy(), po, eo, _drill(mem, ev, n_points, dict(n_perm=12)), n_points,
                       ill=conic_ill_conditioned(ev, n_jets=4))
    assert (po > 0).sum() >= 6


def test_reproducible_partition_invariant_and_host_entry(mem):
    import torch
    ne, n_points = 12, (1 << 15) + 5
    ev = wl.make_tth_events(ne, seed=4)
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


def test_vegas_on_tth(mem):
    """the VEGAS path is process-generic: 2 adaptation passes on the t tbar H integrand"""
    ne = 6
    ev = wl.make_tth_events(ne, seed=17)
    p = oracle.params_default(PROC)
    p.vegas_iters, p.vegas_points = 2, 12000
    po, eo, go = oracle.vegas_integrate(PROC, p, ev, 20000, SEED, return_grid=True)
    with mem.Integrator(PROC, vegas_iters=2, vegas_points=12000) as it:
        pg, eg = it.integrate(_dev(ev), 20000, SEED)
        gg = it.grid(ne).cpu().numpy()
    assert np.max(np.abs(gg - go)) <= 1e-10
    assert np.all(np.abs(pg.cpu().numpy() - po) <= 1e-9 * np.abs(po))


def test_normalisation_and_discriminant(mem):
    """1/sigma (importance-sampled acceptance integral over the i.i.d. generator's density) and D = log10 of the
    normalised likelihood ratio, computed on the device from the two hypotheses' likelihoods"""
    import torch
    ne, n_points = 256, 4096
    ev = wl.make_events(PROC, ne, seed=8)
    g = wl.event_density(PROC, ev)
    dev, gdev = _dev(ev), _dev(g)
    with mem.Integrator(PROC, tth_hyp=0) as s, mem.Integrator(PROC, tth_hyp=1) as b:
        ps, _ = s.integrate(dev, n_points, SEED)
        pb, _ = b.integrate(dev, n_points, SEED)
    sig_s, sig_b = mem.mem_normalisation(ps, gdev), mem.mem_normalisation(pb, gdev)
    # results of the CUDA path are inputs of the post-processing step on both sides
    psn, pbn = ps.cpu().numpy(), pb.cpu().numpy()
    so, bo = oracle.normalisation(psn, g), oracle.normalisation(pbn, g)
    assert so > 0 and bo > 0
    assert abs(sig_s.item() - so) <= 1e-12 * so and abs(sig_b.item() - bo) <= 1e-12 * bo
    assert torch.equal(mem.mem_normalisation(ps, gdev), sig_s)                  # fixed summation order
    live = (psn > 0) & (pbn > 0)
    assert live.sum() >= 8
    D = mem.mem_discriminant(ps, pb, sig_s, sig_b).cpu().numpy()
    Do = oracle.discriminant(psn, pbn, so, bo)
    assert np.all(np.abs(D[live] - Do[live]) <= 1e-12 * np.maximum(1.0, np.abs(Do[live])))
    assert mem.lib().mem_normalisation(None, None, 0, None, None) == mem.MEM_ERR_INVALID_ARG
    assert mem.lib().mem_discriminant(None, None, 5, None, None, None, None) == mem.MEM_ERR_INVALID_ARG


def test_full_size_sampled_outputs(mem):
    """the bench workload (config 6: 16384 closure records x 2^18 points) in the launch configuration bench.py
    times; the oracle recomputes a sample of the per-event outputs one by one"""
    proc, ne, n_points = wl.CONFIGS[6]
    ev = wl.make_tth_events(ne)
    p = oracle.params_default(proc)
    with mem.Integrator(proc) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    assert np.all(np.isfinite(pg)) and np.all(np.isfinite(eg)) and np.all(pg >= 0) and np.all(eg >= 0)
    assert np.mean(pg > 0) > 0.5
    rng = np.random.default_rng(4)
    for e in rng.choice(np.flatnonzero(pg > 0), 3, replace=False):
        one = np.ascontiguousarray(ev[:, e:e + 1])
        po, eo = oracle.integrate(proc, p, one, n_points, SEED, event_offset=int(e))
        check_events_conic(pg[e:e + 1], eg[e:e + 1], po, eo, _drill(mem, one, n_points, offset=int(e)), n_points,
                           ill=conic_ill_conditioned(one, n_jets=4))
