"""GPU parity of the fp32 variant of config 3 (BASELINE.json:configs[2] "fp64 and fp32 variants",
reading A15) against the fp64 CPU oracle: per-event integral relative error <= 1e-4
(BASELINE.json:north_star).  Philox, per-event constants, the overall constant and the sums stay in
fp64/integer; the integrand core runs in single precision on fp32 uniforms built from the same
Philox words (within 2^-23 of the oracle's fp64 uniforms)."""
import numpy as np
import pytest

import oracle
from paper_1407_7595_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SEED = 20140729
PROC = 3
TOL_EVENT_FP32 = 1e-4


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


def test_per_point_error_distribution(mem):
    """fp32 core vs the fp64 oracle point by point: identical cuts except within rounding of a cut,
    typical error a few ulp of fp32, no outliers beyond the conditioning of the top pole"""
    ne, n = 16, 4096 + 37
    ev = wl.make_events(PROC, ne, seed=7)
    dev = _dev(ev)
    p = oracle.params_default(PROC)
    rel, flips, total = [], 0, 0
    with mem.Integrator(PROC, precision=32) as it:
        for e in range(ne):
            wg = it.eval_points(dev, e, 5, n, SEED).cpu().numpy()
            wo = oracle.eval_points(PROC, p, ev, e, 5, n, SEED)
            flips += np.sum((wg == 0) != (wo == 0))
            total += n
            nz = (wo != 0) & (wg != 0)
            rel.append(np.abs(wg[nz] - wo[nz]) / wo[nz])
    rel = np.concatenate(rel)
    assert flips <= 1e-4 * total                     # a cut decided differently in fp32
    assert np.median(rel) < 2e-6
    assert np.percentile(rel, 99) < 5e-5
    assert rel.max() < 5e-3


@pytest.mark.parametrize("ne,n_points", [(8, 2 * (1 << 14) + 301), (4, 1000), (6, 1 << 16)])
def test_per_event_parity_fp32(mem, ne, n_points):
    ev = wl.make_events(PROC, ne, seed=11)
    p = oracle.params_default(PROC)
    po, eo = oracle.integrate(PROC, p, ev, n_points, SEED)
    with mem.Integrator(PROC, precision=32) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    assert np.all(np.abs(pg - po) <= TOL_EVENT_FP32 * np.abs(po))
    assert np.all(np.abs(eg - eo) <= 10 * TOL_EVENT_FP32 * np.abs(eo))


def test_fp32_differs_from_fp64_and_is_reproducible(mem):
    """the fp32 handle really runs another kernel (results differ in the low digits) and is
    bitwise reproducible and partition invariant like the fp64 one"""
    import torch
    ne, n_points = 6, (1 << 15) + 5
    ev = wl.make_events(PROC, ne, seed=4)
    with mem.Integrator(PROC) as it64, mem.Integrator(PROC, precision=32) as it32:
        p64, _ = it64.integrate(_dev(ev), n_points, SEED)
        p32, e32 = it32.integrate(_dev(ev), n_points, SEED)
        p32b, e32b = it32.integrate(_dev(ev), n_points, SEED)
        assert torch.equal(p32, p32b) and torch.equal(e32, e32b)
        assert not torch.equal(p32, p64)
        assert torch.allclose(p32, p64, rtol=1e-4, atol=0)
        it32.set_event_offset(3)
        part, _ = it32.integrate(_dev(ev[:, 3:]), n_points, SEED)
        assert torch.equal(part, p32[3:])


def test_fp32_vegas(mem):
    """config-5 machinery on the fp32 core: grids and estimate track the fp64 oracle"""
    ne = 3
    ev = wl.make_events(PROC, ne, seed=7)
    p = oracle.params_default(PROC)
    p.vegas_iters, p.vegas_points = 2, 20000
    po, eo, go = oracle.vegas_integrate(PROC, p, ev, 30000, SEED, return_grid=True)
    with mem.Integrator(PROC, precision=32, vegas_iters=2, vegas_points=20000) as it:
        pg, eg = it.integrate(_dev(ev), 30000, SEED)
        gg = it.grid(ne).cpu().numpy()
    assert np.max(np.abs(gg - go)) <= 1e-4
    assert np.all(np.abs(pg.cpu().numpy() - po) <= 2e-3 * np.abs(po))   # grids differ at 1e-5: other points
    assert np.all(np.diff(gg, axis=2) > 0)


def test_fp32_only_for_config3(mem):
    for proc in (1, 2, 4):
        with pytest.raises(mem.MemError) as ei:
            mem.Integrator(proc, precision=32)
        assert ei.value.status == mem.MEM_ERR_UNSUPPORTED


def test_full_size_sampled_outputs_fp32(mem):
    proc, ne, n_points = wl.CONFIGS[3]
    ev = wl.make_events(proc, ne)
    p = oracle.params_default(proc)
    with mem.Integrator(proc, precision=32) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    assert np.all(np.isfinite(pg)) and np.all(np.isfinite(eg)) and np.all(pg >= 0)
    for e in (17, 2900):
        po, eo = oracle.integrate(proc, p, ev[:, e:e + 1], n_points, SEED, event_offset=e)
        assert abs(pg[e] - po[0]) <= TOL_EVENT_FP32 * abs(po[0]), e
