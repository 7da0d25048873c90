"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Per-point bar (BASELINE.json:north_star):
  A  |w_gpu - w_ref| <= 1e-12 |w_ref|                     ref = the oracle's algorithm in long double
  B  |w_gpu - w_orc| <= 1e-12 |w_orc| + 2 |w_orc - w_ref|  orc = the fp64 oracle; the second term is
     the fp64 oracle's own measured rounding error at that point (it exceeds 1e-12 at a few
     ill-conditioned points: cancellation in s_t = p_t^2 next to the top pole, in 1 - beta^2 for
     nearly collinear jets, in t_hi - t_lo far above the W pole)
  C  the set of points with w = 0 (kinematic cuts) is identical
Per-event bar: |p_gpu - p_orc| <= 1e-9 |p_orc|, same for the standard error.
"""
import numpy as np
import pytest

import oracle
from paper_1407_7595_b200 import workloads as wl

pytestmark = pytest.mark.gpu

SEED = 20140729
TOL_POINT = 1e-12
TOL_EVENT = 1e-9


@pytest.fixture(scope="module")
def mem():
    import torch
    assert torch.cuda.is_available()
    import paper_1407_7595_b200 as m
    m.lib()          # must load the CUDA library: there is no fallback
    return m


def _dev(ev):
    import torch
    return torch.from_numpy(np.ascontiguousarray(ev)).cuda()


def _check_points(wg, wo, wx, label):
    assert np.array_equal(wg == 0.0, wo == 0.0), label + ": zero pattern differs"
    nz = wo != 0.0
    assert nz.sum() > 0
    rel_ref = np.abs(wg[nz] - wx[nz]) / np.abs(wx[nz])
    assert rel_ref.max() <= TOL_POINT, "%s: gpu vs referee %.3e" % (label, rel_ref.max())
    excess = np.abs(wg[nz] - wo[nz]) - (TOL_POINT * np.abs(wo[nz]) + 2.0 * np.abs(wo[nz] - wx[nz]))
    assert excess.max() <= 0.0, "%s: gpu vs fp64 oracle beyond its own rounding error" % label
    return rel_ref.max()


@pytest.mark.parametrize("proc", [1, 2, 3])
def test_per_point_parity(mem, proc):
    """4133 points (several 128-thread tiles and a ragged tail) of 24 events, first point 5."""
    ne, n, first = 24, 4096 + 37, 5
    ev = wl.make_events(proc, ne, seed=7)
    dev = _dev(ev)
    p = oracle.params_default(proc)
    with mem.Integrator(proc) as it:
        for e in range(ne):
            wg = it.eval_points(dev, e, first, n, SEED).cpu().numpy()
            wo = oracle.eval_points(proc, p, ev, e, first, n, SEED)
            wx = oracle.eval_points_x(proc, p, ev, e, first, n, SEED)
            _check_points(wg, wo, wx, "proc %d event %d" % (proc, e))


@pytest.mark.parametrize("proc", [1, 2, 3])
def test_per_point_parity_high_point_index_and_offset(mem, proc):
    """point counter above 2^32 and a non-zero event offset reach the Philox counter words"""
    ne, n = 3, 700
    ev = wl.make_events(proc, ne, seed=3)
    dev = _dev(ev)
    p = oracle.params_default(proc)
    first = (1 << 32) + 11
    with mem.Integrator(proc) as it:
        it.set_event_offset(1000)
        for e in range(ne):
            wg = it.eval_points(dev, e, first, n, SEED).cpu().numpy()
            wo = oracle.eval_points(proc, p, ev, e, first, n, SEED, event_offset=1000)
            wx = oracle.eval_points_x(proc, p, ev, e, first, n, SEED, event_offset=1000)
            _check_points(wg, wo, wx, "proc %d event %d" % (proc, e))


def test_per_point_parity_generic_pdf_and_tf(mem):
    """non-default toy-PDF exponents (generic pow path), TF parameters and windows"""
    proc, ne, n = 3, 4, 1500
    ev = wl.make_events(proc, ne, seed=5)
    dev = _dev(ev)
    over = dict(pdf_pow_x=-0.4, pdf_pow_1mx=4.5, pdf_A_q=0.7, pdf_A_g=1.9, tf_w_tail=0.2, tf_mu2=-0.05,
                tf_sig1=0.12, jetE_rlo=0.6, jetE_rhi=1.8, nu_eta_max=4.0, bw_nwidths=10.0, n_flav=4)
    p = oracle.params_default(proc)
    for k, v in over.items():
        setattr(p, k, v)
    with mem.Integrator(proc, **over) as it:
        for e in range(ne):
            wg = it.eval_points(dev, e, 0, n, SEED).cpu().numpy()
            wo = oracle.eval_points(proc, p, ev, e, 0, n, SEED)
            wx = oracle.eval_points_x(proc, p, ev, e, 0, n, SEED)
            _check_points(wg, wo, wx, "event %d" % e)


# n_points: below one block, exactly one chunk, one chunk + 1, several chunks + ragged tail
@pytest.mark.parametrize("proc,ne,n_points", [(1, 16, 2), (1, 16, 255), (1, 8, 1 << 14), (1, 8, (1 << 14) + 1),
                                              (1, 8, 3 * (1 << 14) + 4133), (2, 8, 2 * (1 << 14) + 77),
                                              (3, 6, 2 * (1 << 14) + 301), (3, 1, 1000)])
def test_per_event_parity(mem, proc, ne, n_points):
    ev = wl.make_events(proc, ne, seed=11)
    p = oracle.params_default(proc)
    po, eo = oracle.integrate(proc, p, ev, n_points, SEED)
    with mem.Integrator(proc) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    assert np.all(np.abs(pg - po) <= TOL_EVENT * np.abs(po))
    assert np.all(np.abs(eg - eo) <= TOL_EVENT * np.abs(eo) + 1e-300)


def test_host_entry_matches_device_entry(mem):
    import torch
    proc, ne, n_points = 3, 5, (1 << 14) + 9
    ev = wl.make_events(proc, ne, seed=2)
    with mem.Integrator(proc) as it:
        pd, ed = it.integrate(_dev(ev), n_points, SEED)
        ph, eh = it.integrate_host(torch.from_numpy(ev), n_points, SEED)
        assert torch.equal(pd.cpu(), ph) and torch.equal(ed.cpu(), eh)


def test_bitwise_reproducible_and_partition_invariant(mem):
    """same call twice -> same bits; a shard with the right event offset -> the same bits as the
    unsharded call"""
    import torch
    proc, ne, n_points = 3, 12, (1 << 15) + 5
    ev = wl.make_events(proc, ne, seed=4)
    with mem.Integrator(proc) as it:
        p1, e1 = it.integrate(_dev(ev), n_points, SEED)
        p2, e2 = it.integrate(_dev(ev), n_points, SEED)
        assert torch.equal(p1, p2) and torch.equal(e1, e2)
        parts_p, parts_e = [], []
        for rank in range(3):
            lo, hi = wl.shard_range(ne, rank, 3)
            it.set_event_offset(lo)
            a, b = it.integrate(_dev(ev[:, lo:hi]), n_points, SEED)
            parts_p.append(a); parts_e.append(b)
        assert torch.equal(torch.cat(parts_p), p1) and torch.equal(torch.cat(parts_e), e1)


def test_vegas_parity(mem):
    """config 5 at reduced size: grids after 3 adaptation passes and the final estimate"""
    proc, ne = 3, 4
    ev = wl.make_events(proc, ne, seed=7)
    p = oracle.params_default(proc)
    p.vegas_iters, p.vegas_points = 3, (1 << 14) + 999
    n_points = (1 << 15) + 77
    po, eo, go = oracle.vegas_integrate(proc, p, ev, n_points, SEED, return_grid=True)
    with mem.Integrator(proc, vegas_iters=3, vegas_points=(1 << 14) + 999) as it:
        dev = _dev(ev)
        pg, eg = it.integrate(dev, n_points, SEED)
        gg = it.grid(ne).cpu().numpy()
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
        # S9: the refined edges agree to rounding (sum order of the histograms differs)
        assert np.max(np.abs(gg - go)) <= 1e-11
        assert np.all(np.diff(gg, axis=2) > 0) and np.all(gg[:, :, 0] == 0) and np.all(gg[:, :, -1] == 1)
        assert np.all(np.abs(pg - po) <= TOL_EVENT * np.abs(po))
        assert np.all(np.abs(eg - eo) <= TOL_EVENT * np.abs(eo))
        # S1v per point through the oracle's grid
        import torch
        for e in range(ne):
            wg = it.eval_points(dev, e, 0, 3000, SEED, iteration=3, grid=torch.from_numpy(go[e]).cuda()).cpu().numpy()
            wo = oracle.eval_points(proc, p, ev, e, 0, 3000, SEED, iteration=3, grid=go)
            wx = oracle.eval_points_x(proc, p, ev, e, 0, 3000, SEED, iteration=3, grid=go)
            _check_points(wg, wo, wx, "vegas event %d" % e)
        # the adapted estimate is more precise than plain MC of the same size
    with mem.Integrator(proc) as plain:
        _, e_plain = plain.integrate(_dev(ev), n_points, SEED)
    assert np.all(eg < e_plain.cpu().numpy())


@pytest.mark.parametrize("bins", [1, 7, 64])
def test_vegas_bin_counts(mem, bins):
    proc, ne = 2, 3
    ev = wl.make_events(proc, ne, seed=9)
    p = oracle.params_default(proc)
    p.vegas_iters, p.vegas_points, p.vegas_bins = 2, 5000, bins
    po, eo, go = oracle.vegas_integrate(proc, p, ev, 6000, SEED, return_grid=True)
    with mem.Integrator(proc, vegas_iters=2, vegas_points=5000, vegas_bins=bins) as it:
        pg, eg = it.integrate(_dev(ev), 6000, SEED)
        gg = it.grid(ne).cpu().numpy()
    assert np.max(np.abs(gg - go)) <= 1e-11
    assert np.all(np.abs(pg.cpu().numpy() - po) <= TOL_EVENT * np.abs(po))


def test_vegas_grid_reproducible_ragged_and_empty_histogram(mem):
    """S9 edge cases: fewer adaptation points than one block takes per sweep (ragged warps in the histogram rounds), an
    event whose weights all vanish (its grid must stay the uniform one), and bitwise identical grids on a second run"""
    import torch
    proc, ne = 2, 5
    ev = wl.make_events(proc, ne, seed=21)
    ev[0, 2] = ev[3, 2] = 1e5                      # jet energies beyond the beam energy: every point is cut
    p = oracle.params_default(proc)
    p.vegas_iters, p.vegas_points = 3, 301
    po, eo, go = oracle.vegas_integrate(proc, p, ev, 777, SEED, return_grid=True)
    assert po[2] == 0.0 and np.count_nonzero(po) == ne - 1
    with mem.Integrator(proc, vegas_iters=3, vegas_points=301) as it:
        dev = _dev(ev)
        pg, eg = it.integrate(dev, 777, SEED)
        g1 = it.grid(ne).clone()
        pg2, _ = it.integrate(dev, 777, SEED)
        g2 = it.grid(ne)
        assert torch.equal(g1, g2) and torch.equal(pg, pg2)
    gg = g1.cpu().numpy()
    assert np.max(np.abs(gg - go)) <= 1e-11
    B = gg.shape[2] - 1
    assert np.array_equal(gg[2], np.broadcast_to(np.arange(B + 1) / B, gg[2].shape))
    assert pg.cpu().numpy()[2] == 0.0
    live = po > 0
    assert np.all(np.abs(pg.cpu().numpy()[live] - po[live]) <= TOL_EVENT * po[live])


def test_edge_cases_and_errors(mem):
    import torch
    proc = 1
    ev = wl.make_events(proc, 4, seed=1)
    dev = _dev(ev)
    with mem.Integrator(proc) as it:
        # empty event list: MEM_OK, no launch
        n0 = it.launches
        empty = torch.empty((5, 0), dtype=torch.float64, device="cuda")
        p, e = it.integrate(empty, 100, SEED)
        assert p.numel() == 0 and it.launches == n0
        with pytest.raises(mem.MemError) as ei:
            it.integrate(dev, 1, SEED)                  # n_points < 2
        assert ei.value.status == mem.MEM_ERR_INVALID_ARG
        with pytest.raises(mem.MemError):
            it.eval_points(dev, 4, 0, 10, SEED)         # event out of range
        with pytest.raises(mem.MemError):
            it.grid(4)                                  # no VEGAS grids on a plain handle
        assert "VEGAS" in mem.mem_last_error()
    bad = mem.mem_params_default(proc)
    bad.tf_sig1 = -1.0
    with pytest.raises(mem.MemError):
        mem.mem_create(proc, bad)
    bad = mem.mem_params_default(3)
    bad.tf_sig1 = 0.02                                 # core so narrow that exp(z1^2 - z2^2) would overflow in the window
    with pytest.raises(mem.MemError) as ei:
        mem.mem_create(3, bad)
    assert ei.value.status == mem.MEM_ERR_INVALID_ARG and "too narrow" in mem.mem_last_error()
    ok = mem.mem_params_default(3)
    ok.tf_sig1 = 0.05
    mem.mem_destroy(mem.mem_create(3, ok))
    bad = mem.mem_params_default(proc)
    bad.struct_size = 8
    with pytest.raises(mem.MemError):
        mem.mem_create(proc, bad)
    with pytest.raises(mem.MemError) as ei:
        mem.mem_create(99)
    assert ei.value.status == mem.MEM_ERR_INVALID_ARG


def test_forbidden_points_contribute_zero(mem):
    """sqrt(s) below 2 m_t: every point fails the threshold cut (reading A9), p = err = 0 exactly"""
    proc = 3
    ev = wl.make_events(proc, 3, seed=1)
    p = oracle.params_default(proc)
    p.sqrt_s = 300.0
    po, eo = oracle.integrate(proc, p, ev, 4000, SEED)
    with mem.Integrator(proc, sqrt_s=300.0) as it:
        pg, eg = it.integrate(_dev(ev), 4000, SEED)
    assert np.all(po == 0.0) and np.all(eo == 0.0)
    assert np.all(pg.cpu().numpy() == 0.0) and np.all(eg.cpu().numpy() == 0.0)


def test_full_size_sampled_outputs(mem):
    """BASELINE configs 1-3 at full size in the launch configuration bench.py times; the oracle
    recomputes a sample of the per-event outputs one by one"""
    for cfg, n_sample in ((1, 6), (2, 3), (3, 2)):
        proc, ne, n_points = wl.CONFIGS[cfg]
        ev = wl.make_events(proc, ne)
        p = oracle.params_default(proc)
        with mem.Integrator(proc) as it:
            pg, eg = it.integrate(_dev(ev), n_points, SEED)
            pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
        assert np.all(np.isfinite(pg)) and np.all(np.isfinite(eg)) and np.all(pg >= 0) and np.all(eg >= 0)
        rng = np.random.default_rng(cfg)
        for e in rng.choice(ne, n_sample, replace=False):
            po, eo = oracle.integrate(proc, p, ev[:, e:e + 1], n_points, SEED, event_offset=int(e))
            assert abs(pg[e] - po[0]) <= TOL_EVENT * abs(po[0]), (cfg, e)
            assert abs(eg[e] - eo[0]) <= TOL_EVENT * abs(eo[0]), (cfg, e)


def test_full_size_vegas_sampled_output(mem):
    """BASELINE config 5 base cell: 5 x 2^17 adaptation + 2^20 final, 256 events; one event recomputed"""
    proc, ne, n_points = 3, 256, 1 << 20
    ev = wl.make_events(proc, ne)
    p = oracle.params_default(proc)
    p.vegas_iters, p.vegas_points = 5, 1 << 17
    with mem.Integrator(proc, vegas_iters=5, vegas_points=1 << 17) as it:
        pg, eg = it.integrate(_dev(ev), n_points, SEED)
        pg, eg = pg.cpu().numpy(), eg.cpu().numpy()
    e = 137
    po, eo = oracle.vegas_integrate(proc, p, ev[:, e:e + 1], n_points, SEED, event_offset=e)
    assert abs(pg[e] - po[0]) <= TOL_EVENT * abs(po[0])
    assert abs(eg[e] - eo[0]) <= TOL_EVENT * abs(eo[0])


def test_fp64_microbenchmarks(mem):
    """the roofline denominators are measured, not assumed: plausible values, the documented ordering, argument checks"""
    peak = mem.mem_measure_fp64_peak(2)
    rrr = mem.mem_measure_fp64_peak_rrr(2)
    assert 20.0 < peak < 45.0 and 10.0 < rrr < peak
    assert abs(mem.mem_measure_fp64_rate(0, 2) - peak) < 0.1 * peak
    assert mem.mem_measure_fp64_rate(4, 2) < mem.mem_measure_fp64_rate(3, 2) < peak * 1.02
    with pytest.raises(mem.MemError):
        mem.mem_measure_fp64_rate(7, 2)


def test_cuda_graph_capture_and_replay(mem):
    """mem_integrate only enqueues work on the caller's stream, so once a first call has sized the workspace the
    whole pass sequence (here VEGAS: grid init, 2 x (adapt, refine), final, finalize) can be captured into a CUDA
    graph and replayed; the replay reproduces the eager result bit for bit"""
    import torch
    proc = 3
    ev = _dev(wl.make_events(proc, 48, seed=5))
    out_p = torch.empty(48, dtype=torch.float64, device="cuda")
    out_e = torch.empty_like(out_p)
    with mem.Integrator(proc, vegas_iters=2, vegas_points=4096) as it:
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            it.integrate(ev, 8192, SEED, out_p=out_p, out_err=out_e)
        s.synchronize()
        ref_p, ref_e = out_p.clone(), out_e.clone()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            it.integrate(ev, 8192, SEED, out_p=out_p, out_err=out_e)
        out_p.zero_(); out_e.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(out_p, ref_p) and torch.equal(out_e, ref_e)


@pytest.mark.parametrize("proc,over", [(3, {}), (2, {}), (4, {}), (5, {}), (3, dict(vegas_iters=2, vegas_points=4096))])
def test_diagnostic_weights_are_the_summed_weights(mem, proc, over):
    """mem_eval_points evaluates with the same code (same exp, same grid map) as the pass that produces the outputs:
    the mean of the per-point weights it reports is the integral mem_integrate returns"""
    import torch
    ne, n_points = 3, 8192 + 77
    ev = wl.make_tth_events(ne, seed=3) if proc == 5 else wl.make_events(proc, 64, seed=9)
    if proc == 4:            # keep events that have live points
        po, _ = oracle.integrate(proc, oracle.params_default(proc), ev, 1500, SEED)
        ev = np.ascontiguousarray(ev[:, po > 0])
    ev = np.ascontiguousarray(ev[:, :ne])
    dev = _dev(ev)
    with mem.Integrator(proc, **over) as it:
        p, _ = it.integrate(dev, n_points, SEED)
        grid = it.grid(ne) if over else None
        for e in range(ne):
            w = it.eval_points(dev, e, 0, n_points, SEED, iteration=over.get("vegas_iters", 0),
                               grid=None if grid is None else grid[e].contiguous())
            assert abs(w.sum().item() / n_points - p[e].item()) <= 1e-12 * abs(p[e].item())
    assert float(p.max()) > 0
