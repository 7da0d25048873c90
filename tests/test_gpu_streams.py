"""One handle used from several CUDA streams (include/mem.h, conventions paragraph): the workspace is shared by
consecutive calls, so each call orders itself after the previous one on the handle and a growth step waits for it
before freeing.  Also the argument validation of the binding and the capture rule of mem_last_pass_ms."""
import numpy as np
import pytest

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


@pytest.mark.parametrize("proc,over", [(3, {}), (3, dict(vegas_iters=2, vegas_points=3000)), (4, {})])
def test_two_streams_on_one_handle_with_workspace_growth(mem, proc, over):
    import torch
    sizes = [(8 + 6 * k, 3000 + 4097 * (k % 3)) for k in range(20)]          # events grow: the workspace is reallocated
    evs = [torch.from_numpy(wl.make_events(proc, ne, seed=100 + k)).cuda() for k, (ne, _) in enumerate(sizes)]
    # reference: a fresh handle per call on the default stream
    ref = []
    for ev, (ne, npts) in zip(evs, sizes):
        with mem.Integrator(proc, **over) as it:
            p, e = it.integrate(ev, npts, SEED)
            ref.append((p.clone(), e.clone()))
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]                      # non-blocking side streams
    outs = []
    with mem.Integrator(proc, **over) as it:
        for k, (ev, (ne, npts)) in enumerate(zip(evs, sizes)):
            s = streams[k % 2]
            p = torch.empty(ne, dtype=torch.float64, device="cuda")
            e = torch.empty_like(p)
            with torch.cuda.stream(s):
                it.integrate(ev, npts, SEED, out_p=p, out_err=e, stream=s)     # no host synchronisation in between
            outs.append((p, e))
        torch.cuda.synchronize()
    for (p, e), (pr, er) in zip(outs, ref):
        assert torch.equal(p, pr) and torch.equal(e, er)


def test_host_entry_on_a_side_stream(mem):
    import torch
    proc, ne, npts = 3, 32, 5000
    ev = wl.make_events(proc, ne, seed=3)
    s = torch.cuda.Stream()
    with mem.Integrator(proc) as it:
        p0, e0 = it.integrate(torch.from_numpy(ev).cuda(), npts, SEED)
        ph, eh = it.integrate_host(torch.from_numpy(ev).pin_memory(), npts, SEED, stream=s)
        assert torch.equal(p0.cpu(), ph) and torch.equal(e0.cpu(), eh)


def test_binding_rejects_wrong_shapes_and_devices(mem):
    import torch
    ev = torch.from_numpy(wl.make_events(3, 16, seed=1)).cuda()
    with mem.Integrator(3, vegas_iters=1, vegas_points=1000) as it:
        with pytest.raises(ValueError):
            it.integrate(ev.t().contiguous(), 1000, SEED)                      # [n_events, n_fields]: transposed
        with pytest.raises(ValueError):
            it.integrate(torch.from_numpy(wl.make_events(4, 16)).cuda(), 1000, SEED)   # a config-4 record
        with pytest.raises(ValueError):
            it.eval_points(ev, 0, 0, 10, SEED, grid=torch.zeros(6, 7, dtype=torch.float64, device="cuda"))
        with pytest.raises(ValueError):
            it.eval_parton(torch.zeros(16, 24, dtype=torch.float64, device="cuda"))
        with pytest.raises(ValueError):
            it.integrate_host(torch.from_numpy(wl.make_events(1, 16)), 1000, SEED)
        it.integrate(ev, 1000, SEED)                                           # and the right one still works


def test_last_pass_ms_does_not_see_captured_calls(mem):
    import torch
    ev = torch.from_numpy(wl.make_events(3, 16, seed=1)).cuda()
    p = torch.empty(16, dtype=torch.float64, device="cuda")
    e = torch.empty_like(p)
    with mem.Integrator(3) as it:
        it.integrate(ev, 4000, SEED, out_p=p, out_err=e)                      # sizes the workspace
        torch.cuda.synchronize()
        ms, evals = it.last_pass_ms()
        assert ms > 0 and evals == 16 * 4000
        ref = p.clone()
        g = torch.cuda.CUDAGraph()
        s = torch.cuda.Stream()
        with torch.cuda.stream(s):
            with torch.cuda.graph(g, stream=s):
                it.integrate(ev, 4000, SEED, out_p=p, out_err=e, stream=s)
        with pytest.raises(mem.MemError):
            it.last_pass_ms()
        p.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(p, ref)
        it.integrate(ev, 4000, SEED, out_p=p, out_err=e)
        torch.cuda.synchronize()
        assert it.last_pass_ms()[1] == 16 * 4000
