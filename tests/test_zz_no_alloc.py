"""mem_integrate_noalloc (include/mem.h): the integrator for hosts that may not allocate device memory.

Who needs it: a real-time event filter whose GPU memory was handed out once at start-up, an application whose own
memory pool already owns the whole device, any loop that cannot take the device-wide stall of a cudaFree / cudaMalloc
pair.  mem_integrate grows a cudaMalloc'd workspace whenever a call is larger than the ones before; this entry point
keeps the same intermediate arrays in one fixed array of MEM_NOALLOC_SCRATCH_BYTES (8 MiB) inside the library image
and refuses anything that does not fit.

What is checked: the new entry point against the existing mem_integrate on the same inputs, on two calls in a row
that lay the shared array out differently (so the second call runs over the first one's leftovers, including its
arrival counters).  Both paths launch the same kernels in the same geometry, so the comparison is made at the
per-event bar of the parity tests (1e-9 relative, tests/test_gpu_parity.py) and, more strictly, bit for bit.  Also:
the driver's free-memory figure does not move across no-alloc calls that are larger than any before, and the stated
limits are enforced with a clear message.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  The test passes alone in a fresh process and after the rest of the suite."""
import numpy as np
import pytest

from paper_1407_7595_b200 import workloads as wl

pytestmark = pytest.mark.gpu
SEED = 20140729
REL = 1e-9      # per-event bar of the parity tests


@pytest.fixture(scope="module")
def mem():
    import torch
    assert torch.cuda.is_available()
    import paper_1407_7595_b200 as m
    m.lib()
    return m


def _events(proc, n, seed):
    import torch
    return torch.from_numpy(wl.make_events(proc, n, seed=seed)).cuda()


def _outs(n):
    import torch
    # poisoned: a kernel that skips an event cannot pass by accident
    return (torch.full((n,), float("nan"), dtype=torch.float64, device="cuda"),
            torch.full((n,), float("nan"), dtype=torch.float64, device="cuda"))


def _same(got, want):
    import torch
    for g, w in zip(got, want):
        g, w = g.cpu().numpy(), w.cpu().numpy()
        assert np.all(np.isfinite(g))
        assert np.all(np.abs(g - w) <= REL * np.abs(w))
        assert np.array_equal(g, w)                      # same kernels, same reduction order: the same bits


# (process, keyword overrides, events, points) of the two consecutive calls: the second has fewer events and more
# chunks per event than the first, so its constants and partial sums land where the first call kept other things
CASES = [
    ((3, {}, 203, 5000), (3, {}, 37, 70001)),                        # headline process, ragged sizes
    ((4, {}, 61, 9000), (3, dict(n_perm=4), 29, 3001)),              # lane-compacting kernel, then an assignment sum
    ((1, {}, 64, 1 << 16), (5, {}, 19, 12345)),                      # config 1 at full size, then NEXT-4
]


@pytest.mark.parametrize("first,second", CASES)
def test_two_calls_in_a_row_match_mem_integrate(mem, first, second):
    import torch
    for k, (proc, over, ne, npts) in enumerate((first, second)):
        ev = _events(proc, ne, seed=11 + k)
        with mem.Integrator(proc, **over) as it:
            want = it.integrate(ev, npts, SEED)                      # existing path, its own cudaMalloc'd workspace
            got = it.integrate_noalloc(ev, npts, SEED, *_outs(ne))   # fixed array, whatever the last call left in it
            torch.cuda.synchronize()
            _same(got, want)


def test_event_offset_and_side_stream(mem):
    import torch
    proc, ne, npts = 3, 50, 4099
    ev = _events(proc, ne, seed=5)
    s = torch.cuda.Stream()
    with mem.Integrator(proc) as it:
        it.set_event_offset(1000)
        want = it.integrate(ev, npts, SEED)
        torch.cuda.synchronize()
        p, e = _outs(ne)
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            it.integrate_noalloc(ev, npts, SEED, p, e, stream=s)
        s.synchronize()
        _same((p, e), want)


def test_device_memory_does_not_move(mem):
    """Free device memory as the driver reports it is the same before and after no-alloc calls, each larger than
    any before (the ordinary path would have regrown its workspace for them)."""
    import torch
    proc = 3
    sizes = [(16, 3000), (400, 40000), (1500, 1 << 18)]
    evs = [_events(proc, ne, seed=21 + k) for k, (ne, _) in enumerate(sizes)]
    outs = [_outs(ne) for ne, _ in sizes]
    with mem.Integrator(proc) as it:
        it.integrate_noalloc(evs[0], sizes[0][1], SEED, *outs[0])    # first call on the device: address look-up, module load
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        for ev, (ne, npts), (p, e) in zip(evs, sizes, outs):
            it.integrate_noalloc(ev, npts, SEED, p, e)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0
        want = it.integrate(evs[1], sizes[1][1], SEED)
        torch.cuda.synchronize()
        _same(outs[1], want)


def test_limits_are_enforced(mem):
    import torch
    # 4096 events x 2^20 points of the headline process fit (5.4 MiB); 8192 do not
    assert mem.MEM_NOALLOC_SCRATCH_BYTES == 8 << 20
    ne = 8192
    ev = _events(3, ne, seed=1)
    p, e = _outs(ne)
    with mem.Integrator(3) as it:
        with pytest.raises(mem.MemError) as ei:
            it.integrate_noalloc(ev, 1 << 20, SEED, p, e)
        assert ei.value.status == mem.MEM_ERR_INVALID_ARG
        assert "bytes of scratch" in str(ei.value) and str(8 << 20) in str(ei.value)
        torch.cuda.synchronize()
        assert bool(torch.isnan(p).all())                            # rejected before anything was launched
        it.integrate_noalloc(ev, 1 << 12, SEED, p, e)                # the same events with fewer blocks per event fit
        torch.cuda.synchronize()
        _same((p, e), it.integrate(ev, 1 << 12, SEED))
    with mem.Integrator(3, vegas_iters=2, vegas_points=3000) as it:
        with pytest.raises(mem.MemError) as ei:
            it.integrate_noalloc(ev[:, :8].contiguous(), 4096, SEED, p[:8], e[:8])
        assert ei.value.status == mem.MEM_ERR_UNSUPPORTED
