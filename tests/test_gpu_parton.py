"""GPU parity of the parton-level mode (NEXT-2; Table 2) against the CPU oracle."""
import numpy as np
import pytest

import oracle
from paper_1407_7595_b200 import workloads as wl

pytestmark = pytest.mark.gpu


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


@pytest.mark.parametrize("n_perm,n_events", [(1, 1), (1, 1000 + 37), (4, 777), (24, 5000 + 13)])
def test_parton_parity(mem, n_perm, n_events):
    """element by element, several 128-thread tiles and a ragged tail.  Tolerance (DESIGN.md "Parton-level
    mode"): the top propagators are formed from the momenta, s_t - m_t^2 = p_t^2 - m_t^2 with p_t^2 a
    difference of squares of size E_t^2, next to a pole of width m_t Gamma_t; one rounding of relative size
    2^-53 in E_t^2 moves D_t by 2^-53 E_t^2 / (m_t Gamma_t) on either side.  Bar against the long-double
    referee: 1e-12 + 16 * 2^-53 (E_t^2 + E_tbar^2) / (m_t Gamma_t); the median error must stay below 3e-13."""
    ev = wl.make_parton_events(n_events, seed=3 + n_perm)
    p = oracle.params_default(3)
    p.n_perm = n_perm
    wo = oracle.parton_weights(3, p, ev)
    wx = oracle.parton_weights(3, p, ev, extended=True)
    with mem.Integrator(3, n_perm=n_perm) as it:
        wg = it.eval_parton(_dev(ev)).cpu().numpy()
    assert np.array_equal(wg == 0, wo == 0) and np.all(wo > 0)
    m = ev.reshape(6, 4, -1)
    Et, Etb = m[0, 0] + m[1, 0] + m[3, 0], m[2, 0] + m[4, 0] + m[5, 0]
    tol = 1e-12 + 16 * 2.0 ** -53 * (Et ** 2 + Etb ** 2) / (p.m_t * p.Gam_t)
    rel = np.abs(wg - wx) / wx
    assert np.all(rel <= tol), (rel / tol).max()
    if n_events >= 100:
        assert np.median(rel) <= 3e-13
    assert np.all(np.abs(wg - wo) <= tol * wo + 2.0 * np.abs(wo - wx))


def test_parton_cuts_offsets_and_errors(mem):
    import torch
    ev = wl.make_parton_events(300, seed=9)
    # configurations pushed out of the allowed region: x > 1 (scaled up), below threshold (scaled down),
    # unbalanced events (one jet's transverse momentum flipped: O7 boosts, weight stays finite)
    big, small, kick = ev.copy(), ev.copy(), ev.copy()
    big[:, :100] *= 40.0
    small[:, :100] *= 0.02
    kick[9, :] *= -1.0
    p = oracle.params_default(3)
    with mem.Integrator(3) as it:
        for arr in (big, small, kick):
            wo = oracle.parton_weights(3, p, arr)
            wg = it.eval_parton(_dev(arr)).cpu().numpy()
            assert np.array_equal(wg == 0, wo == 0)
            nz = wo != 0
            assert np.max(np.abs(wg[nz] - wo[nz]) / wo[nz]) <= 1e-9      # fp64 vs fp64 next to the top pole; cuts are the point here
        assert np.all(oracle.parton_weights(3, p, big)[:100] == 0) and np.all(oracle.parton_weights(3, p, small)[:100] == 0)
        n0 = it.launches
        out = it.eval_parton(torch.empty((24, 0), dtype=torch.float64, device="cuda"))
        assert out.numel() == 0 and it.launches == n0
    for proc in (1, 2, 4):
        with mem.Integrator(proc) as it:
            with pytest.raises(mem.MemError) as ei:
                it.eval_parton(_dev(ev))
            assert ei.value.status == mem.MEM_ERR_UNSUPPORTED
    with mem.Integrator(3, precision=32) as it:
        with pytest.raises(mem.MemError):
            it.eval_parton(_dev(ev))


def test_parton_full_size(mem):
    """the paper's parton-level experiment size, 10^5 events, all 24 assignments; a
    sample of outputs recomputed by the oracle one by one"""
    n = 100000
    ev = wl.make_parton_events(n)
    p = oracle.params_default(3)
    p.n_perm = 24
    with mem.Integrator(3, n_perm=24) as it:
        wg = it.eval_parton(_dev(ev)).cpu().numpy()
    assert np.all(np.isfinite(wg)) and np.all(wg > 0)
    idx = np.random.default_rng(2).choice(n, 200, replace=False)
    wo = oracle.parton_weights(3, p, ev[:, idx])
    assert np.max(np.abs(wg[idx] - wo) / wo) <= 1e-11
