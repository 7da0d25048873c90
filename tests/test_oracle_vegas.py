"""Pins of the oracle's VEGAS grid (config 5; readings A14) -- CPU only.

The algorithm constants (smoothing, alpha, final-pass-only estimate) are readings, hence
"parity unpinned"; what is pinned here are the properties any correct importance-sampling
grid must have, and agreement of the adapted estimate with plain MC and with a closed form.
"""
import math

import numpy as np

import oracle

HARD = np.array([[60., 0.3, 1.0, 140., -0.4, 2.5, 110., 0.8, 0.2, 90., 0.1, 4.0, 70., -1.0, 5.2, 50., 3.3]]).T


def test_map_is_a_monotone_bijection_with_unit_jacobian_integral():
    rng = np.random.default_rng(1)
    B, D = 50, 3
    edges = np.sort(rng.random((D, B + 1)), axis=1)
    edges[:, 0], edges[:, -1] = 0.0, 1.0
    us = np.linspace(1e-9, 1 - 1e-9, 4001)
    zs = np.array([oracle.vegas_map(edges, [u] * D)[0] for u in us])
    assert np.all(np.diff(zs, axis=0) > 0)
    assert np.allclose(zs[0], 0, atol=1e-7) and np.allclose(zs[-1], 1, atol=1e-7)
    # jac = prod_d dz_d/du_d = prod_d B * width[k_d]; in-bin position is linear
    u = [0.123, 0.5, 0.987]
    z, k, jac = oracle.vegas_map(edges, u)
    assert list(k) == [int(x * B) for x in u]
    assert math.isclose(jac, np.prod([B * (edges[d, k[d] + 1] - edges[d, k[d]]) for d in range(D)]), rel_tol=1e-14)
    for d in range(D):
        frac = u[d] * B - k[d]
        assert math.isclose(z[d], edges[d, k[d]] + frac * (edges[d, k[d] + 1] - edges[d, k[d]]), rel_tol=1e-14)
    # u = 1 - 2^-53 stays in the last bin
    assert oracle.vegas_map(edges, [1 - 2.0 ** -53] * D)[1].tolist() == [B - 1] * D


def test_refine_invariants():
    rng = np.random.default_rng(2)
    B = 50
    uniform = np.arange(B + 1) / B
    # (ii) constant histogram: grid stays uniform;  zero histogram: grid untouched
    assert np.allclose(oracle.vegas_refine(np.full(B, 3.7), uniform, 0.5), uniform, rtol=0, atol=1e-14)
    assert np.array_equal(oracle.vegas_refine(np.zeros(B), uniform, 0.5), uniform)
    # (i) random, spiky and sparse histograms: edges strictly monotone, ends fixed
    for trial in range(20):
        h = rng.random(B) ** 8
        if trial % 3 == 0:
            h[rng.random(B) < 0.7] = 0.0
        e = uniform
        for _ in range(4):
            e = oracle.vegas_refine(h, e, 0.5)
            assert e[0] == 0.0 and e[-1] == 1.0
            assert np.all(np.diff(e) > 0)
    # alpha = 0 compresses every non-empty bin to 1: with all bins hit the grid stays where it is
    assert np.allclose(oracle.vegas_refine(rng.random(B) + 0.1, uniform, 0.0), uniform, atol=1e-14)
    # a single hot bin attracts edges: bins get narrower there
    h = np.full(B, 1e-6)
    h[10] = 1.0
    e = oracle.vegas_refine(h, uniform, 0.5)
    assert (e[11] - e[10]) < 1.0 / B / 2 or np.searchsorted(e, 0.21) - np.searchsorted(e, 0.20) >= 2


def test_grid_converges_on_a_peaked_function():
    """(iii) f(x) = 1/((x-0.3)^2 + 1e-4): the standard error drops and the estimate stays within
    errors of the closed form (SURVEY.md 8(c) probe: 14.0 -> 2.0 over six passes)."""
    a, c = 0.3, 1e-2
    exact = (math.atan((1 - a) / c) + math.atan(a / c)) / c
    B, N = 50, 1 << 13
    e = np.arange(B + 1) / B
    rng = np.random.default_rng(3)
    errs = []
    for it in range(7):
        u = rng.random(N)
        k = np.minimum((u * B).astype(int), B - 1)
        # map check against the oracle on a few points, then vectorised
        for i in range(3):
            z_o, k_o, j_o = oracle.vegas_map(e.reshape(1, -1), [u[i]])
            assert k_o[0] == k[i]
        width = e[k + 1] - e[k]
        z = e[k] + (u * B - k) * width
        w = B * width / ((z - a) ** 2 + c * c)
        est, err = w.mean(), w.std(ddof=1) / math.sqrt(N)
        errs.append(err)
        assert abs(est - exact) < 5 * err
        h = np.bincount(k, weights=w * w, minlength=B)
        e = oracle.vegas_refine(h, e, 0.5)
        assert np.all(np.diff(e) > 0)
    assert errs[-1] < 0.25 * errs[0]
    # equal-mass property: bins are much narrower at the peak than far from it
    widths = np.diff(e)
    assert widths[np.searchsorted(e, a) - 1] < 0.2 * widths.max()


def test_vegas_agrees_with_plain_mc_on_config3():
    """(iv) same integral, smaller error."""
    p = oracle.params_default(3)
    plain, plain_err = oracle.integrate(3, p, HARD, 1 << 16, 77)
    p.vegas_iters, p.vegas_points = 5, 1 << 13
    veg, veg_err, grid = oracle.vegas_integrate(3, p, HARD, 1 << 14, 77, return_grid=True)
    assert abs(veg[0] - plain[0]) < 4 * math.hypot(veg_err[0], plain_err[0])
    assert veg_err[0] * math.sqrt(1 << 14) < plain_err[0] * math.sqrt(1 << 16)   # lower variance per point
    assert grid.shape == (1, 6, 51)
    assert np.all(np.diff(grid, axis=2) > 0) and np.all(grid[:, :, 0] == 0) and np.all(grid[:, :, -1] == 1)
    # iters = 0 reproduces plain MC bit for bit (uniform grid, iteration counter 0)
    p.vegas_iters = 0
    v0, e0 = oracle.vegas_integrate(3, p, HARD, 1 << 10, 77)
    m0, me0 = oracle.integrate(3, p, HARD, 1 << 10, 77)
    assert math.isclose(v0[0], m0[0], rel_tol=1e-13) and math.isclose(e0[0], me0[0], rel_tol=1e-10)
    # eval_points through a grid equals jac * weight at the warped point
    p.vegas_iters = 5
    w = oracle.eval_points(3, p, HARD, 0, 5, 4, 77, iteration=5, grid=grid)
    for i in range(4):
        u = oracle.uniforms(77, 0, 5 + i, 5, 6)
        z, _, jac = oracle.vegas_map(grid[0], u)
        assert math.isclose(w[i], jac * oracle.weight(3, p, HARD[:, 0], z), rel_tol=1e-14, abs_tol=0)
