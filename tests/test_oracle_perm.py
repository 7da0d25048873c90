"""Pins of the oracle's jet-permutation sum (NEXT-1; Eq. 7: "The outer sum is over
all permutations of assigning measured jets to partons in the matrix element").

The definition is written out here with itertools on top of the single-assignment weight, and the
symmetry it implies is checked independently: the summed weight cannot depend on the order in
which the jets are listed in the record.
"""
import itertools
import math

import numpy as np
import pytest

import oracle
from paper_1407_7595_b200 import workloads as wl

SEED = 20140729


def setup_module(module):
    oracle.build()


def _permute(rec, first_jet, sigma):
    r = rec.copy()
    for role, j in enumerate(sigma):
        r[first_jet + 3 * role:first_jet + 3 * role + 3] = rec[first_jet + 3 * j:first_jet + 3 * j + 3]
    return r


def _live_points(proc, p, ev, n_try, want):
    out = []
    D = oracle.n_dims(proc)
    for e in range(ev.shape[1]):
        for i in range(n_try):
            u = oracle.uniforms(SEED, e, i, 0, D)
            if oracle.weight(proc, p, ev[:, e], u) > 0:
                out.append((ev[:, e].copy(), np.array(u)))
                break
        if len(out) >= want:
            break
    assert len(out) >= want
    return out


@pytest.mark.parametrize("proc,n_perm,first_jet,sigmas", [
    (3, 24, 3, list(itertools.permutations(range(4)))),
    (3, 4, 3, [(0, 1, 2, 3), (0, 1, 3, 2), (1, 0, 2, 3), (1, 0, 3, 2)]),
    (4, 2, 6, [(0, 1), (1, 0)]),
])
def test_sum_is_the_definition_written_out(proc, n_perm, first_jet, sigmas):
    base = oracle.params_default(proc)
    assert base.n_perm == 0
    summed = oracle.params_default(proc)
    summed.n_perm = n_perm
    ev = wl.make_events(proc, 40, seed=21)
    for rec, u in _live_points(proc, base, ev, 3000, 6):
        terms = [oracle.weight(proc, base, _permute(rec, first_jet, s), u) for s in sigmas]
        got = oracle.weight(proc, summed, rec, u)
        assert math.isclose(got, math.fsum(terms), rel_tol=1e-13)
        assert got >= terms[0] > 0
        one = oracle.params_default(proc)
        one.n_perm = 1
        assert oracle.weight(proc, one, rec, u) == terms[0]


def test_full_sum_does_not_depend_on_the_jet_order_in_the_record():
    p = oracle.params_default(3)
    p.n_perm = 24
    base = oracle.params_default(3)
    ev = wl.make_events(3, 40, seed=22)
    rng = np.random.default_rng(1)
    for rec, u in _live_points(3, base, ev, 3000, 5):
        w0 = oracle.weight(3, p, rec, u)
        for _ in range(4):
            sigma = rng.permutation(4)
            # reorder the record AND move the energy variables with the jets: parton role r keeps u_r,
            # so the same set of (jet, role, u) triples is covered
            w1 = oracle.weight(3, p, _permute(rec, 3, sigma), u)
            assert math.isclose(w1, w0, rel_tol=1e-12)


def test_btag_sum_symmetries_and_ordering_of_sums():
    p4, p24, p1 = (oracle.params_default(3) for _ in range(3))
    p4.n_perm, p24.n_perm, p1.n_perm = 4, 24, 1
    ev = wl.make_events(3, 40, seed=23)
    for rec, u in _live_points(3, p1, ev, 3000, 5):
        w4 = oracle.weight(3, p4, rec, u)
        assert math.isclose(oracle.weight(3, p4, _permute(rec, 3, (1, 0, 2, 3)), u), w4, rel_tol=1e-12)
        assert math.isclose(oracle.weight(3, p4, _permute(rec, 3, (0, 1, 3, 2)), u), w4, rel_tol=1e-12)
        assert oracle.weight(3, p1, rec, u) <= w4 <= oracle.weight(3, p24, rec, u)


def test_dilepton_sum_is_symmetric_in_the_two_jets():
    p = oracle.params_default(4)
    p.n_perm = 2
    base = oracle.params_default(4)
    ev = wl.make_events(4, 60, seed=24)
    for rec, u in _live_points(4, base, ev, 4000, 5):
        w = oracle.weight(4, p, rec, u)
        assert math.isclose(oracle.weight(4, p, _permute(rec, 6, (1, 0)), u), w, rel_tol=1e-12)


def test_integral_with_permutations():
    """the estimator consumes the same points: p(24) >= p(4) >= p(1), and eval_points agrees with weight"""
    ev = wl.make_events(3, 3, seed=25)
    res = {}
    for n in (1, 4, 24):
        p = oracle.params_default(3)
        p.n_perm = n
        res[n] = oracle.integrate(3, p, ev, 3000, SEED)[0]
    assert np.all(res[24] >= res[4]) and np.all(res[4] >= res[1]) and np.all(res[24] > 0)
    p = oracle.params_default(3)
    p.n_perm = 24
    w = oracle.eval_points(3, p, ev, 1, 0, 50, SEED)
    for i in (0, 7, 49):
        assert w[i] == oracle.weight(3, p, ev[:, 1], oracle.uniforms(SEED, 1, i, 0, 6))
