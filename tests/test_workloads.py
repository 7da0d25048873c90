"""The seeded input generators (paper_1407_7595_b200/workloads.py) and the counts bookkeeping: shapes, determinism,
the physical content the closure generator promises, the generator density used by the normalisation (reading A22)."""
import json
import os

import numpy as np
import pytest

from helpers import mdot
from paper_1407_7595_b200 import counts
from paper_1407_7595_b200 import workloads as wl


def test_records_are_seeded_and_shaped():
    for proc in (wl.W_ENU, wl.Z_BB, wl.TT_LJETS, wl.TT_DILEP, wl.TTH_DILEP):
        a, b = wl.make_events(proc, 33), wl.make_events(proc, 33)
        assert a.shape == (wl.N_FIELDS[proc], 33) and a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
        assert np.array_equal(a, b) and not np.array_equal(a, wl.make_events(proc, 33, seed=1))
        assert np.array_equal(wl.make_events(proc, 40)[:, :0], a[:, :0])
    t = wl.make_tth_events(17)
    assert t.shape == (18, 17) and np.array_equal(t, wl.make_tth_events(17))
    assert not np.array_equal(t, wl.make_tth_events(17, resonant=False))


def test_closure_records_are_physical_tth_configurations():
    ev, tr = wl.make_tth_events(200, smear=False, return_truth=True)
    P = sum(tr[k] for k in ("lp", "nu", "b", "lm", "nub", "bb", "b1", "b2"))
    assert np.max(np.abs(P[1:3])) < 1e-9 * np.max(P[0])                       # balanced in the transverse plane
    mbb = np.sqrt(mdot(tr["b1"] + tr["b2"], tr["b1"] + tr["b2"]))
    assert np.allclose(mbb, 125.0, rtol=1e-9)                                 # resonant sample: m_bb = m_H
    mt = np.sqrt(mdot(tr["lp"] + tr["nu"] + tr["b"], tr["lp"] + tr["nu"] + tr["b"]))
    mw = np.sqrt(mdot(tr["lm"] + tr["nub"], tr["lm"] + tr["nub"]))
    assert np.all(np.abs(mt - 173.0) <= 15 * 1.4 + 1e-6) and np.all(np.abs(mw - 80.4) <= 15 * 2.09 + 1e-6)
    for k in ("lp", "nu", "b", "b1"):
        assert np.max(np.abs(mdot(tr[k], tr[k]))) < 1e-6 * np.max(tr[k][0]) ** 2    # massless
    # the record holds the unsmeared jets: E, eta, phi of b reproduce its three-momentum
    E, eta, phi = ev[6], ev[7], ev[8]
    assert np.allclose(E * np.tanh(eta), tr["b"][3], rtol=1e-9) and np.allclose(E / np.cosh(eta) * np.cos(phi), tr["b"][1], rtol=1e-9, atol=1e-9)
    bkg = wl.make_tth_events(200, resonant=False, smear=False, return_truth=True)[1]
    mb = np.sqrt(mdot(bkg["b1"] + bkg["b2"], bkg["b1"] + bkg["b2"]))
    assert mb.min() >= 20.0 - 1e-9 and mb.max() <= 300.0 + 1e-9 and mb.std() > 30.0


def test_smearing_follows_the_double_gaussian_shape():
    r = np.random.Generator(np.random.PCG64(5))
    E = np.full(400000, 100.0)
    x = wl._smear_jet(r, E) / E - 1.0
    # mixture mean and variance: (1-w) N(0, 0.15) + w N(-0.1, 0.35), w = 0.3
    assert x.mean() == pytest.approx(0.3 * -0.1, abs=2e-3)
    assert x.var() == pytest.approx(0.7 * 0.15 ** 2 + 0.3 * (0.35 ** 2 + 0.01) - 0.03 ** 2, rel=0.02)


def test_event_density_integrates_to_one():
    # importance-sample the density with a different proposal: E[g(X)/q(X)] = 1 for X ~ q covering the support
    rng = np.random.default_rng(1)
    n = 200000
    ev = np.empty((18, n))
    q = np.ones(n)
    for k in range(2):
        ev[3 * k] = 20.0 + rng.exponential(60.0, n); q *= np.exp(-(ev[3 * k] - 20.0) / 60.0) / 60.0
        ev[3 * k + 1] = rng.uniform(-2.5, 2.5, n); ev[3 * k + 2] = rng.uniform(0, 2 * np.pi, n); q *= 1 / 5.0 / (2 * np.pi)
    for k in range(4):
        ev[6 + 3 * k] = 30.0 + rng.exponential(90.0, n); q *= np.exp(-(ev[6 + 3 * k] - 30.0) / 90.0) / 90.0
        ev[7 + 3 * k] = rng.uniform(-2.5, 2.5, n); ev[8 + 3 * k] = rng.uniform(0, 2 * np.pi, n); q *= 1 / 5.0 / (2 * np.pi)
    ratio = wl.event_density(wl.TTH_DILEP, ev) / q
    assert ratio.mean() == pytest.approx(1.0, abs=5 * ratio.std() / np.sqrt(n))
    with pytest.raises(ValueError):
        wl.event_density(wl.TT_DILEP, wl.make_events(wl.TT_DILEP, 4))


def test_shard_ranges_cover_the_bench_layout():
    assert [wl.shard_range(10, r, 3) for r in range(3)] == [(0, 4), (4, 7), (7, 10)]


def test_executed_counts_file_is_consistent():
    data = json.load(open(counts.PATH))
    assert set(data) <= set(counts.KERNELS)
    for key, rec in data.items():
        assert rec["kernel"] == counts.KERNELS[key] and len(rec["sass_sha256"]) == 64 and rec["points_per_launch"] > 0
        assert sum(rec.get(k, 0.0) for k in ("dfma", "dmul", "dadd", "ffma", "fmul", "fadd")) > 50
    # the stored hash is the one of the library as built from the committed sources
    rec = counts.lookup(3, 1, 64)
    assert rec is not None and rec["match"] in (True, None), "fp64_counts.json was measured on another build of the config-3 kernel"
    assert os.path.basename(counts.PATH) == "fp64_counts.json"
