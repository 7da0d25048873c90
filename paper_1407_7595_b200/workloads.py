"""Seeded synthetic event generators shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no Philox, no matrix element, no
transfer function): it only draws event records with the shapes BASELINE.json's configs
state.  It stands in for the paper's MadGraph+Pythia samples
(PAPER.md:145), which are not available.  It imports neither the CUDA binding nor the
oracle.

Records are float64, SoA, field-major: shape [n_fields, n_events].
Only numpy.random.Generator(PCG64).random() is used (a stable stream); exponential and
normal variates are derived here by inversion / Box-Muller so that numpy version changes
cannot alter the events.
"""
from __future__ import annotations

import numpy as np

DEFAULT_SEED = 20140729

W_ENU, Z_BB, TT_LJETS, TT_DILEP = 1, 2, 3, 4
N_FIELDS = {W_ENU: 5, Z_BB: 6, TT_LJETS: 17, TT_DILEP: 14}
N_DIMS = {W_ENU: 1, Z_BB: 2, TT_LJETS: 6, TT_DILEP: 8}

# BASELINE.json:configs[0..3]: (process, n_events, n_points)
CONFIGS = {
    1: (W_ENU, 64, 1 << 16),
    2: (Z_BB, 1024, 1 << 18),
    3: (TT_LJETS, 4096, 1 << 20),
    4: (TT_DILEP, 16384, 1 << 18),
}


def _rng(seed, process):
    return np.random.Generator(np.random.PCG64([int(seed), int(process)]))


def _exp(u, mean):
    return -mean * np.log1p(-u)


def _lepton(r, n):
    """lepton pT ~ Exp(40 GeV) + 20, eta ~ U(-2.5, 2.5), phi ~ U(0, 2 pi)  (configs[0])."""
    return 20.0 + _exp(r.random(n), 40.0), -2.5 + 5.0 * r.random(n), 2.0 * np.pi * r.random(n)


def _jet(r, n):
    """jet E ~ Exp(60) + 30 GeV, |eta| < 2.5, phi ~ U(0, 2 pi)  (configs[2])."""
    return 30.0 + _exp(r.random(n), 60.0), -2.5 + 5.0 * r.random(n), 2.0 * np.pi * r.random(n)


def make_events(process: int, n_events: int, seed: int = DEFAULT_SEED) -> np.ndarray:
    r = _rng(seed, process)
    n = int(n_events)
    if process == W_ENU:
        pt, eta, phi = _lepton(r, n)
        # PAPER.md:180 Eq. 11: MET = -(sum of visible transverse momenta)
        rows = [pt, eta, phi, -pt * np.cos(phi), -pt * np.sin(phi)]
    elif process == Z_BB:
        rows = [*_jet(r, n), *_jet(r, n)]
    elif process == TT_LJETS:
        rows = [*_lepton(r, n)]
        for _ in range(4):                       # b_had, b_lep, q, qbar'
            rows += [*_jet(r, n)]
        rows += [20.0 + _exp(r.random(n), 40.0), 2.0 * np.pi * r.random(n)]   # met, met_phi
    elif process == TT_DILEP:
        lp, lm = _lepton(r, n), _lepton(r, n)
        b, bb = _jet(r, n), _jet(r, n)
        vx = lp[0] * np.cos(lp[2]) + lm[0] * np.cos(lm[2])
        vy = lp[0] * np.sin(lp[2]) + lm[0] * np.sin(lm[2])
        for E, eta, phi in (b, bb):
            vx = vx + E / np.cosh(eta) * np.cos(phi)
            vy = vy + E / np.cosh(eta) * np.sin(phi)
        u1, u2 = r.random(n), r.random(n)
        rad = np.sqrt(-2.0 * np.log1p(-u1))      # Box-Muller
        rows = [*lp, *lm, *b, *bb, -vx + 10.0 * rad * np.cos(2 * np.pi * u2),
                -vy + 10.0 * rad * np.sin(2 * np.pi * u2)]
    else:
        raise ValueError("unknown process %r" % (process,))
    ev = np.ascontiguousarray(np.stack(rows, axis=0), dtype=np.float64)
    assert ev.shape == (N_FIELDS[process], n)
    return ev


def shard_range(n_events: int, rank: int, world: int):
    """Contiguous event range of `rank`: events are independent units."""
    base, rem = divmod(int(n_events), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
