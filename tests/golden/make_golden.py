"""Writes tests/golden/oracle_values.txt: per-event estimates of the CPU oracle on small seeded cases.

Calls only oracle/ and the input generators (paper_1407_7595_b200.workloads holds no method
arithmetic).  The stored values are a regression pin of the oracle itself (they detect an
accidental change of its arithmetic) and a second reference for the GPU parity tests; they are
not independent evidence.  Run from the repository root:  python tests/golden/make_golden.py
"""
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1407_7595_b200 import workloads as wl  # noqa: E402

SEED = 20140729
# (label, process, oracle-parameter overrides, events, points)
CASES = [
    ("config1", 1, {}, 3, 4000),
    ("config2", 2, {}, 3, 4000),
    ("config3", 3, {}, 3, 4000),
    ("config3_perm24", 3, {"n_perm": 24}, 2, 1500),
    ("config4", 4, {}, 6, 4000),
    ("config4_perm2", 4, {"n_perm": 2}, 6, 2000),
    ("config5_vegas", 3, {"vegas_iters": 2, "vegas_points": 3000}, 2, 4000),
]


def compute(label, proc, over, ne, n_points):
    p = oracle.params_default(proc)
    for k, v in over.items():
        setattr(p, k, v)
    ev = wl.make_events(proc, ne, seed=77)
    if p.vegas_iters:
        return oracle.vegas_integrate(proc, p, ev, n_points, SEED)
    return oracle.integrate(proc, p, ev, n_points, SEED)


def main():
    oracle.build()
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_values.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py (oracle only); label event p err\n")
        for label, proc, over, ne, n_points in CASES:
            pm, pe = compute(label, proc, over, ne, n_points)
            for e in range(ne):
                f.write("%s %d %.17e %.17e\n" % (label, e, pm[e], pe[e]))
    print("wrote", out)


if __name__ == "__main__":
    main()
