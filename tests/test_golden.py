"""Regression pins: the oracle (CPU) and the CUDA path (GPU) against the values stored by
tests/golden/make_golden.py (a committed script that calls only oracle/)."""
import importlib.util
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
mg = importlib.util.module_from_spec(spec)
spec.loader.exec_module(mg)


def _stored():
    vals = {}
    for line in open(os.path.join(HERE, "golden", "oracle_values.txt")):
        if line.startswith("#"):
            continue
        label, e, p, err = line.split()
        vals.setdefault(label, []).append((float(p), float(err)))
    return {k: np.array(v) for k, v in vals.items()}


@pytest.mark.parametrize("case", mg.CASES, ids=[c[0] for c in mg.CASES])
def test_oracle_reproduces_its_stored_values(case):
    """1e-10: the platform libm may differ in the last bits between machines"""
    mg.oracle.build()
    pm, pe = mg.compute(*case)
    ref = _stored()[case[0]]
    assert np.all(np.abs(pm - ref[:, 0]) <= 1e-10 * np.abs(ref[:, 0]))
    assert np.all(np.abs(pe - ref[:, 1]) <= 1e-10 * np.abs(ref[:, 1]))


@pytest.mark.gpu
@pytest.mark.parametrize("case", mg.CASES, ids=[c[0] for c in mg.CASES])
def test_cuda_path_reproduces_the_stored_values(case):
    import torch

    import paper_1407_7595_b200 as mem
    from paper_1407_7595_b200 import workloads as wl
    label, proc, over, ne, n_points = case
    ev = torch.from_numpy(wl.make_events(proc, ne, seed=77)).cuda()
    with mem.Integrator(proc, **over) as it:
        p, err = it.integrate(ev, n_points, mg.SEED)
    ref = _stored()[label]
    assert np.all(np.abs(p.cpu().numpy() - ref[:, 0]) <= 1e-9 * np.abs(ref[:, 0]))
    assert np.all(np.abs(err.cpu().numpy() - ref[:, 1]) <= 1e-9 * np.abs(ref[:, 1]) + 1e-300)
