"""Host-side checks of the C-ABI library that need no GPU: it builds, loads, exports every symbol
include/mem.h declares, its parameter struct matches the Python mirror, and the device entry
points fail loudly (no CPU fallback) when there is no CUDA device."""
import ctypes as C
import os
import re

import pytest

import paper_1407_7595_b200 as mem

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    """every function declared by a header under include/ (mem.h: the integrator; mem_bench.h: microbenchmarks)"""
    names = set()
    inc = os.path.join(ROOT, "include")
    for f in sorted(os.listdir(inc)):
        if f.endswith(".h"):
            text = re.sub(r"/\*.*?\*/", "", open(os.path.join(inc, f)).read(), flags=re.S)
            names |= set(re.findall(r"\b(mem_[a-z0-9_]+)\s*\(", text))
    return sorted(names)


def test_microbenchmarks_are_not_in_the_integrator_header():
    text = open(os.path.join(ROOT, "include", "mem.h")).read()
    assert "mem_measure_fp64_rate" not in text and "mem_measure_fp64_peak_rrr" not in text
    assert "mem_measure_fp64_peak(" in text                       # the roofline denominator stays


def test_library_builds_and_exports_every_declared_symbol():
    lib = mem.lib()
    names = _declared_symbols()
    assert set(names) == set(mem.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n


def test_params_struct_matches_header_and_defaults():
    for proc, nf, nd in ((1, 5, 1), (2, 6, 2), (3, 17, 6), (4, 14, 8), (5, 18, 8)):
        p = mem.mem_params_default(proc)
        assert p.struct_size == C.sizeof(mem.mem_params)
        assert p.precision == 64 and p.vegas_iters == 0 and p.vegas_bins == 50
        assert (p.sqrt_s, p.m_W, p.Gam_W, p.m_t, p.Gam_t) == (14000.0, 80.4, 2.09, 173.0, 1.4)   # BASELINE.json:configs
        assert (p.tf_w_tail, p.tf_sig1, p.tf_mu2, p.tf_sig2) == (0.3, 0.15, -0.1, 0.35)
        assert p.n_flav == (3 if proc == 2 else 5)
        assert mem.mem_event_fields(proc) == nf and mem.mem_n_dims(proc) == nd
        assert (p.m_H, p.Gam_H, p.tth_hyp, p.reserved0) == (125.0, 0.00407, 0, 0) and 0.99 < p.yuk_t < 1.0    # reading A21
    assert mem.mem_event_fields(7) == -1
    with pytest.raises(mem.MemError):
        mem.mem_params_default(0)


def test_every_python_field_is_in_the_header_in_order():
    text = open(os.path.join(ROOT, "include", "mem.h")).read()
    start = text.index("typedef struct mem_params {") + len("typedef struct mem_params {")
    body = text[start:text.index("} mem_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        m = re.match(r"\s*(?:uint32_t|int32_t|int64_t|double)\s+(.*)", decl.strip(), flags=re.S)
        if m:
            names += [n.strip() for n in m.group(1).split(",")]
    assert names == [f[0] for f in mem.mem_params._fields_]


def test_reserved_field_must_be_zero():
    # include/mem.h: "reserved0 must be 0"; rejected by the parameter check, before any CUDA call
    p = mem.mem_params_default(mem.MEM_PROC_TT_LJETS)
    p.reserved0 = 1
    with pytest.raises(mem.MemError) as ei:
        mem.mem_create(mem.MEM_PROC_TT_LJETS, p)
    assert ei.value.status == mem.MEM_ERR_INVALID_ARG and "reserved0" in str(ei.value)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(mem.MemError) as ei:
        mem.mem_create(mem.MEM_PROC_TT_LJETS)
    assert ei.value.status == mem.MEM_ERR_CUDA
    assert mem.mem_last_error() != ""


def test_product_package_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1407_7595_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "mem_oracle" not in src, f
