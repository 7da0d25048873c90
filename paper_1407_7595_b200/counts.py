"""Executed FP64 instruction counts per integrand call, tied to the kernel build they were measured on.

`fp64_counts.json` (beside this file) holds, per integrate kernel, the thread-level DFMA / DMUL / DADD (or FFMA /
FMUL / FADD) instructions per sample point from an ncu metric pass, together with the SHA-256 of that kernel's SASS
(`cuobjdump -sass -fun <kernel>` of the in-tree library).  bench.py reads the counts for its "executed" roofline
figures and recomputes the hash of the kernel it is about to time: a count taken on another build is reported as
stale instead of being silently reused (measurement item 8).

Refresh after a kernel change (on the GPU box; writes the JSON in place):

    ncu --metrics smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,\
smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,smsp__sass_thread_inst_executed_op_ffma_pred_on.sum,\
smsp__sass_thread_inst_executed_op_fmul_pred_on.sum,smsp__sass_thread_inst_executed_op_fadd_pred_on.sum \
        --clock-control none -k regex:integrate_kernel --csv --log-file gpurun_out/counts_c3.csv \
        python bench.py --config 3 --events 592 --points 65536 --steps 1 --warmup 3 --no-cpu-baseline
    python -m paper_1407_7595_b200.counts --update gpurun_out/counts_c3.csv --key 3,1,64 --points 38797312

No arithmetic of the method lives here.
"""
from __future__ import annotations

import csv
import hashlib
import json
import os
import re
import subprocess
import sys

from . import build as _build

HERE = os.path.dirname(os.path.abspath(__file__))
PATH = os.path.join(HERE, "fp64_counts.json")

# key "config,assignments,precision" -> substring of the mangled name of the kernel whose launch dominates that
# workload (integrate_kernel<P, MODE, PERM, GRIDPDF>; MODE 0 = plain, 1 = VEGAS final pass)
KERNELS = {
    "1,1,64": "integrate_kernelINS_8ProcWenuELi0ELb0ELb0E",
    "2,1,64": "integrate_kernelINS_7ProcZbbELi0ELb0ELb0E",
    "3,1,64": "integrate_kernelINS_12ProcTTljetsRIdEELi0ELb0ELb0E",
    "3,24,64": "integrate_kernelINS_12ProcTTljetsRIdEELi0ELb1ELb0E",
    "3,1,32": "integrate_kernelINS_12ProcTTljetsRIfEELi0ELb0ELb0E",
    "4,1,64": "integrate_kernelINS_11ProcTTdilepELi0ELb0ELb0E",
    "4,2,64": "integrate_kernelINS_11ProcTTdilepELi0ELb1ELb0E",
    "5,1,64": "integrate_kernelINS_12ProcTTljetsRIdEELi1ELb0ELb0E",
    "5,1,32": "integrate_kernelINS_12ProcTTljetsRIfEELi1ELb0ELb0E",
    "6,1,64": "integrate_kernelINS_12ProcTTHdilepELi0ELb0ELb0E",
    "6,1,64,h1": "integrate_kernelINS_12ProcTTHdilepELi0ELb0ELb0E",      # same kernel, hypothesis 1 (run-time switch)
    "6,12,64": "integrate_kernelINS_12ProcTTHdilepELi0ELb1ELb0E",
}
METRICS = {"dfma": "op_dfma_pred_on", "dmul": "op_dmul_pred_on", "dadd": "op_dadd_pred_on",
           "ffma": "op_ffma_pred_on", "fmul": "op_fmul_pred_on", "fadd": "op_fadd_pred_on"}


def _cuobjdump():
    for cand in ("/usr/local/cuda/bin/cuobjdump", "cuobjdump"):
        if not os.path.isabs(cand) or os.path.exists(cand):
            return cand
    return "cuobjdump"


def kernel_name(key: str, lib: str | None = None):
    """full mangled name of the kernel of `key` in the built library (None if it cannot be listed)"""
    lib = lib or _build.LIB
    try:
        out = subprocess.run([_cuobjdump(), "-elf", "-lelf", lib], capture_output=True, text=True, timeout=60).stdout
        out += subprocess.run([_cuobjdump(), "-symbols", lib], capture_output=True, text=True, timeout=60).stdout
    except (OSError, subprocess.SubprocessError):
        return None
    pat = KERNELS[key]
    for m in re.finditer(r"(_ZN7memb200\w+)", out):
        if pat in m.group(1):
            return m.group(1)
    return None


def _instruction(line: str) -> str:
    """one SASS listing line reduced to what the kernel executes: address, opcode, operands.  The encoding comment is
    dropped and the slot of constant bank 4 (where the linker keeps the addresses of the library's global arrays) is
    masked: that slot moves whenever a global is added anywhere in the library (the fixed array of
    mem_integrate_noalloc moved kExpTab's from 0x0 to 0x8) without changing a single instruction."""
    line = re.sub(r"/\*\s*0x[0-9a-f]+\s*\*/\s*$", "", line.strip()).rstrip()
    return re.sub(r"c\[0x4\]\[[^\]]*\]", "c[0x4][*]", line)


def sass_sha256(key: str, lib: str | None = None):
    """SHA-256 of the SASS listing (addresses, opcodes, operands; see _instruction) of the kernel of `key`; None if unavailable"""
    lib = lib or _build.LIB
    name = kernel_name(key, lib)
    if name is None:
        return None
    try:
        out = subprocess.run([_cuobjdump(), "-sass", "-fun", name, lib], capture_output=True, text=True,
                             timeout=120).stdout
    except (OSError, subprocess.SubprocessError):
        return None
    lines = [_instruction(l) for l in out.splitlines() if re.match(r"\s+/\*[0-9a-f]{4,}\*/", l)]
    if not lines:
        return None
    return hashlib.sha256("\n".join(lines).encode()).hexdigest()


def load():
    if not os.path.exists(PATH):
        return {}
    with open(PATH) as f:
        return json.load(f)


def lookup(config: int, perm: int = 1, precision: int = 64, check_build: bool = True, variant: str = ""):
    """counts of one kernel + "match": whether they were taken on the SASS that is built now (None = unknown)"""
    key = "%d,%d,%d" % (config, max(perm, 1), precision) + ("," + variant if variant else "")
    rec = load().get(key)
    if rec is None:
        return None
    rec = dict(rec, key=key)
    if check_build:
        h = sass_sha256(key)
        rec["match"] = None if h is None else (h == rec.get("sass_sha256"))
    return rec


def update(csv_path: str, key: str, points: int, note: str = ""):
    """parse an ncu --csv metric log, take the launch of KERNELS[key] with the most FP instructions, store per-point counts"""
    rows = list(csv.reader(l for l in open(csv_path) if l.startswith('"')))
    hdr = rows[0]
    i_name, i_metric, i_val, i_id = hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Value"), hdr.index("ID")
    cfg, perm, prec = (int(x) for x in key.split(",")[:3])
    proc = {1: "ProcWenu", 2: "ProcZbb", 3: "ProcTTljetsR", 4: "ProcTTdilep", 5: "ProcTTljetsR", 6: "ProcTTHdilep"}[cfg]
    if proc == "ProcTTljetsR":
        proc += "<double>" if prec == 64 else "<float>"
    # ncu's CSV prints the short demangled form: integrate_kernel<ProcTTljetsR<double>, 1, 0, 0>
    want = re.compile(r"integrate_kernel<(memb200::)?%s, (\(int\))?%d, (\(bool\))?%d, (\(bool\))?0>" % (re.escape(proc), 1 if cfg == 5 else 0, 1 if perm > 1 else 0))
    demangled = want.pattern
    per_launch = {}
    for r in rows[1:]:
        if not want.search(r[i_name]):
            continue
        for short, m in METRICS.items():
            if m in r[i_metric]:
                per_launch.setdefault(r[i_id], {})[short] = float(r[i_val].replace(",", ""))
    if not per_launch:
        raise SystemExit("no integrate_kernel<%s> launch in %s" % (demangled, csv_path))
    best = max(per_launch.values(), key=lambda d: sum(d.values()))
    rec = {k: round(v / points, 2) for k, v in best.items() if v > 0}
    rec.update(kernel=KERNELS[key], sass_sha256=sass_sha256(key), points_per_launch=points, source=os.path.basename(csv_path))
    if note:
        rec["note"] = note
    data = load()
    for keep in ("dram_bytes", "dram_bytes_source"):          # full-size traffic figures survive a count refresh
        if keep in data.get(key, {}):
            rec[keep] = data[key][keep]
    data[key] = rec
    with open(PATH, "w") as f:
        json.dump(data, f, indent=1, sort_keys=True)
        f.write("\n")
    return rec


if __name__ == "__main__":
    import argparse
    ap = argparse.ArgumentParser()
    ap.add_argument("--update", help="ncu --csv metric log")
    ap.add_argument("--key", help="config,assignments,precision")
    ap.add_argument("--points", type=int, help="sample points of the measured launch")
    ap.add_argument("--note", default="")
    ap.add_argument("--check", action="store_true", help="print every stored key with its build match")
    a = ap.parse_args()
    if a.update:
        print(json.dumps(update(a.update, a.key, a.points, a.note)))
    if a.check:
        for k in sorted(load()):
            f = k.split(",")
            print(k, lookup(int(f[0]), int(f[1]), int(f[2]), variant=f[3] if len(f) > 3 else ""))
    sys.exit(0)
