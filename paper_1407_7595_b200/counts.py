"""Executed FP64 instruction counts per integrand call, tied to the kernel build they were measured on.

`fp64_counts.json` (beside this file) holds, per integrate kernel, the thread-level DFMA / DMUL / DADD (or FFMA /
FMUL / FADD) instructions per sample point from an ncu metric pass, together with the SHA-256 of that kernel's SASS
(`cuobjdump -sass -fun <kernel>` of the in-tree library).  bench.py reads the counts for its "executed" roofline
figures and recomputes the hash of the kernel it is about to time: a count taken on another build is reported as
stale instead of being silently reused (measurement item 8).

How a record is made (after a kernel change, on the GPU box): one ncu metric pass over a short bench.py run,

    ncu --metrics smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,\
smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,smsp__sass_thread_inst_executed_op_ffma_pred_on.sum,\
smsp__sass_thread_inst_executed_op_fmul_pred_on.sum,smsp__sass_thread_inst_executed_op_fadd_pred_on.sum \
        --clock-control none -k regex:integrate_kernel --csv --log-file gpurun_out/counts_c3.csv \
        python bench.py --config 3 --events 37 --steps 1 --warmup 3 --no-cpu-baseline

then, for the launch of KERNELS[key] with the most FP instructions, each metric divided by the sample points of that
launch (events x points), rounded to 0.01, stored with sass_sha256(key) of the library that ran
(profiles/r03_fp64_counts.md lists the runs of this round).  This module only reads the file.

No arithmetic of the method lives here.
"""
from __future__ import annotations

import hashlib
import json
import os
import re
import subprocess

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
