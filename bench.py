#!/usr/bin/env python
"""Benchmark of the hot path.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]

One step = one pass of the whole hot path (S0-S8, plus S1v/S9 for config 5) over one batch of
seeded synthetic events: mem_integrate on BASELINE.json's configs[2] by default (4096 t tbar
lepton+jets events x 2^20 points, 6-D, fp64 -- the configuration north_star's target is quoted
on).  Rank 0 prints ONE JSON line.  With N > 1 (torchrun) every rank integrates its own shard of
4096 events of a 4096*N list (weak scaling, no data-path collective); the time is the max over
ranks.

--impl reference times the CPU oracle as it stands on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

SEED = 20140729

# FP64 work per integrand call of the dominant kernel, two counts:
#  - executed: thread-level DFMA / DMUL / DADD per point from an ncu metric pass, read from
#    paper_1407_7595_b200/fp64_counts.json together with the SASS hash of the kernel they were taken on
#    (counts.py); a count that belongs to another build is reported as stale, never silently reused;
#  - algorithmic: a fixed reference, flop = 2 FMA + MUL + ADD of the formulas as first implemented (the round-1
#    kernels' executed counts, profiles/r01_fp64_counts.md, with every exponential at the cost of the table-driven
#    implementation), NOT updated when later kernels remove instructions; reported as frac_fixed_reference.
#    roofline.frac uses the executed count; the fixed one only where no executed count exists.
#    Key = (config, jet-parton assignments per point).
ALGORITHMIC_FLOP = {
    (1, 1): 240.0,       # 87.3 DFMA, 47.0 DMUL, 18.4 DADD
    (2, 1): 224.6,       # 86.0, 37.0, 15.6
    (3, 1): 451.2,       # 196.0, 90.0, 41.2 with libdevice exp = 523.2; six exponentials at table cost: -72
    (3, 24): 4007.2,     # 1597, 1335, 551.2 = 4079.2; -72 as above
    (4, 1): 622.8,       # 241.0, 82.9, 57.9
    (4, 2): 854.2,       # 327.2, 120.2, 79.8
    (5, 1): 502.8,       # 166.0, 115.1, 55.7 (grid-mapped final pass)
}
# NEXT-4 (config 6), per hypothesis: executed count of the first parity-green kernel of round 2 (profiles/r02_fp64_counts.md)
TTH_ALGORITHMIC_FLOP = {0: 536.3, 1: 462.2}   # 209.5 / 68.0 / 49.4 and 181.2 / 56.6 / 43.2 (DFMA / DMUL / DADD)
NOMINAL_FP64_FMA_PER_CLK_PER_SM = 64      # 4 SMSPs x 16 lanes; confirmed by the microbenchmark
VEGAS_ITERS, VEGAS_POINTS = 5, 1 << 17    # BASELINE.json:configs[4]


def executed_counts(cfg, perm=1, precision=64, variant=""):
    """(record or None) from fp64_counts.json, with "match" = taken on the SASS that is built now"""
    from paper_1407_7595_b200 import counts
    return counts.lookup(cfg, perm, precision, variant=variant)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5, 6],
                    help="1-5: BASELINE.json configs; 6: NEXT-4, t tbar H(-> b bbar) dilepton with four b jets")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--events", type=int, default=0, help="override the event count (default: the config's)")
    ap.add_argument("--points", type=int, default=0, help="override points/event (default: the config's)")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32],
                    help="32 = fp32 integrand core of config 3 (reading A15)")
    ap.add_argument("--perm", type=int, default=0,
                    help="jet-parton assignments summed per point (NEXT-1): config 3/5: 4 or 24, config 4: 2")
    ap.add_argument("--pdf", default="toy", choices=["toy", "grid"],
                    help="grid = NEXT-3: bilinear (ln x, ln Q) tables synthesised from the toy PDF (configs 3-5)")
    ap.add_argument("--hyp", type=int, default=0, choices=[0, 1],
                    help="config 6: hypothesis of PAPER.md Eq. 10 (0 = t tbar H, 1 = non-resonant t tbar b bbar)")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="process-group backend for N > 1 (gloo: several ranks sharing one GPU, for tests)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--parton", action="store_true",
                    help="NEXT-2 parton-level mode: ME evaluations of --events configurations (default 10^5)")
    ap.add_argument("--microbench", action="store_true",
                    help="FP64 issue microbenchmarks behind the roofline discussion (mem_measure_fp64_rate)")
    ap.add_argument("--sweep", action="store_true",
                    help="config-5 sweep of BASELINE.json:configs[4]: events x final points, one JSON line")
    return ap.parse_args()


def workload(cfg, args):
    from paper_1407_7595_b200 import workloads as wl
    proc, ne, npts = wl.CONFIGS[3 if cfg == 5 else cfg]
    if args.events:
        ne = args.events
    if args.points:
        npts = args.points
    name = {1: "config1 W->e nu 1-D", 2: "config2 Z->bb 2-D", 3: "config3 ttbar l+jets 6-D",
            4: "config4 ttbar dilepton 8-D",
            5: "config5 ttbar l+jets 6-D + VEGAS 5x2^17",
            6: "NEXT-4 ttH(->bb) dilepton 8-D (Eq. 7-9, 11), hypothesis %d, closure records" % args.hyp}[cfg]
    return proc, ne, npts, "%s, %d events x %d points/event, %s%s" % (
        name, ne, npts, "fp32 core (A15)" if args.precision == 32 else "fp64",
        (", %d jet-parton assignments per point" % args.perm if args.perm > 1 else "") +
        (", grid PDFs" if args.pdf == "grid" else ""))


def make_records(cfg, proc, n):
    """config 6 is measured on physical t tbar H records (they stand in for the paper's MadGraph + Pythia sample,
    PAPER.md:145); the BASELINE configs on their i.i.d. records"""
    from paper_1407_7595_b200 import workloads as wl
    return wl.make_tth_events(n) if cfg == 6 else wl.make_events(proc, n)


# --------------------------------------------------------------------------------------------
# clocks during the timed region
# --------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        """index: what nvidia-smi -i accepts -- a physical index or a GPU UUID (robust under CUDA_VISIBLE_DEVICES)"""
        self.proc = None
        self.index = index
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def _one_shot(self):
        try:
            return subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                   "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=10).stdout
        except (OSError, subprocess.SubprocessError):
            return ""

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        if not out.strip():          # timed region shorter than one sampling period: query once, right after it
            out = self._one_shot()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------------------------
# CPU oracle legs
# --------------------------------------------------------------------------------------------
def _oracle_worker(job):
    cfg, proc, ev, lo, n_points, seed, hyp = job
    import oracle
    p = oracle.params_default(proc)
    p.tth_hyp = hyp
    t0 = time.perf_counter()
    if cfg == 5:
        p.vegas_iters, p.vegas_points = VEGAS_ITERS, VEGAS_POINTS
        oracle.vegas_integrate(proc, p, ev, n_points, seed, event_offset=lo)
        evals = ev.shape[1] * (n_points + VEGAS_ITERS * VEGAS_POINTS)
    else:
        oracle.integrate(proc, p, ev, n_points, seed, event_offset=lo)
        evals = ev.shape[1] * n_points
    return evals, time.perf_counter() - t0


def oracle_sample(cfg, proc, ev, n_points, events_per_core, pool, cores, hyp=0):
    """The oracle, single-threaded by design, run as `cores` independent processes over disjoint
    event ranges.  Returns (evaluations, wall seconds, events)."""
    jobs = []
    for k in range(cores):
        lo = k * events_per_core
        jobs.append((cfg, proc, ev[:, lo:lo + events_per_core].copy(), lo, n_points, SEED, hyp))
    t0 = time.perf_counter()
    res = pool.map(_oracle_worker, jobs)
    wall = time.perf_counter() - t0
    return sum(r[0] for r in res), wall, cores * events_per_core


def run_reference(args):
    import multiprocessing as mp
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1407_7595_b200 import workloads as wl
    import oracle
    oracle.build()
    cfg = args.config
    proc, ne, n_points, name = workload(cfg, args)
    cores = min(os.cpu_count() or 1, 64)
    per_core = 1 if n_points >= (1 << 20) else max(1, (1 << 20) // n_points)
    per_core = min(per_core, max(1, ne // cores))
    ev = make_records(cfg, proc, ne)
    with mp.get_context("spawn").Pool(cores) as pool:
        for _ in range(args.warmup):
            oracle_sample(cfg, proc, ev, n_points, per_core, pool, cores, args.hyp)
        evals = wall = events = 0
        for _ in range(args.steps):
            a, b, c = oracle_sample(cfg, proc, ev, n_points, per_core, pool, cores, args.hyp)
            evals += a; wall += b; events += c
    value = evals / wall
    sample = "%d events (%d per core) x %d points/event per step" % (cores * per_core, per_core, n_points)
    line = {
        "impl": "reference", "metric": "integrand_evals_per_s", "value": value, "unit": "evals/s",
        "events_per_s": events / wall, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * wall / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": name, "sample": sample},
        "cpu_baseline": {"value": value, "unit": "evals/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "evals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
# the CUDA path
# --------------------------------------------------------------------------------------------
def run_b200(args):
    import torch

    import paper_1407_7595_b200 as mem
    from paper_1407_7595_b200 import sharding
    from paper_1407_7595_b200 import workloads as wl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    rank, local_rank, world = sharding.dist_env()
    local_rank %= torch.cuda.device_count()         # several ranks may share a GPU in a plumbing test (--dist-backend gloo)
    torch.cuda.set_device(local_rank)
    if world > 1:
        sharding.init_process_group(args.dist_backend)
    red_dev = "cuda" if args.dist_backend == "nccl" else "cpu"
    import torch.distributed as dist

    cfg = args.config
    proc, ne, n_points, name = workload(cfg, args)
    # weak scaling: every rank owns `ne` events of a list of ne * world (contiguous shard)
    ev_all = make_records(cfg, proc, ne * world)
    lo = rank * ne
    ev_host = torch.from_numpy(ev_all[:, lo:lo + ne].copy()).pin_memory()
    ev_dev = ev_host.cuda()
    over = dict(vegas_iters=VEGAS_ITERS, vegas_points=VEGAS_POINTS) if cfg == 5 else {}
    if args.precision == 32:
        over["precision"] = 32
    if args.perm > 1:
        over["n_perm"] = args.perm
    if cfg == 6:
        over["tth_hyp"] = args.hyp
    it = mem.Integrator(proc, **over)
    if args.pdf == "grid":
        g = wl.PDF_GRID
        it.set_pdf_grid(wl.make_pdf_table(), g["lxmin"], g["lxmax"], g["lqmin"], g["lqmax"], 173.0)
    it.set_event_offset(lo)
    out_p = torch.empty(ne, dtype=torch.float64, device="cuda")
    out_err = torch.empty_like(out_p)
    hp = torch.empty(ne, dtype=torch.float64).pin_memory()
    he = torch.empty(ne, dtype=torch.float64).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")       # > 126 MB L2
    evals_per_step = ne * (n_points + (VEGAS_ITERS * VEGAS_POINTS if cfg == 5 else 0))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps, collect_kernel=False):
        """time exactly `steps` steps: per-step CUDA events on torch's current stream (the stream
        the library launches on), L2 flushed between steps outside the event pairs"""
        ms, kms = [], []
        for _ in range(steps):
            flush.fill_(0)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn()
            b.record()
            b.synchronize()
            ms.append(a.elapsed_time(b))
            if collect_kernel:
                kms.append(it.last_pass_ms()[0])
        return ms, kms

    def step_dev():
        it.integrate(ev_dev, n_points, SEED, out_p=out_p, out_err=out_err)

    def step_host():
        it.integrate_host(ev_host, n_points, SEED, out_p=hp, out_err=he)

    for _ in range(max(args.warmup, 3)):
        step_dev()
    step_host()
    barrier()
    # nvidia-smi wants the physical device: address it by UUID, which survives CUDA_VISIBLE_DEVICES remapping
    uuid = getattr(torch.cuda.get_device_properties(local_rank), "uuid", None)
    sampler = ClockSampler("GPU-%s" % uuid if uuid is not None else local_rank) if rank == 0 else None
    launches0 = it.launches
    barrier()
    ms, kms = timed(step_dev, args.steps, collect_kernel=True)
    barrier()
    launches = it.launches - launches0
    clocks = sampler.stop() if sampler else None
    t_dev = sharding.max_over_ranks(sum(ms) / 1e3, device=red_dev)
    barrier()
    ms_h, _ = timed(step_host, args.steps)
    barrier()
    t_host = sharding.max_over_ranks(sum(ms_h) / 1e3, device=red_dev)

    # outside the timed region: the global event index reached the Philox counter on every rank -- the first event of
    # this rank's shard, integrated alone with event_offset = lo, reproduces out_p[0] bit for bit; and the optional
    # all-gather of the 16 B/event results works (first 8 events of every shard)
    one_p = torch.empty(1, dtype=torch.float64, device="cuda")
    one_e = torch.empty_like(one_p)
    it.integrate(ev_dev[:, :1].contiguous(), n_points, SEED, out_p=one_p, out_err=one_e)
    torch.cuda.synchronize()
    shard_ok = bool(torch.equal(one_p, out_p[:1]) and torch.equal(one_e, out_err[:1]))
    n_head = min(8, ne)
    head = out_p[:n_head].clone() if args.dist_backend == "nccl" else out_p[:n_head].cpu()
    gathered = sharding.gather_results(head, n_head * world)
    shard_ok_all = sharding.sum_over_ranks(1.0 if shard_ok else 0.0, device=red_dev) == float(world)

    if rank != 0:
        it.close()
        return

    total_evals = evals_per_step * world * args.steps
    value = total_evals / t_dev
    # roofline of the dominant kernel (the integrate pass that produces the outputs)
    k_ms = sum(kms) / len(kms)
    k_evals = ne * n_points
    peak_meas = mem.mem_measure_fp64_peak(5)
    peak_rrr = mem.mem_measure_fp64_peak_rrr(5)
    perm = max(args.perm, 1)
    ex = executed_counts(cfg, perm, 64, "h1" if (cfg == 6 and args.hyp == 1) else "") if args.pdf == "toy" else None
    fl_ex = None if ex is None else 2.0 * ex.get("dfma", 0.0) + ex.get("dmul", 0.0) + ex.get("dadd", 0.0)
    pipe_inst = None if ex is None else ex.get("dfma", 0.0) + ex.get("dmul", 0.0) + ex.get("dadd", 0.0)
    fl_alg = ALGORITHMIC_FLOP.get((cfg, perm))
    if fl_alg is None and cfg == 6 and perm == 1:
        fl_alg = TTH_ALGORITHMIC_FLOP.get(args.hyp)
    rate = k_evals / (k_ms * 1e-3) / 1e12                  # 1e12 evaluations/s of the dominant kernel
    sms = torch.cuda.get_device_properties(local_rank).multi_processor_count
    sm_mhz = (clocks or {}).get("sm_mhz") or 0.0
    # Headline: the FP64 flops the timed kernel executes (thread-level DFMA x 2 + DMUL + DADD per call from
    # fp64_counts.json, tied to this build by its SASS hash), so that achieved / frac can be reproduced from profiles/.
    # The fixed round-1 count stays beside it as "useful work per call as first implemented"; it is the fallback only
    # for variants without an executed count (grid PDFs), and the line says which basis it used.
    stale = ex is not None and ex.get("match") is False
    if fl_ex is not None:
        achieved, basis = rate * fl_ex, "executed" + (" (STALE: the counts were taken on another build of this kernel)" if stale else "")
    elif fl_alg is not None:
        achieved, basis = rate * fl_alg, "fixed_reference (no executed count for this variant)"
    else:
        achieved, basis = None, None
    fixed = None if fl_alg is None else rate * fl_alg
    roofline = {
        "bound": "alu", "kernel": "integrate_kernel<%s>" % ("ProcTTljets,GRID" if cfg == 5 else "proc%d,PLAIN" % proc),
        "achieved": achieved, "peak": peak_meas, "unit": "TFLOP/s",
        "frac": None if achieved is None else achieved / peak_meas,
        "frac_basis": basis,
        "flop_per_call_executed": fl_ex,
        "achieved_executed": None if fl_ex is None else rate * fl_ex,
        "frac_executed": None if fl_ex is None else rate * fl_ex / peak_meas,
        "flop_per_call_algorithmic": fl_alg,
        "flop_per_call_algorithmic_note": "fixed reference count (bench.py: ALGORITHMIC_FLOP, DESIGN.md section 5), "
                                          "not updated when kernels shed instructions",
        "achieved_fixed_reference": fixed,
        "frac_fixed_reference": None if fixed is None else fixed / peak_meas,
        "executed_counts": None if ex is None else {k: ex[k] for k in ("dfma", "dmul", "dadd") if k in ex},
        "executed_counts_match_build": None if ex is None else ex.get("match"),
        "peak_source": "measured in this run: independent DFMA chains on all SMs (mem_measure_fp64_peak)",
        "peak_three_register_operands": peak_rrr,
        "peak_three_register_operands_note": "same microbenchmark with x = fma(x, y, z), y and z in registers: the "
                                             "register file feeds such DFMAs at ~2/3 of the pipe's nominal rate",
        "peak_nominal_at_observed_clock": 2e-6 * NOMINAL_FP64_FMA_PER_CLK_PER_SM * sms * sm_mhz,
        "fp64_pipe_frac": None if pipe_inst is None else rate * pipe_inst / (peak_meas / 2.0),
        "fp64_inst_per_call": pipe_inst, "kernel_ms": k_ms,
        "kernel_share_of_step": k_ms * len(kms) / sum(ms),
        "traffic": ((ex or {}).get("dram_bytes") or {}).get("%dx%d" % (ne, n_points)),
        "hbm_gbs_event_result_path": (ne * mem.mem_event_fields(proc) * 8 + ne * 16) / (sum(ms) / len(ms) * 1e-3) / 1e9,
    }
    if args.precision == 32:
        # fp32 core: the bound is instruction issue (FP32 + INT share the 4 x 32-lane datapaths), so
        # the roofline is counted in executed FP32 flops against 128 FFMA/clk/SM at the observed clock
        f = executed_counts(cfg, perm, 32) or {}
        fl32 = 2.0 * f.get("ffma", 0.0) + f.get("fmul", 0.0) + f.get("fadd", 0.0)
        peak32 = 2e-6 * 128 * sms * (sm_mhz or 1965.0)
        ach32 = rate * fl32
        roofline.update({"kernel": roofline["kernel"].replace("proc3", "ProcTTljetsF"), "achieved": ach32,
                         "peak": peak32, "frac": ach32 / peak32, "flop_per_call_executed": fl32,
                         "flop_per_call_algorithmic": None, "executed_counts_match_build": f.get("match"),
                         "peak_source": "derived: 128 FP32 FMA/clk/SM x SMs x sampled SM clock (DESIGN.md); executed FP32 flops",
                         "fp64_flop_per_call_kept": fl_ex})
        roofline["frac_basis"] = "executed FP32 flops" + (" (STALE: counts from another build)" if f.get("match") is False else "")
        for k in ("fp64_pipe_frac", "fp64_inst_per_call", "achieved_executed", "frac_executed", "executed_counts",
                  "achieved_fixed_reference", "frac_fixed_reference", "flop_per_call_algorithmic_note"):
            roofline.pop(k, None)
    h2d = ne * mem.mem_event_fields(proc) * 8
    d2h = 2 * ne * 8
    line = {
        "metric": "integrand_evals_per_s", "value": value, "unit": "evals/s",
        "events_per_s": ne * world * args.steps / t_dev,
        "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * t_dev / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32" if args.precision == 32 else "f64", "data": "synthetic",
        "config": {"workload": name, "events_per_gpu": ne, "points_per_event": n_points, "seed": SEED,
                   "l2": "flushed between timed steps (256 MiB fill); inputs are 0.5 MB",
                   "parallelism": "events sharded over %d GPU(s), no collective" % world},
        "clocks": clocks,
        "e2e": {"value": total_evals / t_host, "unit": "evals/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": 1e3 * t_host / args.steps, "entry": "mem_integrate_host (pinned host buffers)"},
        "gpu_launches": launches,
        "roofline": roofline,
        "shard_check": {"first_event_recomputed_with_offset_is_bit_identical_on_every_rank": bool(shard_ok_all),
                        "gathered_first_events_p": [float(x) for x in gathered.cpu().tolist()]},
    }
    it.close()
    if world == 1 and not args.no_cpu_baseline:
        import multiprocessing as mp
        import oracle
        oracle.build()
        cores = min(os.cpu_count() or 1, 64)
        per_core = 8 if n_points >= (1 << 20) else max(1, (8 << 20) // n_points)
        per_core = max(1, min(per_core, ne // cores))
        with mp.get_context("spawn").Pool(cores) as pool:
            evals, wall, events = oracle_sample(cfg, proc, ev_all, n_points, per_core, pool, cores, args.hyp)
        line["cpu_baseline"] = {"value": evals / wall, "unit": "evals/s", "cores": cores, "kind": "oracle",
                                "events_per_s": events / wall, "seconds": wall,
                                "sample": "first %d events (%d per core) x %d points/event of the same workload"
                                          % (events, per_core, n_points)}
    print(json.dumps(line), flush=True)


def run_sweep(args):
    """BASELINE.json:configs[4]: events in {256, 4096, 65536} x N_f in {2^12..2^22}, 5 adaptation passes of
    N_a = max(N_f / 8, 2^9) points (the base cell's ratio), then the final pass.  One GPU, device-resident
    inputs, CUDA events, L2 flushed between steps."""
    import torch

    import paper_1407_7595_b200 as mem
    from paper_1407_7595_b200 import workloads as wl

    torch.cuda.set_device(0)
    proc = wl.TT_LJETS
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    cells = []
    for ne in (256, 4096, 65536):
        ev_dev = torch.from_numpy(wl.make_events(proc, ne)).cuda()
        out_p = torch.empty(ne, dtype=torch.float64, device="cuda")
        out_err = torch.empty_like(out_p)
        for lg in range(12, 23):
            n_f = 1 << lg
            n_a = max(n_f // 8, 1 << 9)
            over = dict(vegas_iters=VEGAS_ITERS, vegas_points=n_a)
            if args.precision == 32:
                over["precision"] = 32
            with mem.Integrator(proc, **over) as it:
                it.integrate(ev_dev, n_f, SEED, out_p=out_p, out_err=out_err)       # warm-up, sizes the workspace
                torch.cuda.synchronize()
                ms = []
                for _ in range(max(1, args.steps if ne * n_f < (1 << 34) else 1)):
                    flush.fill_(0)
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    it.integrate(ev_dev, n_f, SEED, out_p=out_p, out_err=out_err)
                    b.record()
                    b.synchronize()
                    ms.append(a.elapsed_time(b))
            t = min(ms)
            evals = ne * (n_f + VEGAS_ITERS * n_a)
            cells.append({"events": ne, "final_points": n_f, "adapt_points": n_a, "ms": t,
                          "evals_per_s": evals / (t * 1e-3), "events_per_s": ne / (t * 1e-3),
                          "mean_rel_err": float((out_err[out_p > 0] / out_p[out_p > 0]).mean())})
    print(json.dumps({"metric": "integrand_evals_per_s", "unit": "evals/s", "n_gpus": 1, "data": "synthetic",
                      "dtype": "f32" if args.precision == 32 else "f64",
                      "config": {"workload": "config5 sweep: t tbar l+jets 6-D, VEGAS 5 x N_a + N_f, 50 bins/dim"},
                      "sweep": cells}), flush=True)


def run_parton(args):
    """NEXT-2 (Table 2): parton-level weights of N fully specified t tbar -> 6 parton
    configurations, summed over --perm assignments.  One step = one mem_eval_parton call.  The kernel reads
    192 B and writes 8 B per event: at one assignment it is HBM/latency bound, at 24 FP64 bound."""
    import torch

    import paper_1407_7595_b200 as mem
    from paper_1407_7595_b200 import workloads as wl

    torch.cuda.set_device(0)
    n = args.events or 100000
    perm = max(args.perm, 1)
    ev_host = torch.from_numpy(wl.make_parton_events(n)).pin_memory()
    ev = ev_host.cuda()
    out = torch.empty(n, dtype=torch.float64, device="cuda")
    out_host = torch.empty(n, dtype=torch.float64).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    with mem.Integrator(wl.TT_LJETS, **({"n_perm": perm} if perm > 1 else {})) as it:
        def dev_step():
            it.eval_parton(ev, out_w=out)

        def host_step():
            d = ev_host.cuda(non_blocking=True)
            it.eval_parton(d, out_w=out)
            out_host.copy_(out, non_blocking=True)
            torch.cuda.synchronize()

        for _ in range(max(args.warmup, 3)):
            dev_step()
        host_step()
        res = {}
        for name, fn in (("dev", dev_step), ("host", host_step)):
            ms = []
            for _ in range(args.steps):
                flush.fill_(0)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                fn()
                b.record()
                b.synchronize()
                ms.append(a.elapsed_time(b))
            res[name] = sum(ms) / len(ms)
    t = res["dev"] * 1e-3
    traffic = n * (24 + 1) * 8
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(
        os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    hbm = peaks.get("hbm_gbs", 6650.0)
    line = {"metric": "parton_level_me_evals_per_s", "value": n * perm / t, "unit": "assignment evaluations/s",
            "events_per_s": n / t, "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": res["dev"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "parton-level t tbar l+jets (NEXT-2), %d events x %d assignments" % (n, perm),
                       "l2": "flushed between timed steps (256 MiB fill)"},
            "e2e": {"value": n * perm / (res["host"] * 1e-3), "unit": "assignment evaluations/s",
                    "h2d_bytes_per_step": n * 24 * 8, "d2h_bytes_per_step": n * 8, "ms_per_step": res["host"]},
            "gpu_launches": args.steps,
            "roofline": {"bound": "hbm", "kernel": "parton_ttljets_kernel", "achieved": traffic / t / 1e9, "peak": hbm,
                         "unit": "GB/s", "frac": traffic / t / 1e9 / hbm, "traffic": None,
                         "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650 GB/s",
                         "note": "200 B/event algorithmic; with 24 assignments the kernel is FP64 bound instead"}}
    print(json.dumps(line), flush=True)


def run_microbench(args):
    import torch

    import paper_1407_7595_b200 as mem
    torch.cuda.set_device(0)
    names = ["DFMA, two uniform operands (nominal peak)", "DFMA, three register operands",
             "5 DFMA : 2 DMUL : 1 DADD, shuffled register operands", "8 DFMA (uniform) + 8 integer instructions",
             "8 DFMA (uniform) + 16 integer instructions", "DMUL, two register operands", "DADD, two register operands"]
    res = [{"kind": k, "what": n, "tera_fp64_inst_per_s": mem.mem_measure_fp64_rate(k, 5) / 2.0} for k, n in enumerate(names)]
    for r in res:
        r["frac_of_kind0"] = r["tera_fp64_inst_per_s"] / res[0]["tera_fp64_inst_per_s"]
    print(json.dumps({"metric": "fp64_instruction_rate", "unit": "T inst/s", "n_gpus": 1, "microbench": res}), flush=True)


def main():
    args = parse_args()
    if args.microbench:
        run_microbench(args)
    elif args.parton:
        run_parton(args)
    elif args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
