"""Thin ctypes binding of the C ABI in include/mem.h -- argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libmem_b200.so; PyTorch is used only
for device memory and streams.  There is no CPU fallback: if the library cannot be built or
loaded, or no CUDA device is present, the calls raise.  This package never imports oracle/.

Functions carry the names of the C entry points (mem_create, mem_integrate, ...); the small
`Integrator` class at the end only owns a handle.
"""
from __future__ import annotations

import ctypes as C

from . import build as _build
from . import workloads  # noqa: F401  (seeded input generators; no arithmetic of the method)

MEM_OK, MEM_ERR_INVALID_ARG, MEM_ERR_UNSUPPORTED, MEM_ERR_CUDA, MEM_ERR_NOMEM = 0, 1, 2, 3, 4
MEM_PROC_W_ENU, MEM_PROC_Z_BB, MEM_PROC_TT_LJETS, MEM_PROC_TT_DILEP, MEM_PROC_TTH_DILEP = 1, 2, 3, 4, 5

EXPORTS = ("mem_params_default", "mem_event_fields", "mem_n_dims", "mem_create", "mem_destroy",
           "mem_set_event_offset", "mem_integrate", "mem_integrate_noalloc", "mem_integrate_host", "mem_eval_points",
           "mem_eval_parton", "mem_set_pdf_grid", "mem_get_grid", "mem_launch_count", "mem_last_error", "mem_last_pass_ms", "mem_measure_fp64_peak",
           "mem_measure_fp64_peak_rrr", "mem_measure_fp64_rate", "mem_normalisation", "mem_discriminant")


class mem_params(C.Structure):
    """Mirror of `struct mem_params` (include/mem.h)."""
    _fields_ = ([("struct_size", C.c_uint32), ("precision", C.c_uint32)] +
                [(n, C.c_double) for n in (
                    "sqrt_s", "G_F", "m_W", "Gam_W", "m_Z", "Gam_Z", "sin2_thw", "m_t", "Gam_t", "alpha_s",
                    "V_ud", "V_tb", "pdf_A_q", "pdf_A_g", "pdf_pow_x", "pdf_pow_1mx",
                    "tf_w_tail", "tf_mu1", "tf_sig1", "tf_mu2", "tf_sig2", "jetE_rlo", "jetE_rhi",
                    "bw_nwidths", "nu_pz_max", "nu_eta_max", "met_sigma", "met_nsigma", "vegas_alpha")] +
                [("vegas_points", C.c_int64), ("vegas_iters", C.c_int32), ("vegas_bins", C.c_int32),
                 ("n_flav", C.c_int32), ("n_perm", C.c_int32),
                 ("m_H", C.c_double), ("Gam_H", C.c_double), ("yuk_t", C.c_double), ("yuk_b", C.c_double),
                 ("tth_hyp", C.c_int32), ("reserved0", C.c_int32)])


class MemError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("mem status %d: %s" % (status, message))
        self.status = status


_lib = None


def library_path() -> str:
    return _build.LIB


def lib():
    """Load (building first if the sources are newer) libmem_b200.so; raises if that fails."""
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        vp, dp, i64, u64 = C.c_void_p, C.c_void_p, C.c_int64, C.c_uint64
        L.mem_params_default.argtypes = [C.c_int, C.POINTER(mem_params)]
        L.mem_event_fields.argtypes = [C.c_int]
        L.mem_event_fields.restype = C.c_int32
        L.mem_n_dims.argtypes = [C.c_int]
        L.mem_n_dims.restype = C.c_int32
        L.mem_create.argtypes = [C.c_int, C.POINTER(mem_params), C.POINTER(vp)]
        L.mem_destroy.argtypes = [vp]
        L.mem_set_event_offset.argtypes = [vp, u64]
        L.mem_integrate.argtypes = [vp, dp, i64, i64, u64, dp, dp, vp]
        L.mem_integrate_host.argtypes = [vp, dp, i64, i64, u64, dp, dp, vp]
        L.mem_integrate_noalloc.argtypes = [vp, dp, i64, i64, u64, dp, dp, vp]
        L.mem_eval_points.argtypes = [vp, dp, i64, i64, i64, i64, u64, C.c_int32, dp, dp, vp]
        L.mem_eval_parton.argtypes = [vp, dp, i64, dp, vp]
        L.mem_set_pdf_grid.argtypes = [vp, dp, C.c_int32, C.c_int32] + [C.c_double] * 5
        L.mem_get_grid.argtypes = [vp, i64, dp, vp]
        L.mem_launch_count.argtypes = [vp]
        L.mem_launch_count.restype = i64
        L.mem_last_pass_ms.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.mem_measure_fp64_peak.argtypes = [C.c_int32, C.POINTER(C.c_double), vp]
        L.mem_measure_fp64_peak_rrr.argtypes = [C.c_int32, C.POINTER(C.c_double), vp]
        L.mem_measure_fp64_rate.argtypes = [C.c_int32, C.c_int32, C.POINTER(C.c_double), vp]
        L.mem_normalisation.argtypes = [dp, dp, i64, dp, vp]
        L.mem_discriminant.argtypes = [dp, dp, i64, dp, dp, dp, vp]
        L.mem_last_error.argtypes = []
        L.mem_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def mem_last_error() -> str:
    return lib().mem_last_error().decode("utf-8", "replace")


def _check(status):
    if status != MEM_OK:
        raise MemError(status, mem_last_error())


def mem_params_default(process: int) -> mem_params:
    p = mem_params()
    _check(lib().mem_params_default(int(process), C.byref(p)))
    return p


def mem_event_fields(process: int) -> int:
    return lib().mem_event_fields(int(process))


def mem_n_dims(process: int) -> int:
    return lib().mem_n_dims(int(process))


class Handle(C.c_void_p):
    """The opaque mem_handle* plus what the binding needs to validate arguments: the process and the device
    the handle was created on (the C ABI cannot see tensor shapes or devices)."""
    process = 0
    device = -1
    bins = 50


def mem_create(process: int, params: mem_params | None = None) -> Handle:
    h = Handle()
    _check(lib().mem_create(int(process), None if params is None else C.byref(params), C.byref(h)))
    import torch
    h.process, h.device = int(process), torch.cuda.current_device()
    h.bins = int(params.vegas_bins) if params is not None else 50
    return h


def _check_tensor(handle, t, name, rows=None):
    """shape[0] == rows and the tensor lives on the handle's device (a transposed record array or a record of
    another process would make the kernels read beyond the allocation)"""
    if rows is not None and (t.dim() != 2 or int(t.shape[0]) != rows):
        raise ValueError("%s must have shape [%d, n_events], got %s" % (name, rows, tuple(t.shape)))
    dev = getattr(handle, "device", -1)
    if dev >= 0 and t.is_cuda and t.device.index != dev:
        raise ValueError("%s is on cuda:%d, the handle was created on cuda:%d" % (name, t.device.index, dev))


def mem_destroy(handle) -> None:
    _check(lib().mem_destroy(handle))


def mem_set_event_offset(handle, first_event: int) -> None:
    _check(lib().mem_set_event_offset(handle, int(first_event)))


def mem_launch_count(handle) -> int:
    return int(lib().mem_launch_count(handle))


def mem_last_pass_ms(handle):
    """(milliseconds, integrand evaluations) of the dominant kernel of the last mem_integrate."""
    ms, ev = C.c_double(), C.c_int64()
    _check(lib().mem_last_pass_ms(handle, C.byref(ms), C.byref(ev)))
    return ms.value, ev.value


def mem_measure_fp64_peak(repeats: int = 5, stream=None) -> float:
    """Measured FP64 FMA peak of the current device in TFLOP/s."""
    t = C.c_double()
    _check(lib().mem_measure_fp64_peak(int(repeats), C.byref(t), _stream_ptr(stream)))
    return t.value


def mem_measure_fp64_peak_rrr(repeats: int = 5, stream=None) -> float:
    """The same with three register operands per DFMA (what generic fused multiply-adds sustain), TFLOP/s."""
    t = C.c_double()
    _check(lib().mem_measure_fp64_peak_rrr(int(repeats), C.byref(t), _stream_ptr(stream)))
    return t.value


def mem_measure_fp64_rate(kind: int, repeats: int = 5, stream=None) -> float:
    """FP64 issue microbenchmarks (include/mem_bench.h): 2 x FP64 instructions/s/1e12 for instruction mix `kind`."""
    t = C.c_double()
    _check(lib().mem_measure_fp64_rate(int(kind), int(repeats), C.byref(t), _stream_ptr(stream)))
    return t.value


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dev_f64(t, name, shape=None):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError("%s must be a contiguous float64 CUDA tensor" % name)
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError("%s has shape %s, expected %s" % (name, tuple(t.shape), tuple(shape)))
    return C.c_void_p(t.data_ptr())


def mem_integrate(handle, events, n_points: int, seed: int, out_p=None, out_err=None, stream=None):
    """events: float64 CUDA tensor [n_fields, n_events] (SoA).  Returns (out_p, out_err), CUDA tensors
    [n_events]; asynchronous on `stream` (default: torch's current stream)."""
    import torch
    if events.dim() != 2:
        raise ValueError("events must be [n_fields, n_events]")
    _check_tensor(handle, events, "events", mem_event_fields(handle.process) if getattr(handle, "process", 0) else None)
    n_events = int(events.shape[1])
    if out_p is None:
        out_p = torch.empty(n_events, dtype=torch.float64, device=events.device)
    if out_err is None:
        out_err = torch.empty(n_events, dtype=torch.float64, device=events.device)
    _check_tensor(handle, out_p, "out_p")
    _check_tensor(handle, out_err, "out_err")
    _check(lib().mem_integrate(handle, _dev_f64(events, "events"), n_events, int(n_points), int(seed),
                               _dev_f64(out_p, "out_p", (n_events,)), _dev_f64(out_err, "out_err", (n_events,)),
                               _stream_ptr(stream)))
    return out_p, out_err


MEM_NOALLOC_SCRATCH_BYTES = 8 << 20


def mem_integrate_noalloc(handle, events, n_points: int, seed: int, out_p, out_err, stream=None):
    """mem_integrate for hosts that must not allocate device memory (a real-time loop with a fixed memory plan, an
    application whose own pool owns the GPU): plain Monte Carlo only, intermediate arrays in the library's fixed
    MEM_NOALLOC_SCRATCH_BYTES array, same bits as mem_integrate.  The caller brings `out_p` and `out_err`
    (float64 CUDA tensors [n_events]) -- nothing is allocated here either.  A call that needs more scratch than the
    array has raises MemError (MEM_ERR_INVALID_ARG).  All calls on a device share the array: do not let two of
    them overlap on the GPU.  See include/mem.h for the size formula and the first-call rule."""
    if events.dim() != 2:
        raise ValueError("events must be [n_fields, n_events]")
    _check_tensor(handle, events, "events", mem_event_fields(handle.process) if getattr(handle, "process", 0) else None)
    n_events = int(events.shape[1])
    _check_tensor(handle, out_p, "out_p")
    _check_tensor(handle, out_err, "out_err")
    _check(lib().mem_integrate_noalloc(handle, _dev_f64(events, "events"), n_events, int(n_points), int(seed),
                                       _dev_f64(out_p, "out_p", (n_events,)), _dev_f64(out_err, "out_err", (n_events,)),
                                       _stream_ptr(stream)))
    return out_p, out_err


def mem_integrate_host(handle, events, n_points: int, seed: int, out_p=None, out_err=None, stream=None):
    """events: float64 CPU tensor or numpy array [n_fields, n_events].  Copies in, integrates, copies the
    results back into float64 CPU tensors, all on `stream` (default: torch's current stream), and synchronises it."""
    import torch
    ev = torch.as_tensor(events)
    if not (ev.dtype == torch.float64 and ev.is_contiguous() and not ev.is_cuda and ev.dim() == 2):
        raise TypeError("events must be a contiguous float64 host array [n_fields, n_events]")
    _check_tensor(handle, ev, "events", mem_event_fields(handle.process) if getattr(handle, "process", 0) else None)
    n_events = int(ev.shape[1])
    if out_p is None:
        out_p = torch.empty(n_events, dtype=torch.float64)
    if out_err is None:
        out_err = torch.empty(n_events, dtype=torch.float64)
    _check(lib().mem_integrate_host(handle, C.c_void_p(ev.data_ptr()), n_events, int(n_points), int(seed),
                                    C.c_void_p(out_p.data_ptr()), C.c_void_p(out_err.data_ptr()), _stream_ptr(stream)))
    return out_p, out_err


def mem_eval_points(handle, events, event: int, first_point: int, n: int, seed: int, iteration: int = 0,
                    grid=None, out_w=None, stream=None):
    """Diagnostic: weights of points [first_point, first_point + n) of one event (CUDA tensor [n])."""
    import torch
    _check_tensor(handle, events, "events", mem_event_fields(handle.process) if getattr(handle, "process", 0) else None)
    n_events = int(events.shape[1])
    if out_w is None:
        out_w = torch.empty(int(n), dtype=torch.float64, device=events.device)
    if grid is not None:
        _check_tensor(handle, grid, "grid")
        if grid.dim() != 2 or int(grid.shape[0]) != mem_n_dims(handle.process) or int(grid.shape[1]) != handle.bins + 1:
            raise ValueError("grid must have shape [D, vegas_bins + 1] = [%d, %d], got %s"
                             % (mem_n_dims(handle.process), handle.bins + 1, tuple(grid.shape)))
    g = None if grid is None else _dev_f64(grid, "grid")
    _check(lib().mem_eval_points(handle, _dev_f64(events, "events"), n_events, int(event), int(first_point), int(n),
                                 int(seed), int(iteration), g, _dev_f64(out_w, "out_w", (int(n),)),
                                 _stream_ptr(stream)))
    return out_w


def mem_set_pdf_grid(handle, table, lxmin, lxmax, lqmin, lqmax, Q):
    """NEXT-3: table = float64 host array [6, NQ, NX] (None: back to the toy PDF)."""
    import numpy as np
    if table is None:
        _check(lib().mem_set_pdf_grid(handle, None, 0, 0, 0.0, 0.0, 0.0, 0.0, 0.0))
        return
    t = np.ascontiguousarray(table, dtype=np.float64)
    if t.ndim != 3 or t.shape[0] != 6:
        raise ValueError("table must have shape [6, NQ, NX]")
    _check(lib().mem_set_pdf_grid(handle, C.c_void_p(t.ctypes.data), t.shape[2], t.shape[1], float(lxmin), float(lxmax),
                                  float(lqmin), float(lqmax), float(Q)))


def mem_eval_parton(handle, momenta, out_w=None, stream=None):
    """Parton-level mode (NEXT-2): momenta = CUDA float64 tensor [24, n_events]; returns out_w [n_events]."""
    import torch
    _check_tensor(handle, momenta, "momenta", 24)
    n_events = int(momenta.shape[1])
    if out_w is None:
        out_w = torch.empty(n_events, dtype=torch.float64, device=momenta.device)
    _check(lib().mem_eval_parton(handle, _dev_f64(momenta, "momenta"), n_events,
                                 _dev_f64(out_w, "out_w", (n_events,)), _stream_ptr(stream)))
    return out_w


def mem_normalisation(p, g, out_sigma=None, stream=None):
    """sigma = mean(p / g) over events drawn from the density g (reading A22): CUDA tensor [1]."""
    import torch
    n = int(p.shape[0])
    if out_sigma is None:
        out_sigma = torch.empty(1, dtype=torch.float64, device=p.device)
    _check(lib().mem_normalisation(_dev_f64(p, "p", (n,)), _dev_f64(g, "g", (n,)), n, _dev_f64(out_sigma, "out_sigma", (1,)),
                                   _stream_ptr(stream)))
    return out_sigma


def mem_discriminant(p_sig, p_bkg, sigma_sig, sigma_bkg, out_D=None, stream=None):
    """D = log10((p_sig / sigma_sig) / (p_bkg / sigma_bkg)) per event (Eq. 10): CUDA tensor [n]."""
    import torch
    n = int(p_sig.shape[0])
    if out_D is None:
        out_D = torch.empty(n, dtype=torch.float64, device=p_sig.device)
    _check(lib().mem_discriminant(_dev_f64(p_sig, "p_sig", (n,)), _dev_f64(p_bkg, "p_bkg", (n,)), n,
                                  _dev_f64(sigma_sig, "sigma_sig", (1,)), _dev_f64(sigma_bkg, "sigma_bkg", (1,)),
                                  _dev_f64(out_D, "out_D", (n,)), _stream_ptr(stream)))
    return out_D


def mem_get_grid(handle, n_events: int, n_dims: int, bins: int, device=None, stream=None):
    """Diagnostic: VEGAS grids of the last mem_integrate, CUDA tensor [n_events, D, bins + 1]."""
    import torch
    out = torch.empty((int(n_events), int(n_dims), int(bins) + 1), dtype=torch.float64,
                      device=device or torch.device("cuda"))
    _check(lib().mem_get_grid(handle, int(n_events), _dev_f64(out, "out_grid"), _stream_ptr(stream)))
    return out


class Integrator:
    """Owns one handle: `with Integrator(MEM_PROC_TT_LJETS) as it: p, err = it.integrate(ev, N, seed)`."""

    def __init__(self, process: int, params: mem_params | None = None, **overrides):
        self.process = int(process)
        self.params = params if params is not None else mem_params_default(process)
        for k, v in overrides.items():
            if not hasattr(self.params, k):
                raise AttributeError("mem_params has no field %r" % k)
            setattr(self.params, k, v)
        self.handle = mem_create(process, self.params)

    def integrate(self, events, n_points, seed, **kw):
        return mem_integrate(self.handle, events, n_points, seed, **kw)

    def integrate_noalloc(self, events, n_points, seed, out_p, out_err, **kw):
        return mem_integrate_noalloc(self.handle, events, n_points, seed, out_p, out_err, **kw)

    def integrate_host(self, events, n_points, seed, **kw):
        return mem_integrate_host(self.handle, events, n_points, seed, **kw)

    def eval_points(self, events, event, first_point, n, seed, **kw):
        return mem_eval_points(self.handle, events, event, first_point, n, seed, **kw)

    def set_pdf_grid(self, table, lxmin=0.0, lxmax=0.0, lqmin=0.0, lqmax=0.0, Q=0.0):
        mem_set_pdf_grid(self.handle, table, lxmin, lxmax, lqmin, lqmax, Q)

    def eval_parton(self, momenta, **kw):
        return mem_eval_parton(self.handle, momenta, **kw)

    def grid(self, n_events, **kw):
        return mem_get_grid(self.handle, n_events, mem_n_dims(self.process), self.params.vegas_bins, **kw)

    def set_event_offset(self, first_event):
        mem_set_event_offset(self.handle, first_event)

    def last_pass_ms(self):
        return mem_last_pass_ms(self.handle)

    @property
    def launches(self):
        return mem_launch_count(self.handle)

    def close(self):
        if self.handle is not None:
            mem_destroy(self.handle)
            self.handle = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
