"""ctypes binding of include/epr.h — same names, argument marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

EPR_LOCAL, EPR_NONLOCAL = 0, 1
_STATUS = {0: "EPR_OK", 1: "EPR_EINVAL", 2: "EPR_ESIZE", 3: "EPR_ECUDA", 4: "EPR_ENOMEM"}
_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

EXPORTS = ["epr_default_options", "epr_plan", "epr_forward", "epr_adjoint", "epr_transport", "epr_precondition",
           "epr_retrieve", "epr_retrieve_oversampled", "epr_set_diagnostics", "epr_retrieve_host", "epr_plan_lines", "epr_launch_count", "epr_destroy",
           "epr_last_error", "epr_version", "epr_profile_enable", "epr_profile_read", "epr_read_flags",
           "epr_plan_profiles", "epr_plan_columns", "epr_shift_histogram",
           "epr_retrieve_oversampled_host", "epr_residual_rms_static", "epr_static_last_error",
           "epr_retrieve_host_async", "epr_host_wait", "epr_retrieve_host_multi", "epr_shard_range"]
EPR_STATIC_MAX_BATCH = 1024
EPR_FLAG_SPLAT_OVERFLOW = 1


class EprError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class Options(C.Structure):
    """Mirror of `epr_options` (include/epr.h)."""
    _fields_ = [("order", C.c_int), ("wkb1", C.c_int), ("symbol", C.c_int), ("max_shift_px", C.c_float),
                ("i_min", C.c_float), ("newton_iters", C.c_int), ("init", C.c_int), ("output", C.c_int),
                ("out_bin", C.c_int), ("mu_rel", C.POINTER(C.c_double)), ("nonlocal_wkb1", C.c_int)]


def lib_path():
    return os.path.join(_HERE, "libepr.so")


def load_library():
    """dlopen libepr.so (built by paper_2601_22793_b200.build).  Raises if it is missing — no fallback."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = lib_path()
    if not os.path.exists(path):
        raise EprError(3, f"{path} not built: run `python -m paper_2601_22793_b200.build` (needs nvcc)")
    lib = C.CDLL(path)
    vp, ci, cf, cd = C.c_void_p, C.c_int, C.c_float, C.c_double
    lib.epr_default_options.argtypes = [C.POINTER(Options)]
    lib.epr_default_options.restype = None
    lib.epr_plan.argtypes = [C.POINTER(vp), ci, ci, cd, cd, ci, C.POINTER(cd), C.POINTER(cd), C.POINTER(cd), ci, ci,
                             C.POINTER(Options)]
    lib.epr_forward.argtypes = [vp, ci, vp, vp, vp, vp]
    lib.epr_adjoint.argtypes = [vp, ci, vp, vp, vp]
    lib.epr_transport.argtypes = [vp, ci, vp, vp, vp]
    lib.epr_precondition.argtypes = [vp, ci, vp, vp, vp]
    lib.epr_retrieve.argtypes = [vp, ci, vp, vp, ci, cf, vp]
    lib.epr_retrieve_oversampled.argtypes = [vp, ci, ci, vp, vp, ci, cf, vp]
    lib.epr_set_diagnostics.argtypes = [vp, vp, ci]
    lib.epr_retrieve_host.argtypes = [vp, ci, vp, vp, ci, cf]
    lib.epr_retrieve_host_async.argtypes = [vp, ci, vp, vp, ci, cf]
    lib.epr_retrieve_host_async.restype = ci
    lib.epr_host_wait.argtypes = [vp]
    lib.epr_host_wait.restype = ci
    lib.epr_retrieve_host_multi.argtypes = [C.POINTER(vp), ci, ci, vp, vp, ci, cf]
    lib.epr_retrieve_host_multi.restype = ci
    lib.epr_shard_range.argtypes = [ci, ci, ci, C.POINTER(ci), C.POINTER(ci)]
    lib.epr_shard_range.restype = ci
    lib.epr_retrieve_oversampled_host.argtypes = [vp, ci, ci, vp, vp, ci, cf]
    lib.epr_retrieve_oversampled_host.restype = ci
    lib.epr_plan_lines.argtypes = [vp, C.POINTER(cd), C.POINTER(cd), C.POINTER(cd), C.POINTER(cd)]
    lib.epr_launch_count.argtypes = [vp]
    lib.epr_launch_count.restype = C.c_longlong
    lib.epr_destroy.argtypes = [vp]
    lib.epr_profile_enable.argtypes = [vp, ci]
    lib.epr_profile_enable.restype = ci
    lib.epr_profile_read.argtypes = [vp, ci, C.POINTER(C.c_char_p), C.POINTER(cd), C.POINTER(C.c_longlong), ci]
    lib.epr_profile_read.restype = ci
    lib.epr_plan_profiles.argtypes = [vp, ci, C.POINTER(cd), C.POINTER(cd), C.POINTER(cd)]
    lib.epr_plan_profiles.restype = ci
    lib.epr_plan_columns.argtypes = [vp, C.POINTER(cd), C.POINTER(cd), C.POINTER(cd)]
    lib.epr_plan_columns.restype = ci
    lib.epr_shift_histogram.argtypes = [vp, ci, vp, ci, cf, vp, vp]
    lib.epr_shift_histogram.restype = ci
    lib.epr_read_flags.argtypes = [vp, C.POINTER(C.c_uint), ci]
    lib.epr_read_flags.restype = ci
    lib.epr_residual_rms_static.argtypes = [ci, ci, ci, ci, vp, vp, vp]
    lib.epr_residual_rms_static.restype = ci
    lib.epr_static_last_error.argtypes = []
    lib.epr_static_last_error.restype = C.c_char_p
    lib.epr_last_error.argtypes = [vp]
    lib.epr_last_error.restype = C.c_char_p
    lib.epr_version.restype = C.c_char_p
    for name in ("epr_plan", "epr_forward", "epr_adjoint", "epr_transport", "epr_precondition", "epr_retrieve",
                 "epr_retrieve_oversampled", "epr_set_diagnostics", "epr_retrieve_host", "epr_plan_lines", "epr_destroy"):
        getattr(lib, name).restype = ci
    _LIB = lib
    return lib


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev(t, shape=None, name="tensor"):
    import torch
    if t is None:
        return C.c_void_p(0)
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous float32 CUDA tensor")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    return C.c_void_p(t.data_ptr())


class Plan:
    """Owner of an `epr_plan_t`.  Create with `epr_plan(...)`."""

    def __init__(self, handle, nx, ny, n_bins, solver, max_batch):
        self._h, self.nx, self.ny, self.n_bins, self.solver, self.max_batch = handle, nx, ny, n_bins, solver, max_batch

    def _check(self, status):
        if status != 0:
            raise EprError(status, load_library().epr_last_error(self._h).decode())

    def lines(self):
        """Per-line scalars derived by the plan: dict of float64 arrays f, gamma, a, alpha."""
        arrs = [np.zeros(self.n_bins) for _ in range(4)]
        ptrs = [a.ctypes.data_as(C.POINTER(C.c_double)) for a in arrs]
        self._check(load_library().epr_plan_lines(self._h, *ptrs))
        return dict(zip(("f", "gamma", "a", "alpha"), arrs))

    @property
    def launches(self):
        return int(load_library().epr_launch_count(self._h))

    def profile(self, on):
        """Enable / disable per-kernel CUDA-event timing inside the library."""
        self._check(load_library().epr_profile_enable(self._h, 1 if on else 0))

    def profile_read(self, reset=True):
        """{kernel family: (total_ms, launches)} accumulated while profiling was enabled (synchronises)."""
        n = 16
        names = (C.c_char_p * n)()
        ms = (C.c_double * n)()
        cnt = (C.c_longlong * n)()
        k = load_library().epr_profile_read(self._h, n, names, ms, cnt, 1 if reset else 0)
        return {names[i].decode(): (float(ms[i]), int(cnt[i])) for i in range(k)}

    def columns(self):
        """Per-column scalars the plan uses: dict of float64 arrays [n_bins][nx] f, gamma, a (epr_plan_columns)."""
        arrs = [np.zeros((self.n_bins, self.nx)) for _ in range(3)]
        ptrs = [a.ctypes.data_as(C.POINTER(C.c_double)) for a in arrs]
        self._check(load_library().epr_plan_columns(self._h, *ptrs))
        return dict(zip(("f", "gamma", "a"), arrs))

    def read_flags(self, clear=True):
        """EPR_FLAG_* bits raised by kernels since the last clear (epr_read_flags; synchronises)."""
        v = C.c_uint(0)
        self._check(load_library().epr_read_flags(self._h, C.byref(v), 1 if clear else 0))
        return int(v.value)

    def destroy(self):
        if self._h is not None:
            load_library().epr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def epr_plan(nx, ny, pixel_m, L_m, energy_keV, weight, delta_over_beta, solver="local", max_batch=1, **opts):
    """epr_plan of include/epr.h.  `opts`: fields of epr_options (order, wkb1, symbol, max_shift_px, i_min,
    newton_iters, init, output, out_bin, mu_rel, nonlocal_wkb1)."""
    lib = load_library()
    E = np.ascontiguousarray(np.atleast_1d(energy_keV), dtype=np.float64)
    w = np.ascontiguousarray(np.atleast_1d(weight), dtype=np.float64)
    db = np.ascontiguousarray(np.atleast_1d(delta_over_beta), dtype=np.float64)
    if not (E.size == w.size == db.size):
        raise ValueError("energy_keV, weight, delta_over_beta must have the same length")
    sv = {"local": EPR_LOCAL, "nonlocal": EPR_NONLOCAL}.get(solver, solver)
    o = Options()
    lib.epr_default_options(C.byref(o))
    keep = None
    for k, v in opts.items():
        if k == "mu_rel":
            keep = np.ascontiguousarray(v, dtype=np.float64)
            o.mu_rel = keep.ctypes.data_as(C.POINTER(C.c_double))
        elif hasattr(o, k):
            setattr(o, k, v)
        else:
            raise TypeError(f"unknown option {k}")
    h = C.c_void_p(0)
    dp = C.POINTER(C.c_double)
    st = lib.epr_plan(C.byref(h), int(nx), int(ny), float(pixel_m), float(L_m), int(E.size), E.ctypes.data_as(dp),
                      w.ctypes.data_as(dp), db.ctypes.data_as(dp), int(sv), int(max_batch), C.byref(o))
    if st != 0:
        msg = lib.epr_last_error(h).decode() if h.value else "invalid argument or unsupported size"
        if h.value:
            lib.epr_destroy(h)
        raise EprError(st, msg)
    return Plan(h, int(nx), int(ny), int(E.size), sv, int(max_batch))


def epr_plan_profiles(plan, weight_blk, delta_over_beta_blk, mu_rel_blk=None):
    """epr_plan_profiles of include/epr.h: [n_blocks][n_bins] arrays (x-dependent effective spectrum, reading R17)."""
    w = np.ascontiguousarray(np.atleast_2d(weight_blk), dtype=np.float64)
    db = np.ascontiguousarray(np.atleast_2d(delta_over_beta_blk), dtype=np.float64)
    if w.shape != db.shape or w.shape[1] != plan.n_bins:
        raise ValueError("weight_blk, delta_over_beta_blk: expected [n_blocks][n_bins]")
    dp = C.POINTER(C.c_double)
    mu = None
    if mu_rel_blk is not None:
        mu = np.ascontiguousarray(np.atleast_2d(mu_rel_blk), dtype=np.float64)
        if mu.shape != w.shape:
            raise ValueError("mu_rel_blk: expected [n_blocks][n_bins]")
    plan._check(load_library().epr_plan_profiles(plan._h, int(w.shape[0]), w.ctypes.data_as(dp), db.ctypes.data_as(dp),
                                                 mu.ctypes.data_as(dp) if mu is not None else None))


def epr_forward(plan, tau, P_sum, P_bins=None):
    b = tau.shape[0]
    plan._check(load_library().epr_forward(plan._h, b, _dev(tau, (b, plan.ny, plan.nx), "tau"),
                                           _dev(P_sum, (b, plan.ny, plan.nx), "P_sum"),
                                           _dev(P_bins, (b, plan.n_bins, plan.ny, plan.nx), "P_bins"), _stream()))


def epr_adjoint(plan, e_bins, r_bins):
    b = e_bins.shape[0]
    sh = (b, plan.n_bins, plan.ny, plan.nx)
    plan._check(load_library().epr_adjoint(plan._h, b, _dev(e_bins, sh, "e_bins"), _dev(r_bins, sh, "r_bins"), _stream()))


def epr_transport(plan, I_bins, P_bins):
    b = I_bins.shape[0]
    sh = (b, plan.n_bins, plan.ny, plan.nx)
    plan._check(load_library().epr_transport(plan._h, b, _dev(I_bins, sh, "I_bins"), _dev(P_bins, sh, "P_bins"), _stream()))


def epr_precondition(plan, r_bins, q_bins):
    b = r_bins.shape[0]
    sh = (b, plan.n_bins, plan.ny, plan.nx)
    plan._check(load_library().epr_precondition(plan._h, b, _dev(r_bins, sh, "r_bins"), _dev(q_bins, sh, "q_bins"), _stream()))


def epr_retrieve(plan, d, out, iterations, step):
    b = d.shape[0]
    sh = (b, plan.ny, plan.nx)
    plan._check(load_library().epr_retrieve(plan._h, b, _dev(d, sh, "d"), _dev(out, sh, "out"), int(iterations),
                                            float(step), _stream()))


def epr_retrieve_oversampled(plan, factor, d, out, iterations, step):
    """`plan` is the FINE grid's plan; d, out are [batch][ny / factor][nx / factor] (include/epr.h)."""
    b = d.shape[0]
    factor = int(factor)
    if factor < 1 or plan.ny % factor or plan.nx % factor:
        raise ValueError("factor must divide the plan's grid")
    sh = (b, plan.ny // factor, plan.nx // factor)
    plan._check(load_library().epr_retrieve_oversampled(plan._h, factor, b, _dev(d, sh, "d"), _dev(out, sh, "out"),
                                                        int(iterations), float(step), _stream()))


def epr_shift_histogram(plan, tau, n_hist, bin_px):
    """Per-line histogram of the unclamped shift norm of `tau` (epr_shift_histogram): int32 CUDA tensor [batch][n_bins][n_hist]."""
    import torch
    b = tau.shape[0]
    hist = torch.zeros((b, plan.n_bins, int(n_hist)), dtype=torch.int32, device=tau.device)
    plan._check(load_library().epr_shift_histogram(plan._h, b, _dev(tau, (b, plan.ny, plan.nx), "tau"), int(n_hist), float(bin_px),
                                                   C.c_void_p(hist.data_ptr()), _stream()))
    return hist


def epr_residual_rms_static(e_bins, rms):
    """epr_residual_rms_static of include/epr.h: RMS over the pixels of Σ_s e_bins[b][s], written to rms[b].

    For callers that must not allocate device memory (all of it already belongs to a pool, or a cudaMalloc stall is not
    acceptable in the loop): the reduction scratch is a fixed 512 KiB array inside libepr.so, so neither the library nor
    this wrapper allocates — `rms` ([batch], float32, CUDA) is the caller's, like `e_bins` ([batch][n_bins][ny][nx]).
    batch <= EPR_STATIC_MAX_BATCH.  Runs on the current device and torch's current stream; calls share the scratch, so
    keep them on one stream (or order them with events).  Make the first call on a device during set-up."""
    if e_bins.dim() != 4:
        raise ValueError("e_bins: expected [batch][n_bins][ny][nx]")
    b, n_bins, ny, nx = (int(v) for v in e_bins.shape)
    st = load_library().epr_residual_rms_static(b, n_bins, nx, ny, _dev(e_bins, None, "e_bins"), _dev(rms, (b,), "rms"),
                                                 _stream())
    if st != 0:
        raise EprError(st, load_library().epr_static_last_error().decode())


def epr_set_diagnostics(plan, diag):
    """diag: contiguous float32 CUDA tensor [batch][capacity_iters][2] (kept alive by the caller), or None to switch off."""
    if diag is None:
        plan._check(load_library().epr_set_diagnostics(plan._h, C.c_void_p(0), 0))
        return
    if diag.dim() != 3 or diag.shape[2] != 2:
        raise ValueError("diag: expected [batch][capacity_iters][2]")
    plan._check(load_library().epr_set_diagnostics(plan._h, _dev(diag, None, "diag"), int(diag.shape[1])))


def _host_ptr(a, name):
    if isinstance(a, np.ndarray):
        if a.dtype != np.float32 or not a.flags.c_contiguous:
            raise TypeError(f"{name}: expected C-contiguous float32")
        return C.c_void_p(a.ctypes.data), a.shape
    import torch
    if not isinstance(a, torch.Tensor) or a.is_cuda or a.dtype != torch.float32 or not a.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float32 host tensor")
    return C.c_void_p(a.data_ptr()), tuple(a.shape)


def epr_retrieve_host(plan, d_host, out_host, iterations, step, factor=1, wait=True):
    """HOST buffers (pinned float32 torch tensors or C-contiguous numpy arrays), copies inside the call.
    factor > 1: epr_retrieve_oversampled_host — buffers on the detector grid [batch][ny/factor][nx/factor].
    wait=False: epr_retrieve_host_async — the call only enqueues; keep the buffers alive and call epr_host_wait(plan)."""
    pd, sd = _host_ptr(d_host, "d_host")
    po, so = _host_ptr(out_host, "out_host")
    factor = int(factor)
    if factor < 1 or plan.ny % factor or plan.nx % factor:
        raise ValueError("factor must divide the plan's grid")
    if tuple(sd) != tuple(so) or tuple(sd[1:]) != (plan.ny // factor, plan.nx // factor):
        raise ValueError("d_host / out_host must both be [batch][ny / factor][nx / factor]")
    if not wait:
        if factor != 1:
            raise ValueError("the streaming session takes buffers on the plan's grid (factor = 1)")
        plan._check(load_library().epr_retrieve_host_async(plan._h, int(sd[0]), pd, po, int(iterations), float(step)))
    elif factor == 1:
        plan._check(load_library().epr_retrieve_host(plan._h, int(sd[0]), pd, po, int(iterations), float(step)))
    else:
        plan._check(load_library().epr_retrieve_oversampled_host(plan._h, factor, int(sd[0]), pd, po, int(iterations), float(step)))


def epr_shard_range(total, k, parts):
    """epr_shard_range of include/epr.h: (start, stop) of part k — host arithmetic, works without a device."""
    a, b = C.c_int(0), C.c_int(0)
    st = load_library().epr_shard_range(int(total), int(k), int(parts), C.byref(a), C.byref(b))
    if st != 0:
        raise EprError(st, "epr_shard_range: total >= 0, parts >= 1 and 0 <= k < parts required")
    return int(a.value), int(b.value)


def epr_host_wait(plan):
    """epr_host_wait of include/epr.h: returns when every epr_retrieve_host(..., wait=False) of the session has completed."""
    plan._check(load_library().epr_host_wait(plan._h))


def epr_retrieve_host_multi(plans, d_host, out_host, iterations, step):
    """epr_retrieve_host_multi of include/epr.h: ONE host batch split over `plans` (one per GPU), no exchange between them."""
    pd, sd = _host_ptr(d_host, "d_host")
    po, so = _host_ptr(out_host, "out_host")
    p0 = plans[0]
    if tuple(sd) != tuple(so) or tuple(sd[1:]) != (p0.ny, p0.nx):
        raise ValueError("d_host / out_host must both be [batch][ny][nx]")
    hs = (C.c_void_p * len(plans))(*[p._h.value for p in plans])
    st = load_library().epr_retrieve_host_multi(hs, len(plans), int(sd[0]), pd, po, int(iterations), float(step))
    if st != 0:
        msgs = [load_library().epr_last_error(p._h).decode() for p in plans]
        raise EprError(st, "; ".join(m for m in msgs if m))
