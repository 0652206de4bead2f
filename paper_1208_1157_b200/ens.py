"""Thin ctypes binding over the C ABI of ``include/ens.h`` (``libens.so``).  Same names, argument marshalling only:
every step of the path runs in the CUDA kernels of ``csrc/``.  torch is used for device memory and streams.

There is NO CPU fallback: if ``libens.so`` is missing it is compiled with nvcc on first use; if that fails the load
raises, and every call raises ``EnsError`` when the C function returns an error (e.g. no CUDA device).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np
import torch

OK, EINVAL, ENOMEM, ECUDA, ESTATE, EUNSUPPORTED, ETOOLARGE = 0, -1, -2, -3, -4, -5, -6
STATIC_MAX_GROUPS = 65536  # ens_hermite_static: warp-groups of systems its static scratch holds (include/ens.h)
# HERMITE_ADAPTIVE: `dt` is the step size scale tau of Eq. 5; RKCK_ADAPTIVE: `dt` is the first trial step
HERMITE, MVS, HERMITE_ADAPTIVE, HERMITE_CARRY, RKCK, MVS_MERGED, RKCK_ADAPTIVE = 0, 1, 2, 3, 4, 5, 6
HOST, DEVICE = 0, 1
ACTIVE, DONE_TIME, DONE_STEPS, STOP_CLOSE, STOP_EJECT, STOP_NONFINITE, STOP_STEPSIZE = range(7)
LOG_SNAPSHOTS, LOG_STOPS = 1, 2
OPT_THREADS, OPT_ADAPTIVE_UNORDERED, OPT_SLICE_MODE, OPT_SLICE_STEPS, OPT_SLICE_WARPS_PER_SM = range(5)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libens.so")
# every symbol include/ens.h declares (tests check that the library exports exactly these)
SYMBOLS = (
    "ens_create", "ens_destroy", "ens_set_state", "ens_set_monitors", "ens_integrate", "ens_get_state",
    "ens_energy", "ens_strerror", "ens_get_info", "ens_last_kernel_ms", "ens_fp64_peak", "ens_test_rsqrt",
    "ens_test_rcp", "ens_log_enable", "ens_integrate_logged", "ens_log_read", "ens_reserve_host_staging",
    "ens_test_set_option", "ens_set_rk_tolerance", "ens_get_rejected", "ens_hermite_static",
)
_lib = None


class EnsError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = lib().ens_strerror(code).decode() if _lib is not None else "?"
        super().__init__(f"{where}: error {code} ({msg})")


def lib() -> ctypes.CDLL:
    """Load ``libens.so`` (built in-tree by ``paper_1208_1157_b200.build``); fails loudly when it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            # a fresh checkout (the .so is git-ignored): compile it, once, with nvcc; never fall back to anything else
            try:
                from . import build as _build
                if os.path.abspath(LIB_PATH) != os.path.abspath(_build.LIB):
                    raise RuntimeError("a non-default LIB_PATH is never built implicitly")
                _build.build()
            except Exception as ex:
                raise ImportError(
                    f"{LIB_PATH} not found and could not be built ({ex}): run `python -m paper_1208_1157_b200.build` "
                    "(nvcc, sm_100a). There is no CPU fallback.") from ex
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, ci, cd = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
        L.ens_create.argtypes = [i64, ci, ctypes.POINTER(vp)]
        L.ens_destroy.argtypes = [vp]
        L.ens_set_state.argtypes = [vp, vp, vp, vp, vp, ci, vp]
        L.ens_set_monitors.argtypes = [vp, cd, cd]
        L.ens_integrate.argtypes = [vp, ci, cd, cd, i64, vp]
        L.ens_get_state.argtypes = [vp, vp, vp, vp, vp, vp, ci, vp]
        L.ens_energy.argtypes = [vp, vp, vp, ci, vp]
        L.ens_strerror.argtypes = [ci]
        L.ens_strerror.restype = ctypes.c_char_p
        L.ens_get_info.argtypes = [vp, ctypes.POINTER(i64)]
        L.ens_last_kernel_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
        L.ens_fp64_peak.argtypes = [i64, ctypes.POINTER(cd), vp]
        L.ens_test_rsqrt.argtypes = [vp, vp, i64, vp]
        L.ens_test_rcp.argtypes = [vp, vp, i64, vp]
        L.ens_log_enable.argtypes = [vp, i64, vp]
        L.ens_integrate_logged.argtypes = [vp, ci, cd, cd, i64, i64, ci, vp]
        L.ens_reserve_host_staging.argtypes = [vp]
        L.ens_set_rk_tolerance.argtypes = [vp, cd]
        L.ens_get_rejected.argtypes = [vp, vp, ci, vp]
        L.ens_test_set_option.argtypes = [vp, ci, i64]
        L.ens_hermite_static.argtypes = [vp, vp, vp, vp, vp, vp, i64, i64, ci, cd, cd, i64, cd, cd, vp]
        L.ens_log_read.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i64), vp, vp, vp, vp, vp, vp, i64, ci, vp]
        for name in SYMBOLS:
            if name != "ens_strerror":
                getattr(L, name).restype = ci
        _lib = L
    return _lib


def _check(rc: int, where: str):
    if rc != OK:
        raise EnsError(rc, where)


def _stream_ptr(stream) -> int | None:
    if stream is None:
        stream = torch.cuda.current_stream()
    if isinstance(stream, int):
        return stream or None
    return stream.cuda_stream or None


def _ptr(a, dtype, count: int, what: str):
    """(address, memspace, keepalive) of a numpy array / torch tensor holding >= count contiguous elements."""
    if a is None:
        return None, None, None
    if isinstance(a, torch.Tensor):
        tdt = {np.float64: torch.float64, np.int32: torch.int32, np.int64: torch.int64}[dtype]
        if a.dtype != tdt or not a.is_contiguous() or a.numel() < count:
            raise ValueError(f"{what}: need a contiguous {tdt} tensor with >= {count} elements")
        return a.data_ptr(), (DEVICE if a.is_cuda else HOST), a
    arr = np.ascontiguousarray(a, dtype=dtype)
    if arr.size < count:
        raise ValueError(f"{what}: need >= {count} elements")
    return arr.ctypes.data, HOST, arr


def _same_space(spaces, where):
    s = {x for x in spaces if x is not None}
    if len(s) > 1:
        raise ValueError(f"{where}: all arrays must live in the same memory space")
    return s.pop() if s else HOST


class Ensemble:
    """Handle on an ensemble of ``n_sys`` systems of ``n_body`` bodies resident on the current CUDA device."""

    def __init__(self, n_sys: int, n_body: int):
        self.n_sys, self.n_body = int(n_sys), int(n_body)
        h = ctypes.c_void_p()
        self._lib = lib()  # kept on the instance: module globals may already be gone when __del__ runs at exit
        _check(self._lib.ens_create(self.n_sys, self.n_body, ctypes.byref(h)), "ens_create")
        self._h = h

    def close(self):
        if getattr(self, "_h", None):
            self._lib.ens_destroy(self._h)
            self._h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- ens_set_state ------------------------------------------------------------------------------
    def set_state(self, pos, vel, mass, time=None, stream=None):
        n, nb = self.n_sys, self.n_body
        p, sp, k1 = _ptr(pos, np.float64, n * nb * 3, "pos")
        v, sv, k2 = _ptr(vel, np.float64, n * nb * 3, "vel")
        m, sm, k3 = _ptr(mass, np.float64, n * nb, "mass")
        t, st, k4 = _ptr(time, np.float64, n, "time")
        space = _same_space([sp, sv, sm, st], "ens_set_state")
        _check(lib().ens_set_state(self._h, p, v, m, t, space, _stream_ptr(stream)), "ens_set_state")
        if space == DEVICE:
            self._keep = (k1, k2, k3, k4)  # caller-owned inputs must outlive the enqueued kernels

    # -- ens_set_monitors ---------------------------------------------------------------------------
    def set_monitors(self, r_close: float = 0.0, r_eject: float = float("inf")):
        _check(lib().ens_set_monitors(self._h, float(r_close), float(r_eject)), "ens_set_monitors")

    # -- ens_set_rk_tolerance / ens_get_rejected -------------------------------------------------------
    def set_rk_tolerance(self, eps: float):
        _check(lib().ens_set_rk_tolerance(self._h, float(eps)), "ens_set_rk_tolerance")

    def get_rejected(self, stream=None):
        out = np.empty(self.n_sys, np.int64)
        _check(lib().ens_get_rejected(self._h, out.ctypes.data, HOST, _stream_ptr(stream)), "ens_get_rejected")
        return out

    # -- ens_integrate ------------------------------------------------------------------------------
    def integrate(self, integrator: int, dt: float, max_steps: int, t_end: float = float("inf"), stream=None):
        _check(lib().ens_integrate(self._h, int(integrator), float(dt), float(t_end), int(max_steps),
                                   _stream_ptr(stream)), "ens_integrate")

    # -- ens_get_state ------------------------------------------------------------------------------
    def get_state(self, device: bool = False, stream=None, out=None):
        """Returns dict(pos, vel, time, status, nsteps): numpy arrays (host) or torch CUDA tensors (device=True).
        ``out`` may supply preallocated arrays/tensors (e.g. pinned host tensors) under the same keys."""
        n, nb = self.n_sys, self.n_body
        out = dict(out) if out else {}
        if device:
            mk = lambda shape, dt: torch.empty(shape, dtype=dt, device="cuda")
            dts = dict(pos=torch.float64, vel=torch.float64, time=torch.float64, status=torch.int32, nsteps=torch.int64)
        else:
            mk = lambda shape, dt: np.empty(shape, dtype=dt)
            dts = dict(pos=np.float64, vel=np.float64, time=np.float64, status=np.int32, nsteps=np.int64)
        shapes = dict(pos=(n, nb, 3), vel=(n, nb, 3), time=(n,), status=(n,), nsteps=(n,))
        npdt = dict(pos=np.float64, vel=np.float64, time=np.float64, status=np.int32, nsteps=np.int64)
        ptrs, spaces = {}, []
        for key in ("pos", "vel", "time", "status", "nsteps"):
            if key not in out:
                out[key] = mk(shapes[key], dts[key])
            a = out[key]
            if not isinstance(a, torch.Tensor) and not (a.flags.c_contiguous and a.dtype == npdt[key]):
                raise ValueError(f"out[{key}] must be C-contiguous {npdt[key]}")
            ptrs[key], sp, _ = _ptr(a, npdt[key], int(np.prod(shapes[key])), key)
            spaces.append(sp)
        space = _same_space(spaces, "ens_get_state")
        _check(lib().ens_get_state(self._h, ptrs["pos"], ptrs["vel"], ptrs["time"], ptrs["status"], ptrs["nsteps"],
                                   space, _stream_ptr(stream)), "ens_get_state")
        return out

    # -- ens_energy ---------------------------------------------------------------------------------
    def energy(self, device: bool = False, stream=None):
        """(E [n_sys], L [n_sys][3])"""
        n = self.n_sys
        if device:
            E = torch.empty(n, dtype=torch.float64, device="cuda")
            L = torch.empty((n, 3), dtype=torch.float64, device="cuda")
            _check(lib().ens_energy(self._h, E.data_ptr(), L.data_ptr(), DEVICE, _stream_ptr(stream)), "ens_energy")
        else:
            E, L = np.empty(n), np.empty((n, 3))
            _check(lib().ens_energy(self._h, E.ctypes.data, L.ctypes.data, HOST, _stream_ptr(stream)), "ens_energy")
        return E, L

    # -- ens_log_enable / ens_integrate_logged / ens_log_read ------------------------------------------
    def log_enable(self, capacity: int, stream=None):
        _check(lib().ens_log_enable(self._h, int(capacity), _stream_ptr(stream)), "ens_log_enable")
        self._log_capacity = int(capacity)

    def integrate_logged(self, integrator: int, dt: float, max_steps: int, log_every: int, what: int = LOG_SNAPSHOTS,
                         t_end: float = float("inf"), stream=None):
        _check(lib().ens_integrate_logged(self._h, int(integrator), float(dt), float(t_end), int(max_steps),
                                          int(log_every), int(what), _stream_ptr(stream)), "ens_integrate_logged")

    def log_read(self, stream=None):
        """dict(sys, nsteps, time, status, pos, vel, dropped) of the records appended so far (host arrays)."""
        cap, nb = self._log_capacity, self.n_body
        out = dict(sys=np.empty(cap, np.int64), nsteps=np.empty(cap, np.int64), time=np.empty(cap),
                   status=np.empty(cap, np.int32), pos=np.empty((cap, nb, 3)), vel=np.empty((cap, nb, 3)))
        n, dropped = ctypes.c_int64(), ctypes.c_int64()
        _check(lib().ens_log_read(self._h, ctypes.byref(n), ctypes.byref(dropped), out["sys"].ctypes.data,
                                  out["nsteps"].ctypes.data, out["time"].ctypes.data, out["status"].ctypes.data,
                                  out["pos"].ctypes.data, out["vel"].ctypes.data, cap, HOST, _stream_ptr(stream)),
               "ens_log_read")
        out = {k: v[:n.value] for k, v in out.items()}
        out["dropped"] = dropped.value
        return out

    # -- helpers ------------------------------------------------------------------------------------
    def reserve_host_staging(self):
        _check(lib().ens_reserve_host_staging(self._h), "ens_reserve_host_staging")

    def set_option(self, option: int, value: int):
        _check(lib().ens_test_set_option(self._h, int(option), int(value)), "ens_test_set_option")

    def info(self) -> dict:
        buf = (ctypes.c_int64 * 10)()
        _check(lib().ens_get_info(self._h, buf), "ens_get_info")
        keys = ("n_pad", "lanes_per_system", "bodies_per_lane", "threads", "blocks", "regs", "blocks_per_sm", "launches",
                "stack_bytes", "sliced")
        return dict(zip(keys, list(buf)))

    def last_kernel_ms(self) -> float:
        ms = ctypes.c_float()
        _check(lib().ens_last_kernel_ms(self._h, ctypes.byref(ms)), "ens_last_kernel_ms")
        return ms.value


def hermite_static(pos, vel, mass, time, status, nsteps, n_sys: int, n_body: int, dt: float, max_steps: int,
                   t_end: float = float("inf"), r_close: float = 0.0, r_eject: float = float("inf"), stream=None):
    """``ens_hermite_static``: the fixed-step Hermite loop on caller-owned CUDA tensors in the library's SoA layout
    (pos, vel [n_body * 3][n_pad], mass [n_body][n_pad], time, status int32, nsteps int64 [n_pad]), advanced in place;
    the library allocates nothing (its scratch is a static device array shared by all calls: keep calls stream-ordered)."""
    n_pad = int(time.numel())
    ptrs = []
    for a, dt_, cnt, what in ((pos, np.float64, n_body * 3 * n_pad, "pos"), (vel, np.float64, n_body * 3 * n_pad, "vel"),
                              (mass, np.float64, n_body * n_pad, "mass"), (time, np.float64, n_pad, "time"),
                              (status, np.int32, n_pad, "status"), (nsteps, np.int64, n_pad, "nsteps")):
        ptr, space, _ = _ptr(a, dt_, cnt, what)
        if space != DEVICE:
            raise ValueError(f"ens_hermite_static: {what} must be a CUDA tensor")
        ptrs.append(ptr)
    _check(lib().ens_hermite_static(*ptrs, int(n_sys), n_pad, int(n_body), float(dt), float(t_end), int(max_steps),
                                    float(r_close), float(r_eject), _stream_ptr(stream)), "ens_hermite_static")


def fp64_peak(iters: int = 200000, stream=None) -> float:
    """Measured FP64 lane-FMA/s of the device (DFMA-chain microbenchmark)."""
    r = ctypes.c_double()
    _check(lib().ens_fp64_peak(int(iters), ctypes.byref(r), _stream_ptr(stream)), "ens_fp64_peak")
    return r.value


def rsqrt_probe(x: torch.Tensor) -> torch.Tensor:
    y = torch.empty_like(x)
    _check(lib().ens_test_rsqrt(x.data_ptr(), y.data_ptr(), x.numel(), _stream_ptr(None)), "ens_test_rsqrt")
    return y


def rcp_probe(x: torch.Tensor) -> torch.Tensor:
    y = torch.empty_like(x)
    _check(lib().ens_test_rcp(x.data_ptr(), y.data_ptr(), x.numel(), _stream_ptr(None)), "ens_test_rcp")
    return y


def run(cfg_or_integrator, pos, vel, mass, *, dt, steps, r_close=0.0, r_eject=float("inf"), t_end=float("inf"),
        time=None, want_energy=False, rk_eps=None):
    """Convenience: create, set, integrate, get (host arrays in, host arrays out).  Used by the tests."""
    n_sys, n_body = mass.shape
    with Ensemble(n_sys, n_body) as e:
        e.set_state(pos, vel, mass, time)
        e.set_monitors(r_close, r_eject)
        if rk_eps is not None:
            e.set_rk_tolerance(rk_eps)
        E0 = e.energy() if want_energy else None
        e.integrate(cfg_or_integrator, dt, steps, t_end)
        out = e.get_state()
        out["nreject"] = e.get_rejected()
        if want_energy:
            out["E0"], out["L0"] = E0
            out["E"], out["L"] = e.energy()
        out["info"] = e.info()
    return out
