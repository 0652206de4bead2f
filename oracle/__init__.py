"""CPU oracle for the ensemble Hermite / MVS step loop (arxiv 1208.1157).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.  It does not
import ``paper_1208_1157_b200`` and shares no code with it.

``oracle/ens_oracle.cpp`` holds the arithmetic (plain C++, one system at a time, IEEE double or 80-bit
long double).  This module compiles it with g++ on first use (``-O2 -ffp-contract=off``, no fast-math,
OpenMP only for the system-per-thread driver) and exposes it through ctypes with numpy arrays.
Array layout everywhere: C order, ``pos``/``vel`` ``[n_sys][n_body][3]``, ``mass`` ``[n_sys][n_body]``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ens_oracle.cpp")
_LIB = os.path.join(_HERE, "libens_oracle.so")
_lock = threading.Lock()
_lib = None

ACTIVE, DONE_TIME, DONE_STEPS, STOP_CLOSE, STOP_EJECT, STOP_NONFINITE, STOP_STEPSIZE = range(7)
HERMITE, MVS, HERMITE_ADAPTIVE, HERMITE_CARRY, RKCK, MVS_MERGED, RKCK_ADAPTIVE = 0, 1, 2, 3, 4, 5, 6
# MVS_MERGED: the adjacent half drifts / half kicks of consecutive steps merged.  RKCK_ADAPTIVE: `dt` is the first trial
# step, `rk_eps` the accuracy parameter (reading R-RK2').
# HERMITE_ADAPTIVE: `dt` is the step size scale tau of Eq. 5.  HERMITE_CARRY: Alg. 2 as printed, 2 evaluations per step.
DOUBLE, LONG_DOUBLE = 0, 1

CXXFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c++17"]


def build(force: bool = False) -> str:
    """Compile the oracle into ``oracle/libens_oracle.so`` (in-tree, git-ignored)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + f".{os.getpid()}.tmp"
            subprocess.check_call(["g++", *CXXFLAGS, "-o", tmp, _SRC])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        d = ctypes.POINTER(ctypes.c_double)
        i32 = ctypes.POINTER(ctypes.c_int32)
        i64 = ctypes.POINTER(ctypes.c_int64)
        ci, cl, cd = ctypes.c_int, ctypes.c_int64, ctypes.c_double
        lib.orc_acc_jerk.argtypes = [ci, d, d, d, d, d, ci]
        lib.orc_hermite_step.argtypes = [ci, d, d, d, cd, ci, ci]
        lib.orc_integrate.argtypes = [ci, cl, ci, d, d, d, d, i32, i64, cd, cd, cl, cd, cd, ci, ci]
        lib.orc_integrate2.argtypes = [ci, cl, ci, d, d, d, d, i32, i64, cd, cd, cl, cd, cd, ci, ci, cd, i64]
        lib.orc_rkck_adaptive_trial.argtypes = [ci, d, d, d, d, cd, d, ctypes.POINTER(ci), ci]
        lib.orc_adaptive_dt.argtypes = [ci, d, d, d, cd, d, ci]
        lib.orc_rkck_step.argtypes = [ci, d, d, d, cd, d, d, ci]
        lib.orc_rkck_tableau.argtypes = [d, d, d, d]
        lib.orc_energy.argtypes = [cl, ci, d, d, d, d, d, ci]
        lib.orc_stumpff.argtypes = [cd, d, ci]
        lib.orc_kepler_drift.argtypes = [d, d, cd, cd, ci, ctypes.POINTER(ci)]
        lib.orc_dh_roundtrip.argtypes = [ci, d, d, d, d, d, d, d]
        _lib = lib
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1


def acc_jerk(x, v, m, prec=DOUBLE):
    """(a, j) of one system: x, v ``[n][3]``, m ``[n]``.  Eq. 1 and its time derivative."""
    x, v, m = _f64(x), _f64(v), _f64(m)
    n = m.shape[0]
    a, j = np.empty_like(x), np.empty_like(x)
    rc = _load().orc_acc_jerk(n, _p(x), _p(v), _p(m), _p(a), _p(j), prec)
    assert rc == 0
    return a, j


def hermite_step(x, v, m, h, n_corr=2, prec=DOUBLE):
    """One Hermite step (Alg. 2) of one system; returns new (x, v)."""
    x, v, m = _f64(x).copy(), _f64(v).copy(), _f64(m)
    rc = _load().orc_hermite_step(m.shape[0], _p(x), _p(v), _p(m), float(h), int(n_corr), prec)
    assert rc == 0
    return x, v


def rkck_step(x, v, m, h, prec=DOUBLE):
    """One Cash-Karp step of one system; returns (x, v, errx, errv), err = 5th - 4th order solution."""
    x, v, m = _f64(x).copy(), _f64(v).copy(), _f64(m)
    ex, ev = np.empty_like(x), np.empty_like(v)
    rc = _load().orc_rkck_step(m.shape[0], _p(x), _p(v), _p(m), float(h), _p(ex), _p(ev), prec)
    assert rc == 0
    return x, v, ex, ev


def rkck_tableau():
    """(c[6], a[6][5], b5[6], b4[6]) exactly as the oracle holds them."""
    c, a, b5, b4 = np.empty(6), np.empty((6, 5)), np.empty(6), np.empty(6)
    assert _load().orc_rkck_tableau(_p(c), _p(a), _p(b5), _p(b4)) == 0
    return c, a, b5, b4


def adaptive_dt(x, v, m, tau, prec=DOUBLE):
    """Eq. 5: the step the adaptive Hermite integrator takes from state (x, v) of one system."""
    x, v, m = _f64(x), _f64(v), _f64(m)
    out = np.zeros(1)
    rc = _load().orc_adaptive_dt(m.shape[0], _p(x), _p(v), _p(m), float(tau), _p(out), prec)
    if rc:
        raise ValueError("orc_adaptive_dt: bad arguments")
    return float(out[0])


def rkck_adaptive_trial(x, v, m, h, eps, prec=DOUBLE):
    """One trial step of the adaptive Cash-Karp integrator (R-RK2'): returns (x, v, h_next, r, accepted)."""
    x, v, m = _f64(x).copy(), _f64(v).copy(), _f64(m)
    hh, r, ok = np.array([float(h)]), np.zeros(1), ctypes.c_int(0)
    rc = _load().orc_rkck_adaptive_trial(m.shape[0], _p(x), _p(v), _p(m), _p(hh), float(eps), _p(r), ctypes.byref(ok), prec)
    assert rc == 0
    return x, v, float(hh[0]), float(r[0]), bool(ok.value)


def integrate(integrator, pos, vel, mass, time=None, *, dt, t_end=np.inf, max_steps, r_close=0.0, r_eject=np.inf,
              status=None, nsteps=None, prec=DOUBLE, nthreads=None, rk_eps=1e-9):
    """Alg. 1 over an ensemble.  Returns dict(pos, vel, time, status, nsteps, nreject) (new arrays)."""
    pos, vel, mass = _f64(pos).copy(), _f64(vel).copy(), _f64(mass)
    n_sys, n = mass.shape
    assert pos.shape == (n_sys, n, 3) and vel.shape == (n_sys, n, 3)
    time = np.zeros(n_sys) if time is None else _f64(time).copy()
    status = np.zeros(n_sys, np.int32) if status is None else np.ascontiguousarray(status, np.int32).copy()
    nsteps = np.zeros(n_sys, np.int64) if nsteps is None else np.ascontiguousarray(nsteps, np.int64).copy()
    if nthreads is None:
        nthreads = host_cores()
    nreject = np.zeros(n_sys, np.int64)
    rc = _load().orc_integrate2(
        int(integrator), n_sys, n, _p(pos), _p(vel), _p(mass), _p(time),
        status.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), nsteps.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
        float(dt), float(t_end), int(max_steps), float(r_close), float(r_eject), prec, int(nthreads), float(rk_eps),
        nreject.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)))
    if rc != 0:
        raise ValueError("oracle: bad arguments")
    return dict(pos=pos, vel=vel, time=time, status=status, nsteps=nsteps, nreject=nreject)


def energy(pos, vel, mass, prec=DOUBLE):
    """(E [n_sys], L [n_sys][3]); Eq. 6 with each pair once."""
    pos, vel, mass = _f64(pos), _f64(vel), _f64(mass)
    n_sys, n = mass.shape
    E, L = np.empty(n_sys), np.empty((n_sys, 3))
    rc = _load().orc_energy(n_sys, n, _p(pos), _p(vel), _p(mass), _p(E), _p(L), prec)
    assert rc == 0
    return E, L


def stumpff(z, prec=DOUBLE):
    c = np.empty(4)
    assert _load().orc_stumpff(float(z), _p(c), prec) == 0
    return c


def kepler_drift(q, p, mu, tau, prec=DOUBLE):
    """Advance (q, p) along the Kepler orbit about a fixed centre; returns (q', p', newton_iters)."""
    q, p = _f64(q).copy(), _f64(p).copy()
    it = ctypes.c_int(0)
    assert _load().orc_kepler_drift(_p(q), _p(p), float(mu), float(tau), prec, ctypes.byref(it)) == 0
    return q, p, it.value


def dh_roundtrip(x, v, m):
    x, v, m = _f64(x), _f64(v), _f64(m)
    n = m.shape[0]
    Q, V, x2, v2 = (np.zeros_like(x) for _ in range(4))
    assert _load().orc_dh_roundtrip(n, _p(x), _p(v), _p(m), _p(Q), _p(V), _p(x2), _p(v2)) == 0
    return Q, V, x2, v2
