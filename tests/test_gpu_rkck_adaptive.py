"""GPU parity of the adaptive-step Runge-Kutta Cash-Karp kernel (ENS_RKCK_ADAPTIVE; reading
R-RK2') against the CPU oracle, through the C ABI.

What is unique and what is not: the error estimate is a difference of nearly equal sums, so the
error level r of a trial step carries relative rounding noise (1e-9..1e-7) that differs between two correct
implementations.  The control draws the step factors from a discrete set, so both sides take BIT-IDENTICAL step
sequences (same accepted and rejected counts, same times) unless some r falls within that noise of a decision boundary.
Systems with identical (nsteps, nreject, time) are compared at rounding level (1e-11 / 1e-10).  The others (rare:
counted, bounded) took a different but equally valid step sequence: they are compared at the level of the tolerance,
after moving the oracle's state to the GPU's end time to first order."""
import math

import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W
from parity import rel_diff
from test_gpu_mvs import _systems
from test_oracle_hermite import two_body

pytestmark = pytest.mark.gpu


def _compare(g, o, eps, tight, min_same):
    same = (g["nsteps"] == o["nsteps"]) & (g["nreject"] == o["nreject"]) & (g["time"] == o["time"]) & (g["status"] == o["status"])
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    print(f"adaptive rkck eps={eps:g}: {same.sum()} of {len(same)} systems took the oracle's exact step sequence; on those "
          f"pos max {dp[same].max():.2e} vel max {dv[same].max():.2e}")
    assert same.mean() >= min_same, same.mean()
    assert dp[same].max() <= tight and dv[same].max() <= tight
    if (~same).any():  # a different, equally valid sequence: tolerance-level agreement at the same time
        dt = (g["time"] - o["time"])[~same, None, None]
        xo = o["pos"][~same] + o["vel"][~same] * dt
        d = np.abs(g["pos"][~same] - xo).max(axis=(1, 2)) / np.linalg.norm(xo, axis=2).max(axis=1)
        assert np.abs(dt).max() <= 0.5 and d.max() <= 1e4 * eps, (np.abs(dt).max(), d.max())
        assert (g["status"][~same] == o["status"][~same]).all()


@pytest.mark.parametrize("eps", [1e-7, 1e-10])
def test_config0_systems_time_controlled(eps):
    pos, vel, mass = W.generate(0)
    g = ens.run(ens.RKCK_ADAPTIVE, pos, vel, mass, dt=0.02, steps=10**7, t_end=20.0, rk_eps=eps, want_energy=True)
    o = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, dt=0.02, t_end=20.0, max_steps=10**7, rk_eps=eps)
    assert (g["status"] == ens.DONE_TIME).all() and (g["time"] >= 20.0).all()
    assert g["nsteps"].min() != g["nsteps"].max()  # systems really take different numbers of steps
    _compare(g, o, eps, 1e-10, 0.97)
    assert np.abs((g["E"] - g["E0"]) / g["E0"]).max() < 1e3 * eps


@pytest.mark.parametrize("n_body", list(range(2, 17)))
def test_every_body_count_ragged_with_rejections_and_monitors(n_body):
    """Every lane / body split, a ragged ensemble, a first trial step far too large (several rejections), a hand-built
    close approach, step-count control."""
    n_sys = 77
    pos, vel, mass = _systems(n_sys, n_body, 950 + n_body)
    if n_body >= 3:
        pos[5, n_body - 1] = pos[5, n_body - 2] + np.array([0.05, 0.0, 0.0])
        vel[5, n_body - 1] = vel[5, n_body - 2] + np.array([-0.5, 0.0, 0.0])
    kw = dict(dt=3.0, r_close=0.02, r_eject=5000.0)
    g = ens.run(ens.RKCK_ADAPTIVE, pos, vel, mass, steps=60, rk_eps=1e-9, **kw)
    o = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, max_steps=60, rk_eps=1e-9, **kw)
    assert (o["nreject"] >= 2).all()
    if n_body >= 3:
        assert o["status"][5] == oracle.STOP_CLOSE and 0 < o["nsteps"][5] < 60
    _compare(g, o, 1e-9, 1e-11, 0.9)


def test_converges_to_keplers_equation_on_the_gpu():
    """Closed form on the GPU itself (e = 0.6, 1.5 revolutions): the error falls with the tolerance at the rate the
    control implies, as for the oracle (tests/test_oracle_rkck_adaptive.py)."""
    x, v, m = two_body(e=0.6, M=0.4)
    nm = math.sqrt(m.sum())
    t_end = 1.5 * 2 * math.pi / nm
    errs = []
    for eps in (1e-6, 1e-8, 1e-10):
        g = ens.run(ens.RKCK_ADAPTIVE, x[None], v[None], m[None], dt=0.05, steps=10**7, t_end=t_end, rk_eps=eps)
        xe, ve, _ = two_body(e=0.6, M=0.4 + nm * g["time"][0])
        errs.append(max(np.abs(g["pos"][0] - xe).max(), np.abs(g["vel"][0] - ve).max()))
    slope = math.log10(errs[0] / errs[2]) / 4
    assert errs[2] < 3e-8 and 0.7 < slope < 1.1, (errs, slope)


def test_direction_sticky_stops_stepsize_underflow_and_argument_checks():
    pos, vel, mass = W.generate(0, n_sys=100)
    with ens.Ensemble(100, 3) as e:
        e.set_state(pos, vel, mass)
        e.set_rk_tolerance(1e-10)
        e.integrate(ens.RKCK_ADAPTIVE, 0.02, 10**7, 4.0)
        f = e.get_state()
        e.integrate(ens.RKCK_ADAPTIVE, -0.02, 10**7, 0.0)
        b = e.get_state()
        assert (f["status"] == ens.DONE_TIME).all() and (b["status"] == ens.DONE_TIME).all()
        assert (b["time"] <= 0.0).all() and (b["time"] > -0.2).all()
        x0 = pos + vel * b["time"][:, None, None]  # the start, moved to the time reached, to first order
        assert rel_diff(b["pos"], x0).max() < 1e-3 and (e.get_rejected() >= 0).all()
        L = ens.lib()
        assert L.ens_set_rk_tolerance(e._h, 0.0) == ens.EINVAL and L.ens_set_rk_tolerance(None, 1e-9) == ens.EINVAL
        assert L.ens_get_rejected(e._h, None, ens.HOST, None) == ens.EINVAL
        # an unreachable tolerance at a large time: STOP_STEPSIZE, state untouched (as the oracle)
        time = np.full(100, 1e9)
        e.set_state(pos, vel, mass, time)
        e.set_rk_tolerance(5.0e-33)  # the value P:L321 prints
        e.integrate(ens.RKCK_ADAPTIVE, 0.01, 10)
        u = e.get_state()
        assert (u["status"] == ens.STOP_STEPSIZE).all() and (u["nsteps"] == 0).all() and (u["pos"] == pos).all()
        assert (e.get_rejected() > 5).all()
        e.integrate(ens.RKCK_ADAPTIVE, 0.01, 10)  # sticky
        assert (e.get_state()["status"] == ens.STOP_STEPSIZE).all()


def test_config1_full_size_sampled_parity():
    """Config 1's ensemble at FULL size (the persistent grid refills its lane groups ~1.7 times), tau-like run to
    t = 10; a strided sample against the oracle."""
    c = W.CONFIGS[1]
    pos, vel, mass = W.generate(1)
    g = ens.run(ens.RKCK_ADAPTIVE, pos, vel, mass, dt=0.02, steps=10**7, t_end=10.0, r_close=c.r_close, r_eject=c.r_eject,
                rk_eps=1e-9)
    assert np.isin(g["status"], [ens.DONE_TIME, ens.STOP_CLOSE, ens.STOP_EJECT]).all()
    assert (g["time"][g["status"] == ens.DONE_TIME] >= 10.0).all()
    idx = np.unique(np.concatenate([np.arange(0, c.n_sys, c.n_sys // 256), [c.n_sys - 1]]))
    o = oracle.integrate(oracle.RKCK_ADAPTIVE, pos[idx], vel[idx], mass[idx], dt=0.02, t_end=10.0, max_steps=10**7,
                         r_close=c.r_close, r_eject=c.r_eject, rk_eps=1e-9)
    _compare({k: g[k][idx] for k in ("pos", "vel", "time", "status", "nsteps", "nreject")}, o, 1e-9, 1e-10, 0.97)
