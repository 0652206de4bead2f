"""Pins for the adaptive-step Runge-Kutta Cash-Karp integrator of the CPU oracle (reading R-RK2'
of DESIGN.md section 3: the step-size control the GSL manual documents for the stepper the paper says it follows).
What fixes it from outside: the exact two-body solution (Kepler's equation) which the result must approach as eps -> 0
at the rate the control implies; the definition of the control (reject iff the error level exceeds 1.1, shrink by
0.9 r^(-1/4) but not below 1/5, grow by 0.9 r^(-1/5) within [1, 5] when r < 0.5, factors rounded down to multiples of
1/16) checked on single trial steps with r recomputed from the already pinned embedded error of rkck_step; "the step is rejected, e.g. positions, velocities and
time are not updated"; time reversal; the loop semantics shared with the other integrators."""
import math

import numpy as np

import oracle
from paper_1208_1157_b200 import workloads as W
from test_oracle_hermite import two_body


def _level(x, v, m, h, eps):
    """The error level of a trial step, from rkck_step's embedded error (pinned in test_oracle_rkck.py)."""
    _, _, ex, ev = oracle.rkck_step(x, v, m, h)
    X = np.linalg.norm(x, axis=1).max()
    V = np.linalg.norm(v, axis=1).max()
    return max(np.abs(ex).max() / (eps * X), np.abs(ev).max() / (eps * V))


def test_trial_step_follows_the_control_definition():
    pos, vel, mass = W.generate(0, n_sys=3)
    seen = set()
    for s in range(3):
        x, v, m = pos[s], vel[s], mass[s]
        for h in (0.4, 0.1, 0.03, 0.01, -0.05, 0.002):
            for eps in (1e-4, 1e-7, 1e-9, 1e-12):
                r0 = _level(x, v, m, h, eps)
                x1, v1, h1, r, ok = oracle.rkck_adaptive_trial(x, v, m, h, eps)
                assert abs(r / r0 - 1) < 1e-12
                if r0 > 1.1:  # rejected: the state is untouched, the next trial is smaller and never below h / 5
                    assert not ok and (x1 == x).all() and (v1 == v).all()
                    f = max(0.2, math.floor(16 * 0.9 * r0 ** -0.25) / 16)
                    assert abs(h1 / h - f) < 1e-12 and 0.2 <= h1 / h < 0.9
                    seen.add("reject" if f > 0.2 else "reject-floor")
                else:         # accepted: the fifth-order solution of rkck_step, bit for bit
                    x5, v5, _, _ = oracle.rkck_step(x, v, m, h)
                    assert ok and (x1 == x5).all() and (v1 == v5).all()
                    if r0 < 0.5:
                        f = min(5.0, max(1.0, math.floor(16 * 0.9 * r0 ** -0.2) / 16))
                        assert abs(h1 / h - f) < 1e-12 and 1.0 <= h1 / h <= 5.0
                        seen.add("grow" if 1.0 < f < 5.0 else "grow-cap" if f == 5.0 else "keep")
                    else:
                        assert h1 == h
                        seen.add("keep")
    assert {"reject", "reject-floor", "grow", "grow-cap", "keep"} <= seen  # every branch of the control was taken


def _kepler_error(eps, e=0.6, revolutions=1.5):
    x, v, m = two_body(e=e, M=0.4)
    nm = math.sqrt(m.sum())
    t_end = revolutions * 2 * math.pi / nm
    r = oracle.integrate(oracle.RKCK_ADAPTIVE, x[None], v[None], m[None], dt=0.05, t_end=t_end, max_steps=10**7, rk_eps=eps,
                         nthreads=1)
    assert r["status"][0] == oracle.DONE_TIME and r["time"][0] >= t_end
    xe, ve, _ = two_body(e=e, M=0.4 + nm * r["time"][0])  # no clipping of the last step (R10): compare at the time reached
    return max(np.abs(r["pos"][0] - xe).max(), np.abs(r["vel"][0] - ve).max()), int(r["nsteps"][0]), int(r["nreject"][0])


def test_converges_to_keplers_equation_as_the_tolerance_shrinks():
    """Error-per-step control of a method whose embedded estimate is O(h^5): steps ~ eps^(-1/5), global error ~ eps^(4/5)
    (between eps^0.7 and eps^1.1 over four decades), and small in absolute terms."""
    errs, steps = [], []
    for eps in (1e-6, 1e-8, 1e-10):
        err, n, nrej = _kepler_error(eps)
        errs.append(err)
        steps.append(n)
        assert nrej < 0.2 * n + 5
    assert errs[0] < 3e-4 and errs[2] < 3e-8
    slope = math.log10(errs[0] / errs[2]) / 4
    assert 0.7 < slope < 1.1, (errs, slope)
    growth = math.log10(steps[2] / steps[0]) / 4
    assert 0.17 < growth < 0.23, (steps, growth)  # 1/5


def test_step_follows_the_orbit_small_at_pericentre_large_at_apocentre():
    """The accepted steps of an e = 0.6 orbit: the control must shorten them near pericentre.  For a local error
    ~ h^5 x (fifth time derivative ~ r^-... ) the ratio of apocentre to pericentre steps is large; > 3 is enough to
    catch a control that does not react."""
    x, v, m = two_body(e=0.6, M=math.pi)  # start at apocentre
    nm = math.sqrt(m.sum())
    t, h, eps = 0.0, 0.05, 1e-9
    hs, ts = [], []
    while t < 2 * math.pi / nm:
        x1, v1, h1, r, ok = oracle.rkck_adaptive_trial(x, v, m, h, eps)
        if ok:
            hs.append(h)
            ts.append(t)
            t += h
            x, v = x1, v1
        h = h1
    hs, ts = np.array(hs), np.array(ts)
    peri = hs[np.abs(ts - math.pi / nm) < 0.3].mean()
    apo = hs[(ts > 1.0) & (ts < 0.2 * 2 * math.pi / nm)].mean() if ((ts > 1.0) & (ts < 0.2 * 2 * math.pi / nm)).any() else hs[3:8].mean()
    assert apo / peri > 3.0, (apo, peri)


def test_rejected_steps_do_not_advance_time_or_count_as_steps():
    """A first trial step far too large: the run starts with rejections (counted apart), time equals the sum of the
    accepted steps only, and the end state is close to the run that starts from a sensible step."""
    pos, vel, mass = W.generate(0, n_sys=6)
    a = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, dt=50.0, t_end=3.0, max_steps=10**6, rk_eps=1e-10)
    b = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, dt=0.01, t_end=3.0, max_steps=10**6, rk_eps=1e-10)
    assert (a["nreject"] >= 3).all() and (a["status"] == oracle.DONE_TIME).all()
    assert (a["time"] >= 3.0).all() and (a["time"] < 3.2).all()
    # one step budget: accepted steps only
    c = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, dt=50.0, max_steps=7, rk_eps=1e-10)
    assert (c["nsteps"] == 7).all() and (c["status"] == oracle.DONE_STEPS).all() and (c["nreject"] >= 3).all()
    # both runs approximate the same trajectory (compared through the Hermite oracle at the times they reached)
    for r in (a, b):
        for s in range(6):
            n = int(round(r["time"][s] / 1e-3))
            ref = oracle.integrate(oracle.HERMITE, pos[s:s + 1], vel[s:s + 1], mass[s:s + 1], dt=r["time"][s] / n, max_steps=n)
            assert np.abs(ref["pos"] - r["pos"][s]).max() < 2e-8


def test_direction_reversal_and_loop_semantics():
    pos, vel, mass = W.generate(0, n_sys=5)
    f = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, dt=0.02, t_end=4.0, max_steps=10**6, rk_eps=1e-11)
    b = oracle.integrate(oracle.RKCK_ADAPTIVE, f["pos"], f["vel"], mass, f["time"], dt=-0.02, t_end=0.0, max_steps=10**6,
                         rk_eps=1e-11)
    assert (b["status"] == oracle.DONE_TIME).all() and (b["time"] <= 0.0).all() and (b["time"] > -0.2).all()
    # back at (nearly) t = 0: propagate the small remainder exactly enough with Hermite to compare with the start
    for s in range(5):
        n = max(1, int(round(abs(b["time"][s]) / 1e-3)))
        r = oracle.integrate(oracle.HERMITE, b["pos"][s:s + 1], b["vel"][s:s + 1], mass[s:s + 1], dt=-b["time"][s] / n, max_steps=n)
        assert np.abs(r["pos"][0] - pos[s]).max() < 1e-8 and np.abs(r["vel"][0] - vel[s]).max() < 1e-8
    # monitors and sticky stops go through the common loop
    pos[2, 2] = pos[2, 1] + np.array([0.05, 0.0, 0.0])
    vel[2, 2] = vel[2, 1] + np.array([-0.5, 0.0, 0.0])
    m = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, dt=0.01, t_end=5.0, max_steps=10**6, rk_eps=1e-9, r_close=0.02)
    assert m["status"][2] == oracle.STOP_CLOSE and (np.delete(m["status"], 2) == oracle.DONE_TIME).all()
    # an unreachable tolerance (P:L321 prints eps = 5.0e-33) never loops for ever: at t = 0 the steps shrink until the
    # error estimate is exactly zero in FP64 and the run crawls; at a large time the shrinking step stops advancing the
    # clock and the system is stopped with STOP_STEPSIZE, its state untouched
    u = oracle.integrate(oracle.RKCK_ADAPTIVE, pos[:1], vel[:1], mass[:1], dt=0.01, max_steps=10, rk_eps=5.0e-33)
    assert u["status"][0] == oracle.DONE_STEPS and u["nsteps"][0] == 10 and 0 < u["time"][0] < 1e-12 and u["nreject"][0] > 10
    u = oracle.integrate(oracle.RKCK_ADAPTIVE, pos[:1], vel[:1], mass[:1], np.array([1e9]), dt=0.01, max_steps=10,
                         rk_eps=5.0e-33)
    assert u["status"][0] == oracle.STOP_STEPSIZE and u["nsteps"][0] == 0 and u["time"][0] == 1e9
    assert (u["pos"] == pos[:1]).all() and (u["vel"] == vel[:1]).all()


def test_double_and_long_double_take_the_same_steps():
    """The discrete step factors make the step sequence robust against rounding-level differences in the error
    estimate: the double and the 80-bit run take bit-identical steps (same times) for nearly every system, and then
    agree to rounding level; a system whose sequences differ (r within the noise of a boundary) is still within the
    tolerance scale of the other."""
    pos, vel, mass = W.generate(0, n_sys=48)
    a = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, dt=0.02, max_steps=400, rk_eps=1e-8)
    b = oracle.integrate(oracle.RKCK_ADAPTIVE, pos, vel, mass, dt=0.02, max_steps=400, rk_eps=1e-8, prec=oracle.LONG_DOUBLE)
    same = (a["nreject"] == b["nreject"]) & (np.abs(a["time"] - b["time"]) < 1e-12)
    assert same.sum() >= 44, same.sum()
    d = np.abs(a["pos"] - b["pos"]).max(axis=(1, 2)) / np.linalg.norm(b["pos"], axis=2).max(axis=1)
    assert d[same].max() < 1e-11, d
    dt = (a["time"] - b["time"])[:, None, None]
    d1 = np.abs(a["pos"] - (b["pos"] + b["vel"] * dt)).max(axis=(1, 2))
    assert d1.max() < 1e-5
