"""Pins for the adaptive-step Hermite integrator of the CPU oracle (Eq. 5; readings R-A1..R-A3 of
DESIGN.md §3), none of which re-types the oracle's own loop: the closed form of Eq. 5 on a circular two-body orbit,
its scaling laws, the exact Kepler solution at the time actually reached, order of convergence in tau, the gain over
a fixed step on an eccentric orbit, and the loop semantics."""
import math

import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import workloads as W
from test_oracle_hermite import two_body


def run_adaptive(x, v, m, tau, steps=10**9, **kw):
    r = oracle.integrate(oracle.HERMITE_ADAPTIVE, x[None], v[None], m[None], dt=tau, max_steps=steps, nthreads=1, **kw)
    return r["pos"][0], r["vel"][0], r


def test_eq5_closed_form_on_a_circular_two_body_orbit():
    # On a circular orbit every body's acceleration vector rotates at the orbital rate w without changing length, so
    # |j_i| = w |a_i| for BOTH bodies (R-A1: the sum runs over all bodies, star included) and Eq. 5 gives
    # dt = tau / (w sqrt 2), independent of the masses.  A sum over planets only would give tau / w.
    for a, m1 in ((1.0, 1e-3), (2.5, 0.3)):
        x, v, m = two_body(e=0.0, a=a, m1=m1)
        w = math.sqrt(m.sum() / a**3)
        tau = 0.017
        assert abs(oracle.adaptive_dt(x, v, m, tau) * w * math.sqrt(2.0) / tau - 1.0) < 1e-13
        assert abs(oracle.adaptive_dt(x, v, m, -tau) * w * math.sqrt(2.0) / tau + 1.0) < 1e-13  # sign of tau


def test_eq5_scaling_laws():
    # dt is linear in tau, and under x -> L x, v -> L^(-1/2) v (same masses) every time scale of the system grows by
    # L^(3/2): pins the exponent -1/2 and that the ratio is |j|^2/|a|^2 (dimension 1/time^2), for n > 2 bodies.
    pos, vel, mass = W.generate(2, n_sys=4)
    for s in range(4):
        x, v, m = pos[s], vel[s], mass[s]
        d1 = oracle.adaptive_dt(x, v, m, 0.01, prec=oracle.LONG_DOUBLE)
        assert abs(oracle.adaptive_dt(x, v, m, 0.03, prec=oracle.LONG_DOUBLE) / d1 - 3.0) < 1e-14
        lam = 2.7
        d2 = oracle.adaptive_dt(lam * x, v / math.sqrt(lam), m, 0.01, prec=oracle.LONG_DOUBLE)
        assert abs(d2 / d1 / lam**1.5 - 1.0) < 1e-14
        # a Galilean boost changes neither accelerations nor jerks
        d3 = oracle.adaptive_dt(x + 5.0, v + np.array([0.3, -0.2, 0.1]), m, 0.01, prec=oracle.LONG_DOUBLE)
        assert abs(d3 / d1 - 1.0) < 1e-12


def test_eq5_matches_the_pinned_acceleration_and_jerk():
    # plumbing: the dt the integrator takes is Eq. 5 of the (separately pinned) acc/jerk routine, body by body
    pos, vel, mass = W.generate(3, n_sys=2)
    for s in range(2):
        a, j = oracle.acc_jerk(pos[s], vel[s], mass[s])
        ratio = (j * j).sum(axis=1) / (a * a).sum(axis=1)
        assert abs(oracle.adaptive_dt(pos[s], vel[s], mass[s], 0.02) / (0.02 / math.sqrt(ratio.sum())) - 1.0) < 1e-14
        _, _, r = run_adaptive(pos[s], vel[s], mass[s], 0.02, steps=1)
        assert r["time"][0] == oracle.adaptive_dt(pos[s], vel[s], mass[s], 0.02) and r["nsteps"][0] == 1


def test_massless_companion_contributes_nothing():
    # R-A2: a body that feels no acceleration (the only other body is massless) is left out of the sum
    x, v, m = two_body(e=0.0, a=1.0, m1=0.0)  # test particle on a circular orbit of rate w = 1 about a unit mass
    assert m[1] == 0.0
    assert abs(oracle.adaptive_dt(x, v, m, 0.01) / 0.01 - 1.0) < 1e-13  # planet's ratio alone: tau / w


def _kepler_error(e, tau, t_target):
    x, v, m = two_body(e=e, M=0.3)
    x1, v1, r = run_adaptive(x, v, m, tau, t_end=t_target)
    t = r["time"][0]
    nmean = math.sqrt(m.sum())
    xe, ve, _ = two_body(e=e, M=0.3 + nmean * t)  # exact solution at the time actually reached (no clipping, R10)
    return max(np.abs(x1 - xe).max(), np.abs(v1 - ve).max()), int(r["nsteps"][0]), t


def test_fourth_order_convergence_in_tau():
    errs = [_kepler_error(0.5, tau, 2 * math.pi)[0] for tau in (0.04, 0.02, 0.01)]
    assert 13.0 < errs[0] / errs[1] < 19.0 and 13.0 < errs[1] / errs[2] < 19.0, errs


def test_adaptive_beats_fixed_step_on_an_eccentric_orbit():
    # e = 0.9: with the same number of steps over one period the adaptive integrator (steps shrink as r^2 towards
    # pericentre) is orders of magnitude more accurate than the fixed-step one -- the reason Eq. 5 exists.
    e = 0.9
    err_a, n_a, t = _kepler_error(e, 0.02, 2 * math.pi)
    x, v, m = two_body(e=e, M=0.3)
    r = oracle.integrate(oracle.HERMITE, x[None], v[None], m[None], dt=t / n_a, max_steps=n_a, nthreads=1)
    xe, ve, _ = two_body(e=e, M=0.3 + math.sqrt(m.sum()) * r["time"][0])
    err_f = max(np.abs(r["pos"][0] - xe).max(), np.abs(r["vel"][0] - ve).max())
    assert err_a < 1e-5 and err_f > 100 * err_a, (err_a, err_f, n_a)
    # closed form at the apsides: the radial velocity vanishes there, so both bodies' accelerations rotate at the
    # angular rate w = L / r^2 without changing length and Eq. 5 gives dt = tau / (w sqrt 2), w = sqrt(mu a (1-e^2)) / r^2
    for M, r_aps in ((0.0, 1.0 - e), (math.pi, 1.0 + e)):
        x, v, m = two_body(e=e, M=M)
        w = math.sqrt(m.sum() * (1.0 - e * e)) / r_aps**2
        assert abs(oracle.adaptive_dt(x, v, m, 0.02) * w * math.sqrt(2.0) / 0.02 - 1.0) < 1e-9


def test_loop_semantics_time_steps_and_direction():
    pos, vel, mass = W.generate(0, n_sys=6)
    r = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.02, max_steps=10**6, t_end=3.0)
    assert (r["status"] == oracle.DONE_TIME).all() and (r["time"] >= 3.0).all()
    assert (r["time"] < 3.0 + 0.1).all()  # last step not clipped, but short (R10)
    assert len(set(r["nsteps"].tolist())) > 1  # systems take different numbers of steps
    r2 = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.02, max_steps=7)
    assert (r2["status"] == oracle.DONE_STEPS).all() and (r2["nsteps"] == 7).all()
    # split run is bit-identical (the step is a pure function of the state, R6)
    a = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.02, max_steps=4)
    b = oracle.integrate(oracle.HERMITE_ADAPTIVE, a["pos"], a["vel"], mass, a["time"], dt=0.02, max_steps=3)
    assert (b["pos"] == r2["pos"]).all() and (b["time"] == r2["time"]).all()
    # backward: tau < 0 walks time down; not time-symmetric, so the return is only approximate
    f = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.01, max_steps=200)
    g = oracle.integrate(oracle.HERMITE_ADAPTIVE, f["pos"], f["vel"], mass, f["time"], dt=-0.01, max_steps=10**6, t_end=0.0)
    assert (g["status"] == oracle.DONE_TIME).all() and (g["time"] <= 0.0).all() and (g["time"] > -0.1).all()


def test_energy_conservation_improves_as_tau_to_the_fourth():
    pos, vel, mass = W.generate(0, n_sys=8)
    E0, _ = oracle.energy(pos, vel, mass)
    errs = []
    for tau in (0.08, 0.04):
        r = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=tau, max_steps=10**6, t_end=20.0,
                             prec=oracle.LONG_DOUBLE)
        E, _ = oracle.energy(r["pos"], r["vel"], mass, prec=oracle.LONG_DOUBLE)
        errs.append(np.abs((E - E0) / E0))
    ratio = np.median(errs[0] / errs[1])
    assert 8.0 < ratio < 40.0, ratio


def test_close_approach_monitor_works_with_adaptive_steps():
    pos, vel, mass = W.generate(0, n_sys=4)
    pos[1, 2] = pos[1, 1] + np.array([0.05, 0.0, 0.0])  # planet 2 flies straight at planet 1
    vel[1, 2] = vel[1, 1] + np.array([-0.5, 0.0, 0.0])
    r = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.02, max_steps=10**5, t_end=50.0, r_close=0.02,
                         r_eject=100.0)
    assert r["status"][1] == oracle.STOP_CLOSE and (np.delete(r["status"], 1) == oracle.DONE_TIME).all()
    d = np.linalg.norm(r["pos"][1, 2] - r["pos"][1, 1])
    assert d < 0.02 and 0.05 < r["time"][1] < 0.2  # stopped on the first post-step state inside the threshold
