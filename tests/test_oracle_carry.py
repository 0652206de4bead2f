"""Pins for the 2-evaluations-per-step Hermite variant of the oracle (Alg. 2 exactly as printed: a^(0),
j^(0) carried over from the previous step's last evaluation; reading R6-alt).  Order of convergence, the
Kepler closed form, invariants, and its distance from the 3-evaluation reading R6."""
import math

import numpy as np

import oracle
from paper_1208_1157_b200 import workloads as W
from test_oracle_hermite import two_body


def _run(x, v, m, dt, steps, prec=oracle.DOUBLE):
    r = oracle.integrate(oracle.HERMITE_CARRY, x[None], v[None], m[None], dt=dt, max_steps=steps, nthreads=1, prec=prec)
    return r["pos"][0], r["vel"][0], r


def test_fourth_order_convergence_and_keplers_equation():
    e, M0 = 0.3, 0.4
    x, v, m = two_body(e=e, M=M0)
    nm = math.sqrt(m.sum())
    T = 2 * math.pi / nm
    xe, ve, _ = two_body(e=e, M=M0 + nm * 0.37 * T)
    errs = []
    for N in (400, 800, 1600):
        x1, v1, r = _run(x, v, m, 0.37 * T / N, N, prec=oracle.LONG_DOUBLE)
        errs.append(max(np.abs(x1 - xe).max(), np.abs(v1 - ve).max()))
    assert 14.0 < errs[0] / errs[1] < 18.0 and 14.0 < errs[1] / errs[2] < 18.0, errs
    assert errs[2] < 1e-8


def test_first_step_equals_the_three_evaluation_step_and_later_ones_stay_close():
    # the first step of a call evaluates (a0, j0) at the state itself: identical to reading R6; afterwards the carried
    # (a2, j2) belong to the iterate before the last correction, an O(h^5) difference per step
    pos, vel, mass = W.generate(0, n_sys=16)
    a = oracle.integrate(oracle.HERMITE_CARRY, pos, vel, mass, dt=0.01, max_steps=1)
    b = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, max_steps=1)
    assert (a["pos"] == b["pos"]).all() and (a["vel"] == b["vel"]).all()
    a = oracle.integrate(oracle.HERMITE_CARRY, pos, vel, mass, dt=0.01, max_steps=2000)
    b = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, max_steps=2000)
    d = np.abs(a["pos"] - b["pos"]).max(axis=(1, 2)) / np.linalg.norm(b["pos"], axis=2).max(axis=1)
    assert 0 < d.max() < 5e-12, d.max()
    assert (a["status"] == oracle.DONE_STEPS).all() and (a["nsteps"] == 2000).all() and np.allclose(a["time"], 20.0)


def test_energy_angular_momentum_and_monitors():
    pos, vel, mass = W.generate(0, n_sys=16)
    E0, L0 = oracle.energy(pos, vel, mass)
    r = oracle.integrate(oracle.HERMITE_CARRY, pos, vel, mass, dt=0.01, max_steps=2000)
    E, L = oracle.energy(r["pos"], r["vel"], mass)
    assert np.abs((E - E0) / E0).max() < 1e-10
    assert np.abs(L - L0).max() < 1e-10 * np.abs(L0).max()  # Hermite conserves L only to truncation order
    pos[3, 2] = pos[3, 1] + np.array([0.05, 0.0, 0.0])
    vel[3, 2] = vel[3, 1] + np.array([-0.5, 0.0, 0.0])
    r = oracle.integrate(oracle.HERMITE_CARRY, pos, vel, mass, dt=0.001, max_steps=5000, r_close=0.02, r_eject=100.0)
    assert r["status"][3] == oracle.STOP_CLOSE and 50 < r["nsteps"][3] < 200
    assert np.linalg.norm(r["pos"][3, 2] - r["pos"][3, 1]) < 0.02  # the post-step state itself is inside the threshold


def test_double_vs_long_double_floor():
    pos, vel, mass = W.generate(0, n_sys=32)
    a = oracle.integrate(oracle.HERMITE_CARRY, pos, vel, mass, dt=0.01, max_steps=2000)
    b = oracle.integrate(oracle.HERMITE_CARRY, pos, vel, mass, dt=0.01, max_steps=2000, prec=oracle.LONG_DOUBLE)
    d = np.abs(a["pos"] - b["pos"]).max(axis=(1, 2)) / np.linalg.norm(b["pos"], axis=2).max(axis=1)
    assert d.max() < 2e-12
