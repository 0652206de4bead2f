"""Pins for the fixed-step Runge-Kutta Cash-Karp integrator of the CPU oracle (reading R-RK1):
the Runge-Kutta order conditions (rooted trees up to order 5) on the tableau the oracle actually uses, measured order
of convergence 5 (embedded solution: 4) against Kepler's equation, agreement with the Hermite oracle at small steps
(the paper's own cross-validation), invariants and loop semantics."""
import math
from fractions import Fraction

import numpy as np

import oracle
from paper_1208_1157_b200 import workloads as W
from test_oracle_hermite import two_body


def test_tableau_satisfies_the_order_conditions():
    c, A6, b5, b4 = oracle.rkck_tableau()
    A = np.zeros((6, 6))
    A[:, :5] = A6
    assert np.abs(A.sum(axis=1) - c).max() < 1e-15 and np.triu(A).max() == 0.0  # explicit, row sums = nodes
    e = np.ones(6)
    Ac, Ac2, AAc, C = A @ c, A @ (c * c), A @ (A @ c), np.diag(c)
    # (elementary weight, 1 / density) for every rooted tree of order <= 5
    trees = {
        1: [(e, 1)],
        2: [(c, 2)],
        3: [(c**2, 3), (Ac, 6)],
        4: [(c**3, 4), (c * Ac, 8), (Ac2, 12), (AAc, 24)],
        5: [(c**4, 5), (c**2 * Ac, 10), (Ac * Ac, 20), (c * Ac2, 15), (A @ c**3, 20), (c * AAc, 30),
            (A @ (c * Ac), 40), (A @ Ac2, 60), (A @ AAc, 120)],
    }
    for order, lst in trees.items():
        for phi, gamma in lst:
            assert abs(b5 @ phi - 1.0 / gamma) < 2e-16 * 8, (order, gamma)          # fifth-order weights: all 17
            if order <= 4:
                assert abs(b4 @ phi - 1.0 / gamma) < 2e-16 * 8, (order, gamma)      # embedded weights: order 4
    assert abs(b4 @ c**4 - 0.2) > 1e-4  # ... and no more than 4
    # the printed rationals themselves (Cash & Karp 1990, as in every restatement of the method)
    assert Fraction(float(b5[0])).limit_denominator(10**6) == Fraction(37, 378)
    assert Fraction(float(A6[5, 3])).limit_denominator(10**7) == Fraction(44275, 110592)


def _err(N, which="5"):
    e, M0 = 0.3, 0.4
    x, v, m = two_body(e=e, M=M0)
    nm = math.sqrt(m.sum())
    t = 0.37 * 2 * math.pi / nm
    xe, ve, _ = two_body(e=e, M=M0 + nm * t)
    if which == "5":
        r = oracle.integrate(oracle.RKCK, x[None], v[None], m[None], dt=t / N, max_steps=N, nthreads=1, prec=oracle.LONG_DOUBLE)
        assert abs(r["time"][0] - t) < 1e-12
        return max(np.abs(r["pos"][0] - xe).max(), np.abs(r["vel"][0] - ve).max())
    # embedded 4th-order solution propagated instead: y4 = y5 - err, step by step
    h = t / N
    for _ in range(N):
        x5, v5, ex, ev = oracle.rkck_step(x, v, m, h, prec=oracle.LONG_DOUBLE)
        x, v = x5 - ex, v5 - ev
    return max(np.abs(x - xe).max(), np.abs(v - ve).max())


def test_fifth_order_convergence_against_keplers_equation():
    errs = [_err(N) for N in (100, 200, 400)]
    assert 27.0 < errs[0] / errs[1] < 37.0 and 27.0 < errs[1] / errs[2] < 37.0, errs
    assert errs[2] < 1e-9


def test_embedded_solution_is_fourth_order():
    errs = [_err(N, "4") for N in (100, 200, 400)]
    assert 13.0 < errs[0] / errs[1] < 19.0 and 13.0 < errs[1] / errs[2] < 19.0, errs


def test_agrees_with_hermite_at_small_steps():
    # "we compared their results to that of the GPU-based Hermite integrator ... sufficiently small time step"
    pos, vel, mass = W.generate(0, n_sys=8)
    a = oracle.integrate(oracle.RKCK, pos, vel, mass, dt=0.005, max_steps=2000)
    b = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.0025, max_steps=4000)
    d = np.abs(a["pos"] - b["pos"]).max(axis=(1, 2)) / np.linalg.norm(b["pos"], axis=2).max(axis=1)
    assert d.max() < 2e-10, d.max()


def test_invariants_loop_semantics_and_noise_floor():
    pos, vel, mass = W.generate(0, n_sys=16)
    E0, L0 = oracle.energy(pos, vel, mass)
    r = oracle.integrate(oracle.RKCK, pos, vel, mass, dt=0.01, max_steps=2000)
    E, L = oracle.energy(r["pos"], r["vel"], mass)
    assert np.abs((E - E0) / E0).max() < 1e-9 and np.abs(L - L0).max() < 1e-9 * np.abs(L0).max()
    assert (r["status"] == oracle.DONE_STEPS).all() and (r["nsteps"] == 2000).all()
    # the step is a pure function of the state: split runs are bit-identical
    a = oracle.integrate(oracle.RKCK, pos, vel, mass, dt=0.01, max_steps=700)
    b = oracle.integrate(oracle.RKCK, a["pos"], a["vel"], mass, a["time"], dt=0.01, max_steps=1300)
    assert (b["pos"] == r["pos"]).all() and (b["vel"] == r["vel"]).all()
    q = oracle.integrate(oracle.RKCK, pos, vel, mass, dt=0.01, max_steps=2000, prec=oracle.LONG_DOUBLE)
    d = np.abs(r["pos"] - q["pos"]).max(axis=(1, 2)) / np.linalg.norm(q["pos"], axis=2).max(axis=1)
    assert d.max() < 2e-12
    # time stop and monitors go through the same loop
    t = oracle.integrate(oracle.RKCK, pos, vel, mass, dt=0.01, max_steps=10**6, t_end=1.234)
    assert (t["status"] == oracle.DONE_TIME).all() and (t["nsteps"] == 124).all()
    pos[3, 2] = pos[3, 1] + np.array([0.05, 0.0, 0.0])
    vel[3, 2] = vel[3, 1] + np.array([-0.5, 0.0, 0.0])
    s = oracle.integrate(oracle.RKCK, pos, vel, mass, dt=0.001, max_steps=5000, r_close=0.02, r_eject=100.0)
    assert s["status"][3] == oracle.STOP_CLOSE and 50 < s["nsteps"][3] < 200
