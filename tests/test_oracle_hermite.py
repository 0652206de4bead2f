"""Pins for the Hermite half of the CPU oracle (oracle/ens_oracle.cpp), none of which re-types its formulas:
closed forms (2-body force, Kepler orbit, Kepler's equation, E = -m0 m1 / 2a), gradients of the energy
function, finite differences, order of convergence, the symmetric-corrector identity, reversal, invariants,
and hand-built monitor crossings.  `P:L<n>` = /root/reference/PAPER.md line n; R<k> = DESIGN.md §3 readings.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import workloads as W


def two_body(e=0.3, a=1.0, m0=1.0, m1=1e-3, M=0.0):
    """Barycentric 2-body system from Keplerian elements (relative orbit mu = m0 + m1)."""
    z = np.array([0.0])
    q, p = W.elements_to_cartesian(np.array([a]), np.array([e]), z, z, z, np.array([M]), m0 + m1)
    q, p = q[0], p[0]
    mt = m0 + m1
    x = np.array([-m1 / mt * q, m0 / mt * q])
    v = np.array([-m1 / mt * p, m0 / mt * p])
    return x, v, np.array([m0, m1])


def run1(x, v, m, dt, steps, **kw):
    r = oracle.integrate(oracle.HERMITE, x[None], v[None], m[None], dt=dt, max_steps=steps, nthreads=1, **kw)
    return r["pos"][0], r["vel"][0], r


# ------------------------------------------------------------------------------------------ eval (a, j)
def test_acc_two_body_closed_form():
    # Eq. 1 (R1): |a_1| = m_0 / r^2 towards body 0, |a_0| = m_1 / r^2 towards body 1
    x = np.array([[0.1, -0.2, 0.3], [1.3, 0.9, -0.5]])
    v = np.zeros((2, 3))
    m = np.array([2.0, 0.25])
    a, j = oracle.acc_jerk(x, v, m)
    d = x[1] - x[0]
    r = np.linalg.norm(d)
    np.testing.assert_allclose(a[0], m[1] * d / r**3, rtol=1e-15)
    np.testing.assert_allclose(a[1], -m[0] * d / r**3, rtol=1e-15)
    np.testing.assert_allclose(j, 0.0, atol=1e-300)  # bodies at rest: jerk vanishes


def _rand_system(n, seed):
    rng = np.random.default_rng(seed)
    return rng.normal(size=(n, 3)) * 2.0, rng.normal(size=(n, 3)), 10.0 ** rng.uniform(-3, 0, size=n)


@pytest.mark.parametrize("n", [2, 3, 4, 7])
def test_acc_is_gradient_of_the_potential(n):
    # m_i a_i = -dU/dx_i with U the potential part of Eq. 6 (R9); pins every term, sign and index of
    # the acceleration against a DIFFERENT function of the oracle (energy) by central differences.
    x, v, m = _rand_system(n, 10 + n)
    a, _ = oracle.acc_jerk(x, v, m, prec=oracle.LONG_DOUBLE)
    zero = np.zeros_like(v)
    eps = 1e-4
    for i in range(n):
        for c in range(3):
            def U(h):
                xx = x.copy()
                xx[i, c] += h
                return oracle.energy(xx[None], zero[None], m[None], prec=oracle.LONG_DOUBLE)[0][0]
            # 4th-order central difference
            g = (-U(2 * eps) + 8 * U(eps) - 8 * U(-eps) + U(-2 * eps)) / (12 * eps)
            assert abs(m[i] * a[i, c] + g) < 2e-9 * max(1.0, abs(g)), (i, c)


@pytest.mark.parametrize("n", [2, 3, 5])
def test_jerk_is_time_derivative_of_acc(n):
    # j = da/dt along x(t) = x + v t (R2): central finite difference of the oracle's own acceleration
    x, v, m = _rand_system(n, 20 + n)
    _, j = oracle.acc_jerk(x, v, m, prec=oracle.LONG_DOUBLE)
    eps = 1e-4
    acc = lambda h: oracle.acc_jerk(x + v * h, v, m, prec=oracle.LONG_DOUBLE)[0]
    fd = (-acc(2 * eps) + 8 * acc(eps) - 8 * acc(-eps) + acc(-2 * eps)) / (12 * eps)
    np.testing.assert_allclose(j, fd, rtol=0, atol=3e-9 * np.abs(j).max())


def test_newton_third_law_sums_vanish():
    x, v, m = _rand_system(6, 3)
    a, j = oracle.acc_jerk(x, v, m)
    assert np.abs((m[:, None] * a).sum(0)).max() < 1e-14 * np.abs(m[:, None] * a).max()
    assert np.abs((m[:, None] * j).sum(0)).max() < 1e-14 * np.abs(m[:, None] * j).max()


def test_double_matches_long_double_brute_force():
    x, v, m = _rand_system(4, 5)
    a, j = oracle.acc_jerk(x, v, m)
    al, jl = oracle.acc_jerk(x, v, m, prec=oracle.LONG_DOUBLE)
    np.testing.assert_allclose(a, al, rtol=1e-14)
    np.testing.assert_allclose(j, jl, rtol=0, atol=1e-14 * np.abs(jl).max())


# ------------------------------------------------------------------------------------------ whole step
def test_circular_orbit_returns_after_one_period():
    x, v, m = two_body(e=0.0)
    T = 2 * math.pi / math.sqrt(m.sum())
    errs = []
    for N in (100, 200, 400):
        x1, v1, _ = run1(x, v, m, T / N, N)
        errs.append(np.abs(x1 - x).max())
    assert errs[0] < 1e-6
    assert 15.0 < errs[0] / errs[1] < 17.0 and 15.0 < errs[1] / errs[2] < 17.0, errs


def test_fourth_order_convergence_eccentric():
    # N = 400/800/1600 steps per period at e = 0.3 -> 1.93e-7, 1.20e-8, 7.52e-10 (ratios 16.00);
    # the literal 3/10 of P:L85 gives ratio 4, the literal x_k / v_0 bases give 8 / divergence (R3-R5).
    x, v, m = two_body(e=0.3)
    T = 2 * math.pi / math.sqrt(m.sum())
    errs = []
    for N in (400, 800, 1600):
        x1, v1, _ = run1(x, v, m, T / N, N)
        errs.append(max(np.abs(x1 - x).max(), np.abs(v1 - v).max()))
    assert 1e-7 < errs[0] < 4e-7, errs
    assert 15.7 < errs[0] / errs[1] < 16.3 and 15.7 < errs[1] / errs[2] < 16.3, errs


def test_eccentric_orbit_matches_keplers_equation_at_arbitrary_time():
    # position at t = 0.37 T from E - e sin E = M (solved independently in workloads.elements_to_cartesian)
    e, M0 = 0.3, 0.4
    x, v, m = two_body(e=e, M=M0)
    nmean = math.sqrt(m.sum())
    t = 0.37 * 2 * math.pi / nmean
    N = 4000
    x1, v1, r = run1(x, v, m, t / N, N)
    xe, ve, _ = two_body(e=e, M=M0 + nmean * t)
    assert abs(r["time"][0] - t) < 1e-12
    np.testing.assert_allclose(x1, xe, rtol=0, atol=2e-11)
    np.testing.assert_allclose(v1, ve, rtol=0, atol=2e-11)


def test_converged_corrector_is_the_time_symmetric_pair():
    # R5b: with R3-R5 the fixed point of Eq. 4 satisfies the symmetric implicit relations
    #   v1 = v0 + (a0+a1) h/2 + (j0-j1) h^2/12,  x1 = x0 + (v0+v1) h/2 + (a0-a1) h^2/10 + (j0+j1) h^3/120,
    # both invariant under 0<->1, h -> -h.  A wrong coefficient in Eq. 3 or Eq. 4 breaks one of them.
    pos, vel, mass = W.generate(0, n_sys=3)
    h = 0.02
    for s in range(3):
        x0, v0, m = pos[s], vel[s], mass[s]
        x1, v1 = oracle.hermite_step(x0, v0, m, h, n_corr=30, prec=oracle.LONG_DOUBLE)
        a0, j0 = oracle.acc_jerk(x0, v0, m, prec=oracle.LONG_DOUBLE)
        a1, j1 = oracle.acc_jerk(x1, v1, m, prec=oracle.LONG_DOUBLE)
        vs = v0 + 0.5 * (a0 + a1) * h + (j0 - j1) * h * h / 12.0
        xs = x0 + 0.5 * (v0 + v1) * h + (a0 - a1) * h * h / 10.0 + (j0 + j1) * h**3 / 120.0
        np.testing.assert_allclose(v1, vs, rtol=0, atol=5e-16)
        np.testing.assert_allclose(x1, xs, rtol=0, atol=5e-16)
        # and two iterations (the method) are already close to that fixed point
        x2, v2 = oracle.hermite_step(x0, v0, m, h, n_corr=2)
        assert np.abs(x2 - x1).max() < 1e-12 and np.abs(v2 - v1).max() < 1e-10


def test_forward_then_backward_recovers_initial_state():
    # time symmetry: reversal defect is far below the forward truncation error (App. B: 6.6e-13 vs 1.9e-7)
    x, v, m = two_body(e=0.3)
    T = 2 * math.pi / math.sqrt(m.sum())
    N = 400
    x1, v1, _ = run1(x, v, m, T / N, N)
    fwd_err = np.abs(x1 - x).max()
    x2, v2, r = run1(x1, v1, m, -T / N, N, time=np.array([T]), t_end=-np.inf)
    defect = max(np.abs(x2 - x).max(), np.abs(v2 - v).max())
    assert fwd_err > 1e-7 and defect < 1e-11, (fwd_err, defect)
    assert abs(r["time"][0]) < 1e-12 and r["nsteps"][0] == N


def test_energy_and_angular_momentum_drift_config0():
    pos, vel, mass = W.generate(0, n_sys=32)
    E0, L0 = oracle.energy(pos, vel, mass)
    r = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, max_steps=2000)
    E1, L1 = oracle.energy(r["pos"], r["vel"], mass)
    assert np.abs(E1 / E0 - 1).max() < 2e-9       # App. B: median 5.6e-12, max 2.8e-10 over 1024 systems
    assert np.median(np.abs(E1 / E0 - 1)) < 1e-10
    # Hermite is not symplectic: L drifts at truncation order (like E), far below the state error
    assert (np.abs(L1 - L0).max(axis=1) / np.linalg.norm(L0, axis=1)).max() < 1e-9
    # linear momentum stays zero (barycentric input)
    P1 = (mass[:, :, None] * r["vel"]).sum(1)
    assert np.abs(P1).max() < 1e-17


def test_paper_validation_run_double_vs_long_double():
    # CPU vs GPU Hermite agree to 1e-10 in |x|, |v| per body and in t over 10 pi, ICs of P:L298,
    # n = 3..6.  Here the two arithmetic widths of the oracle stand in for the two machines (noise floor).
    for n in (3, 4, 5, 6):
        pos, vel, mass = W.paper_ics(n)
        steps = int(round(10 * math.pi / 1e-3))
        a = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=1e-3, max_steps=steps)
        b = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=1e-3, max_steps=steps, prec=oracle.LONG_DOUBLE)
        assert np.abs(np.linalg.norm(a["pos"], axis=2) - np.linalg.norm(b["pos"], axis=2)).max() < 1e-10
        assert np.abs(np.linalg.norm(a["vel"], axis=2) - np.linalg.norm(b["vel"], axis=2)).max() < 1e-10
        assert abs(a["time"][0] - b["time"][0]) < 1e-10
        # circular orbits stay circular to O(planet mass) (R15)
        rad = np.linalg.norm(a["pos"][0, 1] - a["pos"][0, 0])
        assert abs(rad - 1.0) < 0.02


# ------------------------------------------------------------------------------------------ energy
def test_energy_two_body_closed_form():
    # E = -m0 m1 / (2a), |L| = m0 m1 sqrt(a (1-e^2) / (m0+m1))  (R9: pairs counted once)
    a, e, m0, m1 = 1.7, 0.4, 1.0, 0.01
    x, v, m = two_body(e=e, a=a, m0=m0, m1=m1, M=1.1)
    E, L = oracle.energy(x[None], v[None], m[None])
    assert abs(E[0] + m0 * m1 / (2 * a)) < 1e-15
    assert abs(np.linalg.norm(L[0]) - m0 * m1 * math.sqrt(a * (1 - e * e) / (m0 + m1))) < 1e-15


# ------------------------------------------------------------------------------------------ Alg. 1 loop
def _linear_pair(sep0, speed):
    """Two (almost) massless bodies approaching head-on along x plus a far, (almost) massless 'star'."""
    x = np.array([[0.0, 50.0, 0.0], [-sep0 / 2, 0.0, 0.0], [sep0 / 2, 0.0, 0.0]])
    v = np.array([[0.0, 0.0, 0.0], [speed / 2, 0.0, 0.0], [-speed / 2, 0.0, 0.0]])
    m = np.array([1e-30, 1e-30, 1e-30])
    return x, v, m


def test_close_approach_monitor_fires_at_the_predicted_step():
    # straight-line motion: separation after k steps = 1 - k * 0.01 * 1; first k with sep < 0.0995 is k = 91
    x, v, m = _linear_pair(1.0, 1.0)
    x1, v1, r = run1(x, v, m, 0.01, 1000, r_close=0.0995, r_eject=100.0)
    assert r["status"][0] == oracle.STOP_CLOSE and r["nsteps"][0] == 91
    assert abs((x1[2, 0] - x1[1, 0]) - (1.0 - 0.91)) < 1e-12   # keeps the post-step state
    assert abs(r["time"][0] - 0.91) < 1e-12
    # sticky: a second call does nothing
    r2 = oracle.integrate(oracle.HERMITE, r["pos"], r["vel"], m[None], r["time"], dt=0.01, max_steps=10,
                          status=r["status"], nsteps=r["nsteps"], r_close=0.0995)
    assert r2["status"][0] == oracle.STOP_CLOSE and r2["nsteps"][0] == 91 and np.array_equal(r2["pos"], r["pos"])
    # disabled monitor: runs through
    _, _, r3 = run1(x, v, m, 0.01, 95)
    assert r3["status"][0] == oracle.DONE_STEPS and r3["nsteps"][0] == 95


def test_ejection_monitor_fires_at_the_predicted_step():
    # body 1 leaves along +x at speed 2 from x = 1: |x| > 10.05 first after k = 453 steps of 0.01 (1 + 0.02 k > 10.05)
    x = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [0.0, -3.0, 0.0]])
    v = np.array([[0.0, 0.0, 0.0], [2.0, 0.0, 0.0], [0.0, 0.0, 0.0]])
    m = np.array([1e-30, 1e-30, 1e-30])
    _, _, r = run1(x, v, m, 0.01, 1000, r_close=0.01, r_eject=10.05)
    assert r["status"][0] == oracle.STOP_EJECT and r["nsteps"][0] == 453
    # close approach is tested before ejection when both hold after the same step
    x2, v2, m2 = _linear_pair(1.0, 1.0)
    x2[0] = [0.0, 50.0, 0.0]
    _, _, r2 = run1(x2, v2, m2, 0.01, 1000, r_close=0.0995, r_eject=40.0)
    assert r2["status"][0] == oracle.STOP_EJECT and r2["nsteps"][0] == 1  # star is already outside 40 after step 1
    _, _, r3 = run1(x2, v2, m2, 0.01, 1000, r_close=2.0, r_eject=40.0)
    assert r3["status"][0] == oracle.STOP_CLOSE and r3["nsteps"][0] == 1


def test_nonfinite_state_stops():
    x = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0]])
    v = np.zeros((2, 3))
    m = np.array([1.0, 1.0])
    x[1] = x[0]  # coincident bodies: r = 0 -> inf/nan after the first evaluation
    _, _, r = run1(x, v, m, 0.01, 10)
    assert r["status"][0] == oracle.STOP_NONFINITE and r["nsteps"][0] == 1


def test_loop_stop_conditions_and_status():
    pos, vel, mass = W.generate(0, n_sys=4)
    # time stop: t >= t_end, no clipping of the last step (R10)
    r = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, t_end=0.055, max_steps=100)
    assert (r["status"] == oracle.DONE_TIME).all() and (r["nsteps"] == 6).all()
    assert np.allclose(r["time"], 0.06, atol=1e-15)
    # both limits reached by the same step: time wins
    r = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, t_end=0.055, max_steps=6)
    assert (r["status"] == oracle.DONE_TIME).all()
    # zero steps
    r = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, max_steps=0)
    assert (r["status"] == oracle.DONE_STEPS).all() and np.array_equal(r["pos"], pos)
    with pytest.raises(ValueError):
        oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.0, max_steps=1)


def test_split_run_is_bit_identical():
    # R6: (a0, j0) are re-evaluated at the start of every step, so the step is a pure function of (x, v, m)
    pos, vel, mass = W.generate(0, n_sys=8)
    full = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, max_steps=300)
    h1 = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, max_steps=100)
    h2 = oracle.integrate(oracle.HERMITE, h1["pos"], h1["vel"], mass, h1["time"], dt=0.01, max_steps=200,
                          status=h1["status"], nsteps=h1["nsteps"])
    assert np.array_equal(full["pos"], h2["pos"]) and np.array_equal(full["vel"], h2["vel"])
    assert np.array_equal(full["time"], h2["time"]) and (h2["nsteps"] == 300).all()


def test_thread_count_does_not_change_results():
    pos, vel, mass = W.generate(2, n_sys=16)
    a = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.005, max_steps=50, nthreads=1)
    b = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.005, max_steps=50, nthreads=4)
    assert np.array_equal(a["pos"], b["pos"]) and np.array_equal(a["vel"], b["vel"])
