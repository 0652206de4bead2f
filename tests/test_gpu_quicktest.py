"""The step loops' quick go-test (one test on high words per step; the exact monitor / stop logic only behind a rarely
taken branch) must never change a decision: cases built to sit on both sides of every filter of that test, for every
step-loop kernel, compared with the oracle (status, stop step, time exact: R11, R12; state at rounding level)."""
import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W
from parity import rel_diff

pytestmark = pytest.mark.gpu

INTEGRATORS = [("hermite", ens.HERMITE, oracle.HERMITE, 0.01), ("carry", ens.HERMITE_CARRY, oracle.HERMITE_CARRY, 0.01),
               ("rkck", ens.RKCK, oracle.RKCK, 0.01), ("mvs", ens.MVS, oracle.MVS, 0.02),
               ("mvs_merged", ens.MVS_MERGED, oracle.MVS_MERGED, 0.02), ("adaptive", ens.HERMITE_ADAPTIVE, oracle.HERMITE_ADAPTIVE, 0.02),
               ("rkck_adaptive", ens.RKCK_ADAPTIVE, oracle.RKCK_ADAPTIVE, 0.05)]


def _compare(name, gi, oi, pos, vel, mass, dt, steps, tol=1e-10, **kw):
    g = ens.run(gi, pos, vel, mass, dt=dt, steps=steps, rk_eps=1e-9, **kw)
    o = oracle.integrate(oi, pos, vel, mass, dt=dt, max_steps=steps, rk_eps=1e-9, **kw)
    assert (g["status"] == o["status"]).all(), (name, np.nonzero(g["status"] != o["status"])[0][:5], g["status"][:8], o["status"][:8])
    assert (g["nsteps"] == o["nsteps"]).all(), (name, g["nsteps"][:8], o["nsteps"][:8])
    if name != "rkck_adaptive":  # (its times agree whenever its step sequences do: tests/test_gpu_rkck_adaptive.py)
        assert np.abs(g["time"] - o["time"]).max() <= 1e-13 * max(1.0, np.abs(o["time"]).max()), name
        assert rel_diff(g["pos"], o["pos"]).max() <= tol and rel_diff(g["vel"], o["vel"]).max() <= tol, name
    return g, o


@pytest.mark.parametrize("name,gi,oi,dt", INTEGRATORS, ids=[i[0] for i in INTEGRATORS])
def test_outer_planet_between_the_coordinate_filter_and_r_eject(name, gi, oi, dt):
    """r_eject chosen so that the outer planet's largest coordinate exceeds r_eject / sqrt(3) (the quick test fails on
    every step, the exact logic runs) while its distance from the origin stays below r_eject for the whole run: no
    system may stop; and with r_eject just inside the orbit every system must stop at the oracle's step."""
    pos, vel, mass = W.generate(0, n_sys=257)
    a2 = np.linalg.norm(pos[:, 2], axis=1)
    for r_eject, expect_stop in ((1.15 * a2.max(), False), (float(np.median(a2)), True)):
        g, o = _compare(name, gi, oi, pos, vel, mass, dt, 300, r_eject=r_eject)
        if expect_stop:
            assert (o["status"] == oracle.STOP_EJECT).sum() >= 100
        else:
            assert (o["status"] == oracle.DONE_STEPS).all()


@pytest.mark.parametrize("name,gi,oi,dt", INTEGRATORS, ids=[i[0] for i in INTEGRATORS])
def test_extreme_thresholds(name, gi, oi, dt):
    """Degenerate thresholds: r_eject below every orbit (all systems ejected by the first monitor call), a denormal
    r_eject, r_close above every separation (all systems stop on a close approach at step 1), and a t_end already
    reached (no step at all)."""
    pos, vel, mass = W.generate(0, n_sys=130)
    for kw in (dict(r_eject=0.3), dict(r_eject=1e-310), dict(r_close=50.0), dict(r_close=50.0, r_eject=0.3)):
        g, o = _compare(name, gi, oi, pos, vel, mass, dt, 50, **kw)
        assert (o["nsteps"] == 1).all() and (o["status"] >= oracle.STOP_CLOSE).all(), kw
    g, o = _compare(name, gi, oi, pos, vel, mass, dt, 50, t_end=0.0)
    assert (g["nsteps"] == 0).all() and (g["status"] == ens.DONE_TIME).all()
    g, o = _compare(name, gi, oi, pos, vel, mass, -dt, 50, t_end=0.0)  # backward from t = 0 with t_end = 0: no step either
    assert (g["nsteps"] == 0).all() and (g["status"] == ens.DONE_TIME).all()


@pytest.mark.parametrize("name,gi,oi,dt", INTEGRATORS[:5], ids=[i[0] for i in INTEGRATORS[:5]])
def test_backward_run_stops_on_time_at_the_oracles_step(name, gi, oi, dt):
    """dt < 0 with a finite t_end and staggered start times: the folded time variable (ts = -t) must give the oracle's
    step counts and end times exactly."""
    pos, vel, mass = W.generate(0, n_sys=200)
    t0 = np.linspace(-0.5, 0.7, 200)
    for sign, t_end in ((-1.0, -1.234), (1.0, 1.7)):
        g = ens.run(gi, pos, vel, mass, dt=sign * dt, steps=10 ** 6, t_end=t_end, time=t0)
        o = oracle.integrate(oi, pos, vel, mass, dt=sign * dt, max_steps=10 ** 6, t_end=t_end, time=t0)
        assert (g["status"] == o["status"]).all() and (o["status"] == oracle.DONE_TIME).all()
        assert (g["nsteps"] == o["nsteps"]).all() and len(np.unique(o["nsteps"])) > 10
        assert (g["time"] == o["time"]).all()
        assert rel_diff(g["pos"], o["pos"]).max() <= 1e-11


def test_mvs_planet_close_to_the_star_and_far_from_it():
    """MVS quick test: a planet whose heliocentric coordinates are all below r_close while its distance is above it
    (the filter fails, the exact test must not fire), and one that does come within r_close of the star."""
    pos, vel, mass = W.generate(4, n_sys=300)
    q = np.linalg.norm(pos[:, 1] - pos[:, 0], axis=1)  # innermost planet, 0.5 .. 1.0
    for r_close in (0.62 * q.min(), 1.02 * float(np.median(q))):
        g, o = _compare("mvs", ens.MVS, oracle.MVS, pos, vel, mass, 0.05, 200, r_close=r_close)
        gm, om = _compare("mvs_merged", ens.MVS_MERGED, oracle.MVS_MERGED, pos, vel, mass, 0.05, 200, r_close=r_close)
    assert (o["status"] == oracle.STOP_CLOSE).sum() >= 100 and (o["status"] == oracle.DONE_STEPS).sum() >= 5
