"""GPU parity of the adaptive-step Hermite kernel (Eq. 5; ENS_HERMITE_ADAPTIVE) against the CPU oracle,
through the C ABI.  `dt` is the step size scale tau; every system takes its own steps."""
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


def _run(pos, vel, mass, tau, steps, t_end=np.inf, r_close=0.0, r_eject=np.inf, time=None):
    n_sys, n_body = mass.shape
    with ens.Ensemble(n_sys, n_body) as e:
        e.set_state(pos, vel, mass, time)
        e.set_monitors(r_close, r_eject)
        e.integrate(ens.HERMITE_ADAPTIVE, tau, steps, t_end)
        g = e.get_state()
        g["info"] = e.info()
    return g


def test_step_count_control_matches_oracle():
    """1000 config-0 systems (ragged), 300 adaptive steps each: the times reached (sums of 300 different steps per
    system) and the states agree with the oracle at rounding level."""
    pos, vel, mass = W.generate(0, n_sys=1000)
    g = _run(pos, vel, mass, 0.02, 300)
    o = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.02, max_steps=300)
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == 300).all()
    assert np.abs(g["time"] / o["time"] - 1.0).max() <= 1e-13
    assert o["time"].std() > 0.05  # systems really are at different times
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    assert dp.max() <= 1e-11 and dv.max() <= 1e-11, (dp.max(), dv.max())


def test_time_control_same_step_counts_as_oracle():
    """Run to t_end: systems finish after different numbers of steps (retirement, S§8 a7); step counts match the oracle
    except where the oracle's last time is within rounding of t_end (R12), and none such exists here."""
    pos, vel, mass = W.generate(1, n_sys=2048 + 37)
    g = _run(pos, vel, mass, 0.03, 10**6, t_end=12.0, r_close=0.01, r_eject=100.0)
    o = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.03, max_steps=10**6, t_end=12.0, r_close=0.01,
                         r_eject=100.0)
    assert (o["status"] == oracle.DONE_TIME).all() and len(np.unique(o["nsteps"])) > 20
    knife = np.abs(o["time"] - 12.0) < 1e-9
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"])[~knife].all()
    ok = ~knife
    assert np.abs(g["time"][ok] - o["time"][ok]).max() <= 1e-11
    assert rel_diff(g["pos"], o["pos"])[ok].max() <= 1e-10 and rel_diff(g["vel"], o["vel"])[ok].max() <= 1e-10


@pytest.mark.parametrize("n_body", list(range(2, 17)))
def test_every_body_count_ragged(n_body):
    """Every (L, B) shape, exact and padded (dummy slots must not enter Eq. 5's sum), ragged ensemble."""
    n_sys = 77
    pos, vel, mass = _systems(n_sys, n_body, 500 + n_body)
    g = _run(pos, vel, mass, 0.01, 120)
    o = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.01, max_steps=120)
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all()
    assert np.abs(g["time"] / o["time"] - 1.0).max() <= 1e-13
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    assert dp.max() <= 1e-11 and dv.max() <= 1e-11, (dp.max(), dv.max())


def test_eccentric_two_body_against_keplers_equation():
    """Closed form on the GPU itself: e = 0.9 over one period with tau = 0.01, compared with the exact Kepler solution at
    the time each system actually reached; and the first step against dt = tau / (w sqrt 2) at pericentre."""
    e = 0.9
    xs, vs, ms = zip(*(two_body(e=e, M=M) for M in np.linspace(0.0, 2 * math.pi, 40, endpoint=False)))
    pos, vel, mass = np.array(xs), np.array(vs), np.array(ms)
    g = _run(pos, vel, mass, 0.01, 10**6, t_end=2 * math.pi)
    for s, M in enumerate(np.linspace(0.0, 2 * math.pi, 40, endpoint=False)):
        nm = math.sqrt(mass[s].sum())
        xe, ve, _ = two_body(e=e, M=M + nm * g["time"][s])
        assert np.abs(g["pos"][s] - xe).max() < 2e-7 and np.abs(g["vel"][s] - ve).max() < 2e-6
    one = _run(pos[:1], vel[:1], mass[:1], 0.01, 1)
    w = math.sqrt(mass[0].sum() * (1 - e * e)) / (1 - e) ** 2
    assert abs(one["time"][0] * w * math.sqrt(2.0) / 0.01 - 1.0) < 1e-9


def test_monitors_split_runs_and_direction():
    pos, vel, mass = W.generate(0, n_sys=130)
    pos[7, 2] = pos[7, 1] + np.array([0.05, 0.0, 0.0])
    vel[7, 2] = vel[7, 1] + np.array([-0.5, 0.0, 0.0])
    kw = dict(r_close=0.02, r_eject=100.0)
    g = _run(pos, vel, mass, 0.02, 10**5, t_end=5.0, **kw)
    o = oracle.integrate(oracle.HERMITE_ADAPTIVE, pos, vel, mass, dt=0.02, max_steps=10**5, t_end=5.0, **kw)
    assert o["status"][7] == oracle.STOP_CLOSE
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all()
    assert rel_diff(g["pos"], o["pos"]).max() <= 1e-10
    # split runs are bit-identical, and a negative tau walks time down
    with ens.Ensemble(130, 3) as e:
        e.set_state(pos, vel, mass)
        e.integrate(ens.HERMITE_ADAPTIVE, 0.02, 40)
        a = e.get_state()
        e.set_state(pos, vel, mass)
        e.integrate(ens.HERMITE_ADAPTIVE, 0.02, 15)
        e.integrate(ens.HERMITE_ADAPTIVE, 0.02, 25)
        b = e.get_state()
        assert (a["pos"] == b["pos"]).all() and (a["time"] == b["time"]).all() and (b["nsteps"] == 40).all()
        e.integrate(ens.HERMITE_ADAPTIVE, -0.02, 10**6, t_end=0.0)
        c = e.get_state()
        assert (c["status"] == ens.DONE_TIME).all() and (c["time"] <= 0.0).all() and (c["time"] > -0.1).all()


def test_results_do_not_depend_on_the_hand_out_order_and_stops_are_sticky():
    """The longest-first hand-out (adaptive_order.cu) only schedules: with it switched off every system ends in the
    bit-identical state.  A system stopped by a monitor is not touched by a second call (it is pulled, found stopped,
    and retired without a write-back)."""
    pos, vel, mass = W.generate(1, n_sys=3000)
    pos[11, 2] = pos[11, 1] + np.array([0.05, 0.0, 0.0])
    vel[11, 2] = vel[11, 1] + np.array([-0.5, 0.0, 0.0])
    runs = []
    for unordered in (False, True):
        with ens.Ensemble(3000, 3) as e:
            e.set_option(ens.OPT_ADAPTIVE_UNORDERED, int(unordered))
            e.set_state(pos, vel, mass)
            e.set_monitors(0.02, 100.0)
            e.integrate(ens.HERMITE_ADAPTIVE, 0.03, 10**6, 6.0)
            a = e.get_state()
            e.integrate(ens.HERMITE_ADAPTIVE, 0.03, 50)
            b = e.get_state()
        assert a["status"][11] == ens.STOP_CLOSE and b["status"][11] == ens.STOP_CLOSE
        assert (b["pos"][11] == a["pos"][11]).all() and b["nsteps"][11] == a["nsteps"][11] and b["time"][11] == a["time"][11]
        others = np.arange(3000) != 11
        assert (b["nsteps"][others] == a["nsteps"][others] + 50).all() and (b["status"][others] == ens.DONE_STEPS).all()
        runs.append((a, b))
    for x, y in zip(runs[0], runs[1]):
        for key in ("pos", "vel", "time", "status", "nsteps"):
            assert (x[key] == y[key]).all(), key
