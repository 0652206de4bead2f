"""GPU parity of the fixed-step Runge-Kutta Cash-Karp kernel (ENS_RKCK; reading R-RK1) against
the CPU oracle, through the C ABI."""
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


def test_config0_systems_full_parity():
    c = W.CONFIGS[0]
    pos, vel, mass = W.generate(0)
    g = ens.run(ens.RKCK, pos, vel, mass, dt=c.dt, steps=c.steps, want_energy=True)
    o = oracle.integrate(oracle.RKCK, pos, vel, mass, dt=c.dt, max_steps=c.steps)
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all() and (g["time"] == o["time"]).all()
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    assert dp.max() <= 1e-10 and dv.max() <= 1e-10, (dp.max(), dv.max())
    assert np.abs((g["E"] - g["E0"]) / g["E0"]).max() < 1e-9


@pytest.mark.parametrize("n_body", list(range(2, 17)))
def test_every_body_count_ragged_with_monitors(n_body):
    n_sys = 77
    pos, vel, mass = _systems(n_sys, n_body, 900 + n_body)
    if n_body >= 3:
        pos[5, n_body - 1] = pos[5, n_body - 2] + np.array([0.05, 0.0, 0.0])
        vel[5, n_body - 1] = vel[5, n_body - 2] + np.array([-0.5, 0.0, 0.0])
    kw = dict(dt=0.002, r_close=0.02, r_eject=5000.0)
    g = ens.run(ens.RKCK, pos, vel, mass, steps=150, **kw)
    o = oracle.integrate(oracle.RKCK, pos, vel, mass, max_steps=150, **kw)
    if n_body >= 3:
        assert o["status"][5] == oracle.STOP_CLOSE and 0 < o["nsteps"][5] < 150
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all()
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    assert dp.max() <= 1e-11 and dv.max() <= 1e-11, (dp.max(), dv.max())


def test_fifth_order_on_the_gpu_against_keplers_equation():
    """Closed form on the GPU itself: error ratio ~32 on halving the step (a wrong tableau entry in the kernel's
    precomputed products would lower the order)."""
    e, M0 = 0.3, 0.4
    x, v, m = two_body(e=e, M=M0)
    nm = math.sqrt(m.sum())
    t = 0.37 * 2 * math.pi / nm
    xe, ve, _ = two_body(e=e, M=M0 + nm * t)
    errs = []
    for N in (50, 100, 200):
        g = ens.run(ens.RKCK, x[None], v[None], m[None], dt=t / N, steps=N)
        errs.append(max(np.abs(g["pos"][0] - xe).max(), np.abs(g["vel"][0] - ve).max()))
    assert 26.0 < errs[0] / errs[1] < 38.0 and 26.0 < errs[1] / errs[2] < 38.0, errs


def test_full_size_config1_sampled_parity_split_runs_and_reversal():
    c = W.CONFIGS[1]
    pos, vel, mass = W.generate(1)
    with ens.Ensemble(c.n_sys, c.n_body) as e:
        e.set_state(pos, vel, mass)
        e.set_monitors(c.r_close, c.r_eject)
        e.integrate(ens.RKCK, c.dt, 1500)
        g = e.get_state()
    idx = np.arange(0, c.n_sys, 1024)
    o = oracle.integrate(oracle.RKCK, pos[idx], vel[idx], mass[idx], dt=c.dt, max_steps=1500, r_close=c.r_close,
                         r_eject=c.r_eject)
    assert (g["status"][idx] == o["status"]).all() and (g["nsteps"][idx] == o["nsteps"]).all()
    assert rel_diff(g["pos"][idx], o["pos"]).max() <= 1e-10
    p, v, m = pos[:200], vel[:200], mass[:200]
    a = ens.run(ens.RKCK, p, v, m, dt=c.dt, steps=400)
    with ens.Ensemble(200, 3) as e:
        e.set_state(p, v, m)
        e.integrate(ens.RKCK, c.dt, 150)
        e.integrate(ens.RKCK, c.dt, 250)
        b = e.get_state()
        assert (a["pos"] == b["pos"]).all() and (a["vel"] == b["vel"]).all()  # the step is a pure function of the state
        e.integrate(ens.RKCK, -c.dt, 400, t_end=-np.inf)
        r = e.get_state()
    assert np.abs(r["time"]).max() < 1e-12 and rel_diff(r["pos"], p).max() < 1e-9  # RK is not reversible, only accurate
