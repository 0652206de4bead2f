"""GPU parity of the 2-evaluations-per-step Hermite kernel (ENS_HERMITE_CARRY: Alg. 2 as printed, a and j
carried from step to step; reading R6-alt) against the CPU oracle, through the C ABI."""
import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W
from parity import rel_diff
from test_gpu_mvs import _systems

pytestmark = pytest.mark.gpu


def test_config0_parity_and_distance_from_the_three_evaluation_kernel():
    c = W.CONFIGS[0]
    pos, vel, mass = W.generate(0)
    g = ens.run(ens.HERMITE_CARRY, pos, vel, mass, dt=c.dt, steps=c.steps, want_energy=True)
    o = oracle.integrate(oracle.HERMITE_CARRY, pos, vel, mass, dt=c.dt, max_steps=c.steps)
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all() and (g["time"] == o["time"]).all()
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    assert dp.max() <= 1e-10 and dv.max() <= 1e-10, (dp.max(), dv.max())
    g3 = ens.run(ens.HERMITE, pos, vel, mass, dt=c.dt, steps=c.steps)
    d3 = rel_diff(g["pos"], g3["pos"])
    assert 0 < d3.max() < 5e-12  # a different (equally 4th-order) map, O(h^5) apart per step
    assert np.abs((g["E"] - g["E0"]) / g["E0"]).max() < 1e-9


@pytest.mark.parametrize("n_body", list(range(2, 17)))
def test_every_body_count_ragged_with_monitors(n_body):
    """Every (L, B) shape; the close-approach monitor works on positions of the post-step state (pair_r2min)."""
    n_sys = 77
    pos, vel, mass = _systems(n_sys, n_body, 700 + n_body)
    if n_body >= 3:
        pos[5, n_body - 1] = pos[5, n_body - 2] + np.array([0.05, 0.0, 0.0])  # last planet flies at its neighbour
        vel[5, n_body - 1] = vel[5, n_body - 2] + np.array([-0.5, 0.0, 0.0])
    kw = dict(dt=0.002, r_close=0.02, r_eject=5000.0)
    g = ens.run(ens.HERMITE_CARRY, pos, vel, mass, steps=150, **kw)
    o = oracle.integrate(oracle.HERMITE_CARRY, pos, vel, mass, max_steps=150, **kw)
    if n_body >= 3:
        assert o["status"][5] == oracle.STOP_CLOSE and 0 < o["nsteps"][5] < 150
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all()
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    assert dp.max() <= 1e-11 and dv.max() <= 1e-11, (dp.max(), dv.max())


def test_full_size_config1_sampled_parity_and_split_call_semantics():
    c = W.CONFIGS[1]
    pos, vel, mass = W.generate(1)
    with ens.Ensemble(c.n_sys, c.n_body) as e:
        e.set_state(pos, vel, mass)
        e.set_monitors(c.r_close, c.r_eject)
        e.integrate(ens.HERMITE_CARRY, c.dt, 3000)
        g = e.get_state()
    idx = np.arange(0, c.n_sys, 1024)
    o = oracle.integrate(oracle.HERMITE_CARRY, pos[idx], vel[idx], mass[idx], dt=c.dt, max_steps=3000, r_close=c.r_close,
                         r_eject=c.r_eject)
    assert (g["status"][idx] == o["status"]).all() and (g["nsteps"][idx] == o["nsteps"]).all()
    assert rel_diff(g["pos"][idx], o["pos"]).max() <= 1e-10
    # a second call re-evaluates (a0, j0) at its first state: close to, but not bit-identical with, one long call
    p, v, m = pos[:256], vel[:256], mass[:256]
    a = ens.run(ens.HERMITE_CARRY, p, v, m, dt=c.dt, steps=400)
    with ens.Ensemble(256, 3) as e:
        e.set_state(p, v, m)
        e.integrate(ens.HERMITE_CARRY, c.dt, 150)
        e.integrate(ens.HERMITE_CARRY, c.dt, 250)
        b = e.get_state()
    d = rel_diff(a["pos"], b["pos"])
    assert 0 < d.max() < 1e-12
