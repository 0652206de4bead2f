"""GPU parity of the MVS kernel with merged half sub-steps (ENS_MVS_MERGED)
against the oracle's merged map, and the measured distance of both from the unmerged map (the optimisation's parity
cost).  Tolerances as for ENS_MVS (R-noise)."""
import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W
from parity import rel_diff
from test_gpu_mvs import _systems

pytestmark = pytest.mark.gpu


def test_config4_1000_steps_max_parity_and_parity_cost():
    c = W.CONFIGS[4]
    pos, vel, mass = W.generate(4, n_sys=1024)
    g = ens.run(ens.MVS_MERGED, pos, vel, mass, dt=c.dt, steps=1000, want_energy=True)
    o = oracle.integrate(oracle.MVS_MERGED, pos, vel, mass, dt=c.dt, max_steps=1000)
    u = oracle.integrate(oracle.MVS, pos, vel, mass, dt=c.dt, max_steps=1000)
    assert (g["status"] == ens.DONE_STEPS).all() and (g["nsteps"] == 1000).all() and (g["time"] == o["time"]).all()
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    cp, cv = rel_diff(g["pos"], u["pos"]), rel_diff(g["vel"], u["vel"])
    print(f"merged cfg4 x1000: gpu vs merged oracle pos max {dp.max():.2e} vel max {dv.max():.2e}; "
          f"gpu merged vs UNMERGED oracle (parity cost) pos max {cp.max():.2e} vel max {cv.max():.2e}")
    assert dp.max() <= 1e-10 and dv.max() <= 1e-10
    assert cp.max() <= 1e-10 and cv.max() <= 1e-10
    dL = np.abs(g["L"] - g["L0"]).max(axis=1) / np.linalg.norm(g["L0"], axis=1)
    assert dL.max() <= 1e-11


@pytest.mark.parametrize("n_body", list(range(2, 17)))
def test_every_body_count_ragged(n_body):
    n_sys = 205
    pos, vel, mass = _systems(n_sys, n_body, 300 + n_body)
    g = ens.run(ens.MVS_MERGED, pos, vel, mass, dt=0.02, steps=300)
    o = oracle.integrate(oracle.MVS_MERGED, pos, vel, mass, dt=0.02, max_steps=300)
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all()
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    assert dp.max() <= 1e-11 and dv.max() <= 1e-11, (dp.max(), dv.max())


def test_single_step_equals_the_unmerged_kernel_and_monitors_time_limit_split_runs():
    pos, vel, mass = W.generate(4, n_sys=300)
    a = ens.run(ens.MVS, pos, vel, mass, dt=0.05, steps=1)
    b = ens.run(ens.MVS_MERGED, pos, vel, mass, dt=0.05, steps=1)
    assert rel_diff(a["pos"], b["pos"]).max() <= 2e-16 and rel_diff(a["vel"], b["vel"]).max() <= 4e-16
    z = ens.run(ens.MVS_MERGED, pos, vel, mass, dt=0.05, steps=0)
    assert rel_diff(z["pos"], pos).max() <= 4e-16 and (z["nsteps"] == 0).all()  # the coordinate round trip only
    # hand-built close approach, ejection threshold and a time limit: same decisions as the oracle's merged map
    d = np.array([0.05, 0.003, 0.0])
    for s in range(0, 300, 3):
        pos[s, 2] = pos[s, 1] + d * (1 + 0.01 * (s % 7))
        vel[s, 2] = vel[s, 1] - 0.4 * d / np.linalg.norm(d)
    time = np.linspace(0.0, 0.3, 300)
    kw = dict(dt=0.002, r_close=0.02, r_eject=30.0, t_end=1.0)
    o = oracle.integrate(oracle.MVS_MERGED, pos, vel, mass, time, max_steps=3000, **kw)
    with ens.Ensemble(300, 4) as e:
        e.set_state(pos, vel, mass, time)
        e.set_monitors(0.02, 30.0)
        e.integrate(ens.MVS_MERGED, 0.002, 3000, 1.0)
        g = e.get_state()
        assert (o["status"] == oracle.STOP_CLOSE).sum() >= 80 and (o["status"] == oracle.DONE_TIME).sum() >= 100
        assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all() and (g["time"] == o["time"]).all()
        assert rel_diff(g["pos"], o["pos"]).max() <= 1e-10 and rel_diff(g["vel"], o["vel"]).max() <= 1e-10
        # second call: stopped systems stay, the others re-open the half sub-steps and go on
        e.integrate(ens.MVS_MERGED, 0.002, 50)
        g2 = e.get_state()
    o2 = oracle.integrate(oracle.MVS_MERGED, o["pos"], o["vel"], mass, o["time"], dt=0.002, max_steps=50, r_close=0.02,
                          r_eject=30.0, status=o["status"], nsteps=o["nsteps"])
    assert (g2["status"] == o2["status"]).all() and (g2["nsteps"] == o2["nsteps"]).all()
    assert rel_diff(g2["pos"], o2["pos"]).max() <= 1e-10


def test_config4_full_size_sampled_parity():
    """Config 4 at FULL size in the launch configuration bench.py times, per system against its own noise floor."""
    c = W.CONFIGS[4]
    pos, vel, mass = W.generate(4)
    g = ens.run(ens.MVS_MERGED, pos, vel, mass, dt=c.dt, steps=c.steps)
    idx = np.unique(np.concatenate([np.arange(0, c.n_sys, c.n_sys // 128), [c.n_sys - 1]]))
    o = oracle.integrate(oracle.MVS_MERGED, pos[idx], vel[idx], mass[idx], dt=c.dt, max_steps=c.steps)
    ol = oracle.integrate(oracle.MVS_MERGED, pos[idx], vel[idx], mass[idx], dt=c.dt, max_steps=c.steps, prec=oracle.LONG_DOUBLE)
    assert (g["status"] == ens.DONE_STEPS).all() and (g["nsteps"] == c.steps).all()
    dp, dv = rel_diff(g["pos"][idx], o["pos"]), rel_diff(g["vel"][idx], o["vel"])
    fp, fv = rel_diff(o["pos"], ol["pos"]), rel_diff(o["vel"], ol["vel"])
    print(f"merged cfg4 x{c.steps}: gpu-vs-oracle pos median {np.median(dp):.2e} max {dp.max():.2e}; floor median "
          f"{np.median(fp):.2e} max {fp.max():.2e}")
    assert (dp <= np.maximum(1e-10, 10 * fp)).all() and (dv <= np.maximum(1e-10, 10 * fv)).all()
    assert np.median(dp) <= 1e-10 and np.median(dv) <= 1e-10
