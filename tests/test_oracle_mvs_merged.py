"""Pins for the MVS map with merged sub-steps (oracle.MVS_MERGED; P:L105-109 five sub-steps, "the separation
between planets does not change during Cartesian drift and kick sub-steps").  In exact arithmetic
the merged run visits the same post-step states as the unmerged map (pinned in test_oracle_mvs.py), so the pins are:
one step is bit-identical; the same second-order convergence to the Hermite oracle; exact angular and linear momentum;
the same stop decisions; and the rounding-level distance between the two maps after 10^3 and 10^4 steps, which is the
"parity cost" of the optimisation, stated against the map's own double-vs-long-double noise floor."""
import numpy as np

import oracle
from paper_1208_1157_b200 import workloads as W


def _run(integ, pos, vel, mass, dt, steps, **kw):
    return oracle.integrate(integ, pos, vel, mass, dt=dt, max_steps=steps, **kw)


def _rel(a, b):
    return np.abs(a - b).max(axis=(1, 2)) / np.linalg.norm(b, axis=2).max(axis=1)


def test_a_single_step_is_bit_identical_to_the_unmerged_step():
    pos, vel, mass = W.generate(4, n_sys=16)
    a = _run(oracle.MVS, pos, vel, mass, 0.05, 1)
    b = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, 1)
    assert (a["pos"] == b["pos"]).all() and (a["vel"] == b["vel"]).all() and (a["time"] == b["time"]).all()
    # zero steps: state untouched
    z = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, 0)
    assert np.abs(z["pos"] - pos).max() < 1e-15 and (z["nsteps"] == 0).all()


def test_same_second_order_convergence_to_hermite():
    pos, vel, mass = W.generate(4, n_sys=4)
    T = 5.0
    ref = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=T / 20000, max_steps=20000, prec=oracle.LONG_DOUBLE)
    errs = np.array([np.abs(_run(oracle.MVS_MERGED, pos, vel, mass, T / N, N)["pos"] - ref["pos"]).max(axis=(1, 2))
                     for N in (250, 500, 1000, 2000)])
    assert (errs[0] < 5e-5).all() and (errs[0] > 1e-10).all()
    assert (np.abs(errs[:-1] / errs[1:] - 4.0) < 0.15).all(), errs[:-1] / errs[1:]


def test_invariants_are_exact_and_energy_error_bounded():
    pos, vel, mass = W.generate(4, n_sys=16)
    E0, L0 = oracle.energy(pos, vel, mass)
    r = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, 4000)
    E, L = oracle.energy(r["pos"], r["vel"], mass)
    assert (np.abs(L - L0).max(axis=1) / np.linalg.norm(L0, axis=1)).max() < 2e-13
    assert np.abs((mass[:, :, None] * r["vel"]).sum(1)).max() < 1e-17
    assert np.abs((mass[:, :, None] * r["pos"]).sum(1)).max() < 1e-14
    assert np.abs(E / E0 - 1).max() < 5e-6


def test_parity_cost_distance_from_the_unmerged_map():
    """The measured distance between the merged and the unmerged maps, against the unmerged map's own rounding floor
    (double vs 80-bit long double): the same order of magnitude at 10^3 and at 10^4 steps."""
    pos, vel, mass = W.generate(4, n_sys=64)
    for steps, bar in ((1000, 2e-11), (10000, None)):
        u = _run(oracle.MVS, pos, vel, mass, 0.05, steps)
        m = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, steps)
        ul = _run(oracle.MVS, pos, vel, mass, 0.05, steps, prec=oracle.LONG_DOUBLE)
        d, floor = np.maximum(_rel(m["pos"], u["pos"]), _rel(m["vel"], u["vel"])), np.maximum(_rel(u["pos"], ul["pos"]), _rel(u["vel"], ul["vel"]))
        print(f"merged vs unmerged after {steps} steps: median {np.median(d):.2e} max {d.max():.2e}; "
              f"unmerged double-vs-long-double floor: median {np.median(floor):.2e} max {floor.max():.2e}")
        assert np.median(d) <= 3 * np.median(floor) + 1e-14
        assert (d <= np.maximum(1e-10, 10 * floor)).all()  # R-noise (ii): per system against its own floor
        if bar:
            assert d.max() <= bar
        assert (m["time"] == u["time"]).all() and (m["nsteps"] == u["nsteps"]).all()


def test_loop_semantics_time_limit_monitors_and_split_runs():
    pos, vel, mass = W.generate(4, n_sys=8)
    u = _run(oracle.MVS, pos, vel, mass, 0.05, 100, t_end=0.42)
    m = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, 100, t_end=0.42)
    assert (m["status"] == oracle.DONE_TIME).all() and (m["nsteps"] == 9).all() and (m["time"] == u["time"]).all()
    assert _rel(m["pos"], u["pos"]).max() < 1e-14
    # ejection threshold inside the outermost orbit: the post-step state of step 1 trips it in both maps
    rad = np.linalg.norm(pos, axis=2).max(axis=1)
    m = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, 100, r_eject=float(rad.min()) * 0.5)
    assert (m["status"] == oracle.STOP_EJECT).all() and (m["nsteps"] == 1).all()
    # a close approach built to happen after some tens of steps: same stop step, same stop state to rounding
    d = np.array([0.05, 0.003, 0.0])
    pos[3, 2] = pos[3, 1] + d
    vel[3, 2] = vel[3, 1] - 0.4 * d / np.linalg.norm(d)
    u = _run(oracle.MVS, pos, vel, mass, 0.002, 3000, r_close=0.02)
    m = _run(oracle.MVS_MERGED, pos, vel, mass, 0.002, 3000, r_close=0.02)
    assert u["status"][3] == oracle.STOP_CLOSE and 5 < u["nsteps"][3] < 3000
    assert (m["status"] == u["status"]).all() and (m["nsteps"] == u["nsteps"]).all()
    assert _rel(m["pos"], u["pos"]).max() < 1e-11
    # a run split over two calls closes and re-opens the half sub-steps: equal to the unsplit run to rounding
    pos, vel, mass = W.generate(4, n_sys=8)
    a = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, 400)
    b = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, 150)
    b = oracle.integrate(oracle.MVS_MERGED, b["pos"], b["vel"], mass, b["time"], dt=0.05, max_steps=250, nsteps=b["nsteps"])
    assert (b["nsteps"] == 400).all() and _rel(a["pos"], b["pos"]).max() < 1e-12
    # reversal
    f = _run(oracle.MVS_MERGED, pos, vel, mass, 0.05, 2000)
    r = oracle.integrate(oracle.MVS_MERGED, f["pos"], f["vel"], mass, f["time"], dt=-0.05, t_end=-np.inf, max_steps=2000)
    assert np.abs(r["pos"] - pos).max() < 2e-10 and np.abs(r["time"]).max() < 1e-10
