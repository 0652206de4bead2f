"""The device state log (ens_log_enable / ens_integrate_logged / ens_log_read, DESIGN.md R-L1, R-L2)."""
import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W
from parity import rel_diff

pytestmark = pytest.mark.gpu


def test_periodic_snapshots_match_the_oracle_at_every_logged_step():
    n_sys = 200
    pos, vel, mass = W.generate(0, n_sys=n_sys)
    with ens.Ensemble(n_sys, 3) as e:
        e.log_enable(5 * n_sys + 7)
        e.set_state(pos, vel, mass)
        e.integrate_logged(ens.HERMITE, 0.01, 450, 100)  # segments of 100, 100, 100, 100, 50 steps
        log = e.log_read()
        final = e.get_state()
    assert len(log["sys"]) == 5 * n_sys and log["dropped"] == 0
    assert sorted(set(log["nsteps"].tolist())) == [100, 200, 300, 400, 450]
    for k in (100, 300, 450):
        o = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.01, max_steps=k)
        sel = np.flatnonzero(log["nsteps"] == k)
        order = sel[np.argsort(log["sys"][sel])]
        assert (log["sys"][order] == np.arange(n_sys)).all()
        assert rel_diff(log["pos"][order], o["pos"]).max() <= 1e-12 and rel_diff(log["vel"][order], o["vel"]).max() <= 1e-12
        assert np.abs(log["time"][order] - o["time"]).max() <= 1e-12
    # the step is a pure function of the state: logging in segments changes nothing
    plain = ens.run(ens.HERMITE, pos, vel, mass, dt=0.01, steps=450)
    assert (plain["pos"] == final["pos"]).all() and (plain["vel"] == final["vel"]).all()
    last = np.flatnonzero(log["nsteps"] == 450)
    assert (log["pos"][last[np.argsort(log["sys"][last])]] == final["pos"]).all()


def test_stop_events_only_and_capacity():
    n_sys = 150
    pos, vel, mass = W.generate(0, n_sys=n_sys)
    pos[7, 2] = pos[7, 1] + np.array([0.05, 0.0, 0.0])  # planet 2 of system 7 flies at planet 1
    vel[7, 2] = vel[7, 1] + np.array([-0.5, 0.0, 0.0])
    with ens.Ensemble(n_sys, 3) as e:
        e.set_monitors(0.02, 100.0)
        e.log_enable(16)
        e.set_state(pos, vel, mass)
        e.integrate_logged(ens.HERMITE, 0.001, 1000, 50, what=ens.LOG_STOPS)
        log = e.log_read()
        final = e.get_state()
        assert len(log["sys"]) == 1 and log["sys"][0] == 7 and log["status"][0] == ens.STOP_CLOSE
        assert log["nsteps"][0] == final["nsteps"][7] and 50 < log["nsteps"][0] < 200
        assert (log["pos"][0] == final["pos"][7]).all() and log["time"][0] == final["time"][7]
        o = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.001, max_steps=1000, r_close=0.02, r_eject=100.0)
        assert o["nsteps"][7] == log["nsteps"][0]
        # snapshots of everything overflow a 16-record buffer: the excess is counted, not written
        e.log_enable(16)
        e.set_state(pos, vel, mass)
        e.integrate_logged(ens.MVS, 0.01, 20, 10)
        log = e.log_read()
        # (system 7 stops in the first segment and is therefore logged once, not twice)
        assert len(log["sys"]) == 16 and log["dropped"] == 2 * n_sys - 1 - 16
        # a new state restarts the step counters: systems are logged again from their first segment on
        e.log_enable(n_sys)
        e.set_state(pos, vel, mass)
        e.integrate_logged(ens.RKCK, 0.01, 10, 10)
        e.set_state(pos, vel, mass)
        e.integrate_logged(ens.RKCK, 0.01, 10, 10)
        log = e.log_read()
        assert len(log["sys"]) == n_sys and log["dropped"] == n_sys


def test_log_argument_checks():
    pos, vel, mass = W.generate(0, n_sys=8)
    with ens.Ensemble(8, 3) as e:
        e.set_state(pos, vel, mass)
        with pytest.raises(ens.EnsError):
            e.integrate_logged(ens.HERMITE, 0.01, 10, 5)  # no log buffer
        e.log_enable(4)
        for bad in (dict(log_every=0), dict(what=0)):
            with pytest.raises(ens.EnsError):
                e.integrate_logged(ens.HERMITE, 0.01, 10, **{"log_every": 5, **bad})
        with pytest.raises(ens.EnsError):
            e.log_enable(-1)
        with pytest.raises(ens.EnsError):  # 10^9 steps in segments of 100: ten million segments would be enqueued
            e.integrate_logged(ens.HERMITE, 0.01, 10**9, 100, t_end=1.0)
        e.integrate_logged(ens.HERMITE, 0.01, 10**5, 10**4, t_end=1.0)  # 10 segments; t_end ends the run in the first
        st = e.get_state()
        assert (st["status"] == ens.DONE_TIME).all() and (st["nsteps"] == 100).all()
