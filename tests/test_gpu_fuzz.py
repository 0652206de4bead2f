"""Seeded random differential test: every integrator x random (n_body, ensemble size, step, budget, time limit, start
times, monitors, direction) against the oracle.  Each case is small (the oracle runs it in well under a second); the
point is the combinations the hand-written cases do not enumerate (e.g. a time limit with staggered start times on a
padded 5-lane shape with both monitors armed, run backwards)."""
import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import ens
from parity import rel_diff
from test_gpu_mvs import _systems

pytestmark = pytest.mark.gpu

INTEGRATORS = [
    ("hermite", ens.HERMITE, oracle.HERMITE), ("carry", ens.HERMITE_CARRY, oracle.HERMITE_CARRY),
    ("hermite_adaptive", ens.HERMITE_ADAPTIVE, oracle.HERMITE_ADAPTIVE), ("rkck", ens.RKCK, oracle.RKCK),
    ("rkck_adaptive", ens.RKCK_ADAPTIVE, oracle.RKCK_ADAPTIVE), ("mvs", ens.MVS, oracle.MVS),
    ("mvs_merged", ens.MVS_MERGED, oracle.MVS_MERGED),
]


@pytest.mark.parametrize("name,gi,oi", INTEGRATORS)
def test_random_cases_against_the_oracle(name, gi, oi):
    rng = np.random.default_rng(sum(map(ord, name)))  # a fixed seed per integrator
    for case in range(16):
        n_body = int(rng.integers(2, 17))
        n_sys = int(rng.integers(1, 180))
        pos, vel, mass = _systems(n_sys, n_body, int(rng.integers(1, 10**6)))
        if name.startswith("mvs"):  # the splitting needs planets that stay apart: mild eccentricities come from _systems
            dt = float(rng.choice([0.01, 0.03]))
        elif name == "hermite_adaptive":
            dt = float(rng.choice([0.01, 0.03]))          # tau
        elif name == "rkck_adaptive":
            dt = float(rng.choice([0.005, 0.05, 2.0]))    # first trial step (2.0: starts with rejections)
        else:
            dt = float(rng.choice([0.002, 0.005]))
        backwards = bool(rng.integers(0, 2)) and name != "rkck_adaptive"
        sign = -1.0 if backwards else 1.0
        steps = int(rng.integers(1, 120))
        use_t_end = bool(rng.integers(0, 2))
        time = rng.uniform(-0.05, 0.05, n_sys) if rng.integers(0, 2) else None
        t_end = sign * float(rng.uniform(0.05, 0.4)) if use_t_end else sign * np.inf
        if use_t_end:
            steps = 10**6
        r_close = float(rng.choice([0.0, 0.05, 0.2]))
        r_eject = float(rng.choice([np.inf, 3.0, 50.0]))
        kw = dict(dt=sign * dt, t_end=t_end, r_close=r_close, r_eject=r_eject)
        eps = float(rng.choice([1e-7, 1e-9]))
        g = ens.run(gi, pos, vel, mass, steps=steps, time=time, rk_eps=eps, **kw)
        o = oracle.integrate(oi, pos, vel, mass, time, max_steps=steps, rk_eps=eps, **kw)
        tag = (name, case, n_body, n_sys, dt, steps, t_end, r_close, r_eject, backwards)
        same = (g["status"] == o["status"]) & (g["nsteps"] == o["nsteps"])
        if name == "rkck_adaptive":
            same &= (g["nreject"] == o["nreject"]) & (g["time"] == o["time"])
            assert same.mean() >= 0.9, tag
        else:
            assert same.all(), (tag, np.nonzero(~same)[0][:5], g["status"][~same][:5], o["status"][~same][:5],
                                g["nsteps"][~same][:5], o["nsteps"][~same][:5])
        tol = 1e-10
        if name == "hermite_adaptive":
            assert np.abs(g["time"] - o["time"]).max() <= 1e-12 * max(1.0, np.abs(o["time"]).max()), tag
        elif name != "rkck_adaptive":
            assert (g["time"] == o["time"]).all(), tag
        dp, dv = rel_diff(g["pos"][same], o["pos"][same]), rel_diff(g["vel"][same], o["vel"][same])
        assert dp.max() <= tol and dv.max() <= tol, (tag, dp.max(), dv.max())
