"""GPU parity of the fused MVS step loop (libens, through the C ABI) against the CPU oracle on the same seeded inputs.
Tolerance (BASELINE.json north_star, config 4): max relative position/velocity difference <= 1e-10.
R-noise / DESIGN.md §7: at 10^4 steps the FP64 rounding floor itself (oracle double vs oracle long double) exceeds
1e-10 for a few systems per thousand, so the 10^4-step comparison is made per system against that system's own floor."""
import math

import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W
from parity import rel_diff

pytestmark = pytest.mark.gpu


def test_config4_1000_steps_max_parity():
    """1024 systems of config 4, 10^3 steps: the 1e-10 max criterion is meaningful here (floor ~3e-12)."""
    c = W.CONFIGS[4]
    pos, vel, mass = W.generate(4, n_sys=1024)
    g = ens.run(ens.MVS, pos, vel, mass, dt=c.dt, steps=1000)
    o = oracle.integrate(oracle.MVS, pos, vel, mass, dt=c.dt, max_steps=1000)
    assert (g["status"] == ens.DONE_STEPS).all() and (g["nsteps"] == 1000).all()
    np.testing.assert_allclose(g["time"], o["time"], rtol=0, atol=1e-9)
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    print(f"cfg4 x1000 steps: pos max {dp.max():.3e} median {np.median(dp):.3e}; vel max {dv.max():.3e}")
    assert dp.max() <= 1e-10 and dv.max() <= 1e-10


def test_config4_full_size_sampled_parity():
    """Config 4 at FULL size (131072 x 4, 10^4 steps, the launch bench.py times); the oracle recomputes a strided
    sample in double and in long double.  Per system: GPU-vs-oracle <= max(1e-10, 10 x that system's own
    double-vs-long-double floor); the distribution is printed next to the floor's."""
    c = W.CONFIGS[4]
    pos, vel, mass = W.generate(4)
    g = ens.run(ens.MVS, pos, vel, mass, dt=c.dt, steps=c.steps, want_energy=True)
    idx = np.unique(np.concatenate([np.arange(0, c.n_sys, c.n_sys // 256), [c.n_sys - 1]]))
    o = oracle.integrate(oracle.MVS, pos[idx], vel[idx], mass[idx], dt=c.dt, max_steps=c.steps)
    ol = oracle.integrate(oracle.MVS, pos[idx], vel[idx], mass[idx], dt=c.dt, max_steps=c.steps, prec=oracle.LONG_DOUBLE)
    assert (g["status"] == ens.DONE_STEPS).all() and (g["nsteps"] == c.steps).all()
    assert np.isfinite(g["pos"]).all() and np.isfinite(g["vel"]).all()
    dp, dv = rel_diff(g["pos"][idx], o["pos"]), rel_diff(g["vel"][idx], o["vel"])
    fp, fv = rel_diff(o["pos"], ol["pos"]), rel_diff(o["vel"], ol["vel"])
    q = lambda a: f"median {np.median(a):.2e} p99 {np.percentile(a, 99):.2e} max {a.max():.2e} n>1e-10 {(a > 1e-10).sum()}"
    print(f"cfg4 x{c.steps}: {len(idx)} sampled systems\n  gpu-vs-oracle pos {q(dp)}\n  gpu-vs-oracle vel {q(dv)}\n"
          f"  oracle double-vs-long-double floor pos {q(fp)}\n  floor vel {q(fv)}")
    assert (dp <= np.maximum(1e-10, 10 * fp)).all() and (dv <= np.maximum(1e-10, 10 * fv)).all()
    assert np.median(dp) <= 1e-10 and np.median(dv) <= 1e-10
    assert (dp > 1e-10).mean() <= 0.03 and (dv > 1e-10).mean() <= 0.03
    # invariants that hold at any size (R-M6): L conserved to rounding, bounded energy error
    dL = np.abs(g["L"] - g["L0"]).max(axis=1) / np.linalg.norm(g["L0"], axis=1)
    assert dL.max() <= 1e-11
    dE = np.abs((g["E"] - g["E0"]) / g["E0"])
    print(f"  |dE/E| median {np.median(dE):.2e} max {dE.max():.2e}; |dL/L| max {dL.max():.2e}")
    # bounded for all but the few systems whose planets meet closely, which a fixed-step MVS cannot follow
    assert np.median(dE) <= 1e-6 and np.percentile(dE, 99) <= 1e-5 and (dE > 1e-3).mean() <= 1e-3


def _systems(n_sys, n_body, seed):
    rng = np.random.default_rng(seed)
    pos, vel, mass = np.zeros((n_sys, n_body, 3)), np.zeros((n_sys, n_body, 3)), np.ones((n_sys, n_body))
    a = np.cumprod(np.concatenate([rng.uniform(0.6, 1.0, (n_sys, 1)), rng.uniform(1.3, 1.6, (n_sys, n_body - 1))], 1), 1)
    for b in range(1, n_body):
        m = 10.0 ** rng.uniform(-6, -3, n_sys)
        mass[:, b] = m
        e, inc = rng.uniform(0, 0.3, n_sys), rng.uniform(0, 0.05, n_sys)
        Om, om, M = (rng.uniform(0, 2 * np.pi, n_sys) for _ in range(3))
        pos[:, b], vel[:, b] = W.elements_to_cartesian(a[:, b - 1], e, inc, Om, om, M, 1.0 + m)
    mt = mass.sum(1)[:, None]
    pos -= ((mass[:, :, None] * pos).sum(1) / mt)[:, None]
    vel -= ((mass[:, :, None] * vel).sum(1) / mt)[:, None]
    return pos, vel, mass


@pytest.mark.parametrize("n_body", list(range(2, 17)))
def test_every_body_count_ragged(n_body):
    """Every supported n_body (each lane/planet split, exact and padded), a ragged ensemble that ends inside a warp."""
    n_sys = 205
    pos, vel, mass = _systems(n_sys, n_body, 300 + n_body)
    g = ens.run(ens.MVS, pos, vel, mass, dt=0.02, steps=300)
    o = oracle.integrate(oracle.MVS, pos, vel, mass, dt=0.02, max_steps=300)
    assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all()
    dp, dv = rel_diff(g["pos"], o["pos"]), rel_diff(g["vel"], o["vel"])
    assert dp.max() <= 1e-11 and dv.max() <= 1e-11, (dp.max(), dv.max())


def test_large_steps_eccentric_and_negative_dt():
    """Kepler solver away from the small-z regime: steps of a sizeable fraction of the inner period (Stumpff argument
    quartering active), e up to 0.3, and a backward run (R-M6: reversal)."""
    pos, vel, mass = _systems(160, 4, 77)
    for dt, steps in ((0.4, 200), (1.7, 60)):
        g = ens.run(ens.MVS, pos, vel, mass, dt=dt, steps=steps)
        o = oracle.integrate(oracle.MVS, pos, vel, mass, dt=dt, max_steps=steps)
        ol = oracle.integrate(oracle.MVS, pos, vel, mass, dt=dt, max_steps=steps, prec=oracle.LONG_DOUBLE)
        for key in ("pos", "vel"):
            d, floor = rel_diff(g[key], o[key]), rel_diff(o[key], ol[key])
            # steps this coarse make some systems chaotic: judge the ensemble median and each system against the
            # oracle's own double-vs-long-double rounding floor (R-noise), never against a fixed number
            ratio = d / np.maximum(1e-11, floor)
            print(f"large steps dt={dt} {key}: gpu-vs-oracle median {np.median(d):.2e} max {d.max():.2e}; floor median "
                  f"{np.median(floor):.2e} max {floor.max():.2e}; worst d / max(1e-11, floor) = {ratio.max():.2f}; "
                  f"systems beyond max(1e-10, 10 floor): {(d > np.maximum(1e-10, 10 * floor)).sum()} of {len(d)}")
            assert np.median(d) <= 3 * np.median(floor) + 1e-13, (key, dt, np.median(d), np.median(floor))
            assert (d <= np.maximum(1e-10, 10 * floor)).all(), (key, dt, ratio.max())  # R-noise (ii): 10 x
    with ens.Ensemble(160, 4) as e:
        e.set_state(pos, vel, mass)
        e.integrate(ens.MVS, 0.05, 400)
        f = e.get_state()
        e.integrate(ens.MVS, -0.05, 400, t_end=-np.inf)
        r = e.get_state()
    assert rel_diff(f["pos"], pos).max() > 1e-2
    # the reversal defect is rounding noise amplified by each system's own sensitivity: judge it per system against
    # the oracle's own forward-backward defect (R-M6, R-noise), 1e-11 where the oracle's is smaller than that
    of = oracle.integrate(oracle.MVS, pos, vel, mass, dt=0.05, max_steps=400)
    orv = oracle.integrate(oracle.MVS, of["pos"], of["vel"], mass, of["time"], dt=-0.05, max_steps=400, t_end=-np.inf)
    d, dref = rel_diff(r["pos"], pos), rel_diff(orv["pos"], pos)
    print(f"reversal defect: gpu median {np.median(d):.2e} max {d.max():.2e}; oracle's own median {np.median(dref):.2e} "
          f"max {dref.max():.2e}; systems where the ORACLE's defect exceeds 1e-10: {(dref > 1e-10).sum()}, the gpu's: "
          f"{(d > 1e-10).sum()}; worst d / max(1e-11, oracle's) = {(d / np.maximum(1e-11, dref)).max():.2f}")
    assert (d <= np.maximum(1e-11, 10 * dref)).all(), (d / np.maximum(1e-11, dref)).max()
    assert d.max() <= 1e-10  # the absolute bar of the round-1 test, met again (measured 8.2e-11; the oracle's own: 4.6e-11)
    assert np.median(d) <= 1e-12 and np.abs(r["time"]).max() <= 1e-12


def test_test_particles_follow_kepler_orbits_exactly():
    """R-M5: with massless planets the map is the exact Kepler flow for any step: one period in 7 steps returns."""
    n_sys = 64
    pos, vel, mass = _systems(n_sys, 3, 5)
    mass[:, 1:] = 0.0
    pos -= pos[:, :1]
    vel -= vel[:, :1]
    r = np.linalg.norm(pos[:, 1], axis=1)
    a = 1.0 / (2.0 / r - (vel[:, 1] ** 2).sum(1))
    period = 2 * np.pi * a ** 1.5
    for s in range(n_sys):
        g = ens.run(ens.MVS, pos[s:s + 1], vel[s:s + 1], mass[s:s + 1], dt=period[s] / 7, steps=7)
        assert np.abs(g["pos"][0, 1] - pos[s, 1]).max() <= 2e-13 * a[s]


def test_monitors_time_stop_and_sticky_status():
    pos, vel, mass = _systems(96, 4, 11)
    pos[5, 3] = pos[5, 2] + np.array([0.04, 0.0, 0.0])          # close pair -> STOP_CLOSE early
    vel[9, 3] = vel[9, 3] + np.array([3.0, 0.5, 0.0])            # unbound -> STOP_EJECT
    kw = dict(dt=0.02, r_close=0.05, r_eject=6.0)
    time = np.linspace(0.0, 1.9, 96)
    with ens.Ensemble(96, 4) as e:
        e.set_state(pos, vel, mass, time)
        e.set_monitors(kw["r_close"], kw["r_eject"])
        e.integrate(ens.MVS, kw["dt"], 10**6, t_end=8.0)
        g = e.get_state()
        o = oracle.integrate(oracle.MVS, pos, vel, mass, time, max_steps=10**6, t_end=8.0, **kw)
        assert o["status"][5] == oracle.STOP_CLOSE and o["status"][9] == oracle.STOP_EJECT
        assert (o["status"] == oracle.DONE_TIME).sum() >= 80
        assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all()
        assert (g["time"] == o["time"]).all()
        assert rel_diff(g["pos"], o["pos"]).max() <= 1e-10
        e.integrate(ens.MVS, kw["dt"], 5)
        g2 = e.get_state()
        stopped = g["status"] >= ens.STOP_CLOSE
        assert (g2["pos"][stopped] == g["pos"][stopped]).all() and (g2["nsteps"][~stopped] == g["nsteps"][~stopped] + 5).all()


def test_rcp_within_one_ulp():
    """The MVS kernel's divide-free reciprocal (float rcp seed + cubic FP64 refinement) is within 1 ulp of the
    correctly rounded 1/x over the radii it sees and near the ends of its documented domain, both signs."""
    import torch
    rng = np.random.default_rng(6)
    x = np.concatenate([10.0 ** rng.uniform(-4, 4, 400000), 10.0 ** rng.uniform(-36, 36, 100000),
                        -(10.0 ** rng.uniform(-4, 4, 1000)), np.array([1.0, 2.0, 3.0, 0.1, 7.0, 1e-3])])
    y = ens.rcp_probe(torch.from_numpy(x).cuda()).cpu().numpy()
    ref = 1.0 / x.astype(np.longdouble)
    err = np.abs((y.astype(np.longdouble) - ref) / np.spacing(np.abs(ref).astype(np.float64))).astype(np.float64)
    print(f"rcp: max error {err.max():.3f} ulp, mean {err.mean():.3f}")
    assert err.max() <= 1.0


def test_kepler_drift_stress_against_the_oracle():
    """The kernel's Kepler solver (Chebyshev-corrected Newton, Taylor finish, series / quartered Stumpff, bisection
    fallback) against the oracle's plain Newton solver on 3000 random test particles: circular to strongly hyperbolic,
    steps from a hundredth of a radian to several revolutions, both directions.  With massless planets one MVS step
    is exactly one Kepler drift of each planet about the unit-mass star (R-M5)."""
    rng = np.random.default_rng(2024)
    n_sys, n_pl = 1000, 3
    pos = np.zeros((n_sys, n_pl + 1, 3))
    vel = np.zeros((n_sys, n_pl + 1, 3))
    mass = np.zeros((n_sys, n_pl + 1))
    mass[:, 0] = 1.0
    for b in range(1, n_pl + 1):
        r = 10.0 ** rng.uniform(-0.5, 1.0, n_sys)
        d = rng.normal(size=(n_sys, 3))
        d /= np.linalg.norm(d, axis=1)[:, None]
        pos[:, b] = r[:, None] * d
        w = rng.normal(size=(n_sys, 3))
        w /= np.linalg.norm(w, axis=1)[:, None]
        speed = np.sqrt(1.0 / r) * 10.0 ** rng.uniform(-0.7, 0.35, n_sys)  # 0.2 .. 2.2 of circular: e up to ~4
        vel[:, b] = speed[:, None] * w
    for dt in (0.05, 3.0, -11.0, 40.0):
        g = ens.run(ens.MVS, pos, vel, mass, dt=dt, steps=1, t_end=math.copysign(math.inf, dt))
        worst = 0.0
        for s in range(0, n_sys, 7):  # the oracle is called particle by particle: a strided sample
            for b in range(1, n_pl + 1):
                # reference: the oracle in long double; tolerance: 1e-11, or 10 x the oracle's own double-vs-long-double
                # difference where that is larger (a step of 40 spans up to ~60 revolutions of the tightest orbits)
                q, p, _ = oracle.kepler_drift(pos[s, b], vel[s, b], 1.0, dt, prec=oracle.LONG_DOUBLE)
                qd, pd, _ = oracle.kepler_drift(pos[s, b], vel[s, b], 1.0, dt)
                sq, sp = np.linalg.norm(q) + np.linalg.norm(pos[s, b]), np.linalg.norm(p) + np.linalg.norm(vel[s, b])
                floor = max(np.abs(qd - q).max() / sq, np.abs(pd - p).max() / sp)
                err = max(np.abs(g["pos"][s, b] - q).max() / sq, np.abs(g["vel"][s, b] - p).max() / sp)
                worst = max(worst, err / max(1e-11, 10 * floor))
        assert worst <= 1.0, (dt, worst)
        assert (g["status"] == ens.DONE_STEPS).all() and (g["nsteps"] == 1).all() and np.isfinite(g["pos"]).all()
