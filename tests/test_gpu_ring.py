"""The cross-lane ring of the many-lane shapes exchanges bodies through warp-private shared memory (hermite_kernel.cuh,
acc_pairs.cuh).  Its results must not depend on how many warps share a block (the shared-memory slice of a warp is
indexed by its position in the block), on the neighbours a system shares its warp with, or on stopped neighbours
(partial masks at the warp barriers): bit-identity across launch shapes, and parity with the oracle."""
import numpy as np
import pytest

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W
from parity import rel_diff

pytestmark = pytest.mark.gpu

CASES = [("hermite", ens.HERMITE, oracle.HERMITE, 2e-3, (9, 10, 11, 12, 13, 15, 16)),
         ("carry", ens.HERMITE_CARRY, oracle.HERMITE_CARRY, 2e-3, (9, 10, 15)),
         ("adaptive", ens.HERMITE_ADAPTIVE, oracle.HERMITE_ADAPTIVE, 0.02, (9, 10, 15)),
         ("rkck", ens.RKCK, oracle.RKCK, 2e-3, (6, 8, 10, 11, 16)),
         ("rkck_adaptive", ens.RKCK_ADAPTIVE, oracle.RKCK_ADAPTIVE, 0.02, (6, 10, 15)),
         ("mvs", ens.MVS, oracle.MVS, 0.01, (10, 11, 12, 14, 16)),
         ("mvs_merged", ens.MVS_MERGED, oracle.MVS_MERGED, 0.01, (10, 14))]


def _systems(n_body, n_sys, seed=7):
    """Compact planetary systems with random phases and masses (bounded for the few hundred steps of these tests)."""
    rng = np.random.default_rng(seed + n_body)
    pos, vel, mass = W.paper_ics(n_body, n_sys, planet_mass=1e-5, alpha=0.25)
    ph = rng.uniform(0, 2 * np.pi, (n_sys, n_body))
    c, s = np.cos(ph), np.sin(ph)
    x, y, vx, vy = pos[:, :, 0].copy(), pos[:, :, 1].copy(), vel[:, :, 0].copy(), vel[:, :, 1].copy()
    pos[:, :, 0], pos[:, :, 1] = c * x - s * y, s * x + c * y
    vel[:, :, 0], vel[:, :, 1] = c * vx - s * vy, s * vx + c * vy
    pos[:, 1:, 2] = 0.01 * rng.standard_normal((n_sys, n_body - 1))
    mass[:, 1:] *= rng.uniform(0.5, 2.0, (n_sys, n_body - 1))
    return pos, vel, mass


def _run(gi, pos, vel, mass, dt, steps, threads=None, **kw):
    n_sys, n_body = mass.shape
    with ens.Ensemble(n_sys, n_body) as e:
        if threads:
            e.set_option(ens.OPT_THREADS, threads)
        e.set_state(pos, vel, mass)
        e.set_monitors(kw.get("r_close", 0.0), kw.get("r_eject", float("inf")))
        e.set_rk_tolerance(1e-9)
        e.integrate(gi, dt, steps)
        return e.get_state()


@pytest.mark.parametrize("name,gi,oi,dt,bodies", CASES, ids=[c[0] for c in CASES])
def test_results_do_not_depend_on_warps_per_block_or_on_warp_mates(name, gi, oi, dt, bodies):
    for n_body in bodies:
        pos, vel, mass = _systems(n_body, 203)
        ref = _run(gi, pos, vel, mass, dt, 60)
        for threads in (32, 64, 128):
            g = _run(gi, pos, vel, mass, dt, 60, threads=threads)
            for k in ("pos", "vel", "time", "status", "nsteps"):
                assert np.array_equal(g[k], ref[k]), (name, n_body, threads, k)
        # the same systems in another order share their warps with other systems: same bits, system by system
        perm = np.random.default_rng(3).permutation(203)
        g = _run(gi, pos[perm], vel[perm], mass[perm], dt, 60)
        for k in ("pos", "vel", "time", "status", "nsteps"):
            assert np.array_equal(g[k], ref[k][perm]), (name, n_body, "permuted", k)
        o = oracle.integrate(oi, pos, vel, mass, dt=dt, max_steps=60, rk_eps=1e-9)
        if name != "rkck_adaptive":
            assert (ref["nsteps"] == o["nsteps"]).all() and (ref["status"] == o["status"]).all()
            assert rel_diff(ref["pos"], o["pos"]).max() <= 1e-11 and rel_diff(ref["vel"], o["vel"]).max() <= 1e-11, (name, n_body)


@pytest.mark.parametrize("name,gi,oi,dt,bodies", CASES[:1] + CASES[3:4] + CASES[5:6], ids=["hermite", "rkck", "mvs"])
def test_stopped_neighbours_do_not_disturb_the_ring(name, gi, oi, dt, bodies):
    """Every third system is ejected at its first monitor call (its outer planet starts beyond r_eject), so the warps run
    with partial masks from step 1 on: the others must match the oracle and a run without the ejected systems."""
    for n_body in bodies[:3]:
        pos, vel, mass = _systems(n_body, 120)
        a_out = np.linalg.norm(pos[:, -1], axis=1)
        r_eject = 1.5 * a_out.max()
        pos[::3, -1] *= 2.0  # beyond r_eject from the start (speed unchanged: still bound to the star)
        g = _run(gi, pos, vel, mass, dt, 80, r_eject=r_eject)
        o = oracle.integrate(oi, pos, vel, mass, dt=dt, max_steps=80, r_eject=r_eject)
        assert (g["status"] == o["status"]).all() and (g["nsteps"] == o["nsteps"]).all()
        assert (o["status"][::3] == oracle.STOP_EJECT).all() and (o["nsteps"][::3] == 1).all()
        keep = np.ones(120, bool)
        keep[::3] = False
        assert (o["status"][keep] == oracle.DONE_STEPS).all()
        assert rel_diff(g["pos"], o["pos"]).max() <= 1e-11
        alone = _run(gi, pos[keep], vel[keep], mass[keep], dt, 80, r_eject=r_eject)
        assert np.array_equal(alone["pos"], g["pos"][keep]) and np.array_equal(alone["vel"], g["vel"][keep])
