"""Helpers shared by the GPU parity tests: the parity metric (reading R13) and the oracle/CUDA runners."""
import numpy as np

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W


def rel_diff(a, b):
    """Per system: max_b |a_b - b_b|_inf / max_b |b_b|_2  (R13; `b` is the oracle)."""
    num = np.abs(a - b).max(axis=(1, 2))
    den = np.linalg.norm(b, axis=2).max(axis=1)
    return num / den


def run_oracle(c, pos, vel, mass, steps=None, dt=None, prec=oracle.DOUBLE, **kw):
    return oracle.integrate(c.integrator, pos, vel, mass, dt=c.dt if dt is None else dt,
                            max_steps=c.steps if steps is None else steps,
                            r_close=c.r_close, r_eject=c.r_eject, prec=prec, **kw)


def run_cuda(c, pos, vel, mass, steps=None, dt=None, want_energy=False):
    return ens.run(c.integrator, pos, vel, mass, dt=c.dt if dt is None else dt,
                   steps=c.steps if steps is None else steps, r_close=c.r_close, r_eject=c.r_eject,
                   want_energy=want_energy)


def energy_err(E, E0):
    return np.abs((E - E0) / E0)


def knife_edge_systems(c, pos, vel, mass, g_status, g_nsteps, o_status, o_nsteps, rel=1e-9):
    """Reading R12 as written: (status, stop step) must equal the oracle's except for systems whose deciding quantity
    sits on the knife edge.  For every mismatching system the oracle re-runs it WITHOUT monitors to the earlier of the
    two stop steps and the minimum pair separation / maximum distance from the origin of that state must be within
    `rel` (relative) of the threshold that decided.  Returns the number of such exempt systems; raises otherwise."""
    bad = np.nonzero((g_status != o_status) | (g_nsteps != o_nsteps))[0]
    for s in bad:
        k = int(min(g_nsteps[s], o_nsteps[s]))
        assert k > 0 and abs(int(g_nsteps[s]) - int(o_nsteps[s])) <= 1, (s, g_nsteps[s], o_nsteps[s])
        r = oracle.integrate(c.integrator, pos[s:s + 1], vel[s:s + 1], mass[s:s + 1], dt=c.dt, max_steps=k)
        x = r["pos"][0]
        d = np.linalg.norm(x[:, None, :] - x[None, :, :], axis=2)
        rmin = d[np.triu_indices(len(x), 1)].min()
        rmax = np.linalg.norm(x, axis=1).max()
        on_edge = abs(rmin - c.r_close) <= rel * c.r_close or abs(rmax - c.r_eject) <= rel * c.r_eject
        assert on_edge, (f"system {s}: gpu ({g_status[s]}, {g_nsteps[s]}) vs oracle ({o_status[s]}, {o_nsteps[s]}); at step {k} "
                         f"min separation {rmin!r} (r_close {c.r_close}), max radius {rmax!r} (r_eject {c.r_eject}): not a knife edge")
    return len(bad)
