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
