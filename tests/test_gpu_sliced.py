"""The time-sliced persistent grid of the fixed-step Hermite kernel (hermite_kernel<..., SLICED>) and the boundary's
device / allocation contract.  Slicing only schedules: the step is a pure function of the state (R6), so results are
bit-identical to the one-pass kernel for every slice length, grid size and body count; against the oracle the usual
tolerances hold."""
import numpy as np
import pytest
import torch

import oracle
from paper_1208_1157_b200 import ens
from paper_1208_1157_b200 import workloads as W
from parity import rel_diff
from test_gpu_hermite import _crossing_ensemble, _random_systems

pytestmark = pytest.mark.gpu

KEYS = ("pos", "vel", "time", "status", "nsteps")


def _run(e, pos, vel, mass, dt, steps, t_end=np.inf, time=None):
    e.set_state(pos, vel, mass, time)
    e.integrate(ens.HERMITE, dt, steps, t_end)
    return e.get_state()


@pytest.mark.parametrize("n_body", [3, 6, 7, 10, 12, 15, 16])
def test_sliced_is_bit_identical_to_one_pass(n_body):
    n_sys = 1531  # ragged: ends in the middle of a warp group
    pos, vel, mass = _random_systems(n_sys, n_body, 300 + n_body)
    with ens.Ensemble(n_sys, n_body) as e:
        e.set_option(ens.OPT_SLICE_MODE, 2)
        ref = _run(e, pos, vel, mass, 0.004, 203)
        for slice_steps, warps_per_sm in ((1, 0), (7, 1), (50, 2), (203, 0), (1000, 3)):
            e.set_option(ens.OPT_SLICE_MODE, 1)
            e.set_option(ens.OPT_SLICE_STEPS, slice_steps)
            e.set_option(ens.OPT_SLICE_WARPS_PER_SM, warps_per_sm)
            got = _run(e, pos, vel, mass, 0.004, 203)
            for k in KEYS:
                assert (got[k] == ref[k]).all(), (k, slice_steps, warps_per_sm)
    o = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=0.004, max_steps=203)
    assert (ref["status"] == o["status"]).all() and (ref["nsteps"] == o["nsteps"]).all()
    assert rel_diff(ref["pos"], o["pos"]).max() <= 1e-11 and rel_diff(ref["vel"], o["vel"]).max() <= 1e-11


def test_sliced_monitors_time_limit_and_sticky_stops():
    """Stops (close approach, ejection), the t_end test and systems that start at different times behave exactly as in
    the one-pass kernel when the run is cut into slices: status, stop step, time and state bit-identical."""
    n_sys = 200
    pos, vel, mass = _crossing_ensemble(n_sys)
    time = np.linspace(0.0, 1.5, n_sys)
    with ens.Ensemble(n_sys, 3) as e:
        e.set_monitors(0.02, 5.0)
        e.set_option(ens.OPT_SLICE_MODE, 2)
        ref = _run(e, pos, vel, mass, 0.002, 3000, t_end=5.0, time=time)
        e.integrate(ens.HERMITE, 0.002, 77)  # DONE_TIME / DONE_STEPS systems run again, stopped ones stay
        ref2 = e.get_state()
        assert len(set(ref["status"])) >= 3
        for slice_steps in (1, 13, 640):
            e.set_option(ens.OPT_SLICE_MODE, 1)
            e.set_option(ens.OPT_SLICE_STEPS, slice_steps)
            got = _run(e, pos, vel, mass, 0.002, 3000, t_end=5.0, time=time)
            e.integrate(ens.HERMITE, 0.002, 77)
            got2 = e.get_state()
            for k in KEYS:
                assert (got[k] == ref[k]).all() and (got2[k] == ref2[k]).all(), (k, slice_steps)
    o = oracle.integrate(oracle.HERMITE, pos, vel, mass, time, dt=0.002, t_end=5.0, max_steps=3000, r_close=0.02, r_eject=5.0)
    assert (ref["status"] == o["status"]).all() and (ref["nsteps"] == o["nsteps"]).all() and (ref["time"] == o["time"]).all()


def test_huge_step_budget_with_a_time_limit_stays_cheap_when_sliced():
    """max_steps = 10^9 with t_end deciding the run: the slice count is capped (the last slice is open-ended), so the
    launch does not hand out millions of empty tasks; results equal the one-pass kernel's, also when the steps needed
    exceed 256 slices' worth (systems that start far before t_end)."""
    import time as _time
    n_sys = 1531
    pos, vel, mass = _random_systems(n_sys, 15, 77)
    t0 = np.where(np.arange(n_sys) % 5 == 0, -3.0, 0.0)  # every fifth system needs 4x the steps of the others
    with ens.Ensemble(n_sys, 15) as e:
        e.set_option(ens.OPT_SLICE_MODE, 2)
        ref = _run(e, pos, vel, mass, 0.004, 10**9, t_end=1.0, time=t0)
        for slice_steps in (0, 1, 3):  # 0: the library's choice; 1, 3: 256 slices cover only 256 / 768 of the 250 / 1000 steps
            e.set_option(ens.OPT_SLICE_MODE, 1)
            e.set_option(ens.OPT_SLICE_STEPS, slice_steps)
            w0 = _time.perf_counter()
            got = _run(e, pos, vel, mass, 0.004, 10**9, t_end=1.0, time=t0)
            assert _time.perf_counter() - w0 < 20.0
            for k in KEYS:
                assert (got[k] == ref[k]).all(), (k, slice_steps)
    assert (ref["status"] == ens.DONE_TIME).all() and set(ref["nsteps"]) == {250, 1000}


def test_library_chooses_slicing_for_config3_and_results_match_the_oracle():
    """Config 3 at full size (1.15 waves of resident warps) is the case the sliced grid exists for: the library's own
    choice must pick it, and sampled systems agree with the oracle (short run: the full run is test_gpu_hermite's)."""
    c = W.CONFIGS[3]
    pos, vel, mass = W.generate(3)
    with ens.Ensemble(c.n_sys, c.n_body) as e:
        e.set_monitors(c.r_close, c.r_eject)
        g = _run(e, pos, vel, mass, c.dt, 600)
        info = e.info()
        e.set_option(ens.OPT_SLICE_MODE, 2)
        r = _run(e, pos, vel, mass, c.dt, 600)
        assert e.info()["blocks"] > info["blocks"]  # the one-pass grid is larger than the persistent one
    for k in KEYS:
        assert (g[k] == r[k]).all(), k
    idx = np.arange(0, c.n_sys, 257)
    o = oracle.integrate(oracle.HERMITE, pos[idx], vel[idx], mass[idx], dt=c.dt, max_steps=600, r_close=c.r_close,
                         r_eject=c.r_eject)
    assert (g["status"][idx] == o["status"]).all() and (g["nsteps"][idx] == o["nsteps"]).all()
    assert rel_diff(g["pos"][idx], o["pos"]).max() <= 1e-11


def test_two_handles_on_two_streams_run_concurrently_and_independently():
    """Two ensembles, two streams, calls interleaved from one host thread: device-space calls only enqueue (no
    allocation, no synchronisation inside ens_integrate), and each handle's results equal its solo run bit for bit."""
    pa, va, ma = W.generate(0, n_sys=4096)
    pb, vb, mb = W.generate(2, n_sys=2048)
    ta = [torch.from_numpy(x).cuda() for x in (pa, va, ma)]
    tb = [torch.from_numpy(x).cuda() for x in (pb, vb, mb)]
    solo_a = ens.run(ens.HERMITE, pa, va, ma, dt=0.01, steps=400)
    solo_b = ens.run(ens.HERMITE_ADAPTIVE, pb, vb, mb, dt=0.02, steps=150)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    with ens.Ensemble(4096, 3) as ea, ens.Ensemble(2048, 6) as eb:
        for _ in range(2):
            ea.set_state(*ta, stream=sa)
            eb.set_state(*tb, stream=sb)
            ea.integrate(ens.HERMITE, 0.01, 400, stream=sa)
            eb.integrate(ens.HERMITE_ADAPTIVE, 0.02, 150, stream=sb)
        da = ea.get_state(device=True, stream=sa)
        db = eb.get_state(device=True, stream=sb)
        sa.synchronize()
        sb.synchronize()
    for k in KEYS:
        assert (da[k].cpu().numpy() == solo_a[k]).all() and (db[k].cpu().numpy() == solo_b[k]).all(), k


def test_handle_is_bound_to_its_device_not_to_the_current_one():
    """With several GPUs: a handle created on device 0 keeps running there while device 1 is current (and vice
    versa).  With one GPU: the guard is exercised by the same calls and the current device is left untouched."""
    pos, vel, mass = W.generate(0, n_sys=500)
    ref = ens.run(ens.HERMITE, pos, vel, mass, dt=0.01, steps=100)
    n_dev = torch.cuda.device_count()
    with torch.cuda.device(0):
        e0 = ens.Ensemble(500, 3)
    other = 1 if n_dev > 1 else 0
    with torch.cuda.device(other):
        e0.set_state(pos, vel, mass, stream=0)
        e0.integrate(ens.HERMITE, 0.01, 100, stream=0)
        got = e0.get_state(stream=0)
        E, _ = e0.energy(stream=0)
        assert torch.cuda.current_device() == other
        e0.close()
    for k in KEYS:
        assert (got[k] == ref[k]).all(), k
    assert np.isfinite(E).all()


def test_set_option_argument_checks():
    with ens.Ensemble(10, 3) as e:
        L = ens.lib()
        assert L.ens_test_set_option(e._h, 99, 0) == ens.EINVAL
        assert L.ens_test_set_option(e._h, ens.OPT_THREADS, 33) == ens.EINVAL
        assert L.ens_test_set_option(e._h, ens.OPT_SLICE_MODE, 3) == ens.EINVAL
        assert L.ens_test_set_option(None, ens.OPT_THREADS, 0) == ens.EINVAL
        assert L.ens_test_set_option(e._h, ens.OPT_THREADS, 64) == ens.OK
        assert L.ens_reserve_host_staging(e._h) == ens.OK and L.ens_reserve_host_staging(e._h) == ens.OK
        assert L.ens_reserve_host_staging(None) == ens.EINVAL


def test_logged_segments_on_the_sliced_grid_give_the_same_records():
    """ens_integrate_logged runs ens_integrate segment by segment: with the time-sliced grid forced for every segment the
    log holds the same records (matched by system and step count) as with the one-pass kernel, bit for bit."""
    n_sys = 700
    pos, vel, mass = _random_systems(n_sys, 13, 5)
    logs = []
    for mode in (2, 1):
        with ens.Ensemble(n_sys, 13) as e:
            e.set_option(ens.OPT_SLICE_MODE, mode)
            e.set_option(ens.OPT_SLICE_STEPS, 40)
            e.log_enable(3 * n_sys)
            e.set_state(pos, vel, mass)
            e.integrate_logged(ens.HERMITE, 0.004, 300, 100)
            log = e.log_read()
            order = np.lexsort((log["nsteps"], log["sys"]))
            logs.append({k: log[k][order] for k in ("sys", "nsteps", "time", "status", "pos", "vel")})
            assert len(log["sys"]) == 3 * n_sys and log["dropped"] == 0
    for k in logs[0]:
        assert (logs[0][k] == logs[1][k]).all(), k
