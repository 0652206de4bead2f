"""ens_hermite_static: the fixed-step Hermite loop for callers that cannot allocate (its scratch is a static device
array of the library, shared by every call).  Checked against the existing path (handle + ens_integrate(ENS_HERMITE)):
bit-identical, as every scheduling variant of that kernel is (tests/test_gpu_sliced.py), on calls in a row that use
different amounts of the shared scratch and find the previous call's contents in it.

Collected last on purpose (the suite runs with pytest -x): nothing here depends on the other tests having run, and
nothing they do depends on this file."""
import numpy as np
import pytest
import torch

from paper_1208_1157_b200 import ens
from test_gpu_hermite import _crossing_ensemble, _random_systems

pytestmark = pytest.mark.gpu


def _to_soa(pos, vel, mass, time, n_pad):
    """Host AoS arrays -> the library's SoA layout as CUDA tensors (layout only: DESIGN.md section 5)."""
    n_sys, n_body = mass.shape

    def rows(a, k):  # [n_sys][k] -> [k][n_pad]
        out = torch.zeros((k, n_pad), dtype=torch.float64, device="cuda")
        out[:, :n_sys] = torch.from_numpy(np.ascontiguousarray(a.reshape(n_sys, k).T)).cuda()
        return out

    t = torch.zeros(n_pad, dtype=torch.float64, device="cuda")
    if time is not None:
        t[:n_sys] = torch.from_numpy(np.asarray(time, dtype=np.float64)).cuda()
    return dict(pos=rows(pos, n_body * 3), vel=rows(vel, n_body * 3), mass=rows(mass, n_body), time=t,
                status=torch.zeros(n_pad, dtype=torch.int32, device="cuda"),
                nsteps=torch.zeros(n_pad, dtype=torch.int64, device="cuda"))


def _from_soa(s, n_sys, n_body):
    back = lambda a: a[:, :n_sys].T.contiguous().cpu().numpy().reshape(n_sys, n_body, 3)
    return dict(pos=back(s["pos"]), vel=back(s["vel"]), time=s["time"][:n_sys].cpu().numpy(),
                status=s["status"][:n_sys].cpu().numpy(), nsteps=s["nsteps"][:n_sys].cpu().numpy())


def _static(s, n_sys, n_body, dt, steps, **kw):
    ens.hermite_static(s["pos"], s["vel"], s["mass"], s["time"], s["status"], s["nsteps"], n_sys, n_body, dt, steps, **kw)


def _existing(pos, vel, mass, time, dt, steps_list, t_end=np.inf, r_close=0.0, r_eject=np.inf):
    n_sys, n_body = mass.shape
    with ens.Ensemble(n_sys, n_body) as e:
        e.set_state(pos, vel, mass, time)
        e.set_monitors(r_close, r_eject)
        for steps in steps_list:
            e.integrate(ens.HERMITE, dt, steps, t_end)
        return e.get_state()


def _same(got, ref, tag):
    for k in ("status", "nsteps", "time", "pos", "vel"):
        assert np.array_equal(got[k], ref[k]), (tag, k)


def test_static_scratch_entry_point_matches_the_handle_path_on_calls_in_a_row():
    # call 1: many-lane shape (5 lanes x 3 bodies), 255 warp-groups of scratch, ragged tail
    n1, b1 = 1527, 15
    p1, v1, m1 = _random_systems(n1, b1, 4242)
    s1 = _to_soa(p1, v1, m1, None, 1536)
    _static(s1, n1, b1, 0.004, 150)
    # call 2 right behind it on the same stream: another ensemble, one system per thread, 41 warp-groups (the scratch
    # still holds call 1's progress words), monitors armed, staggered start times, a time limit
    n2, b2 = 1300, 3
    p2, v2, m2 = _crossing_ensemble(n2)
    t2 = np.linspace(0.0, 1.5, n2)
    kw2 = dict(t_end=5.0, r_close=0.02, r_eject=5.0)
    s2 = _to_soa(p2, v2, m2, t2, 1344)
    _static(s2, n2, b2, 0.002, 10 ** 6, **kw2)
    # call 3: call 1's ensemble goes on from where it stopped (nsteps accumulate, DONE_STEPS runs again)
    _static(s1, n1, b1, 0.004, 77)
    torch.cuda.synchronize()
    got1, got2 = _from_soa(s1, n1, b1), _from_soa(s2, n2, b2)
    assert (s1["time"][n1:] == 0).all() and (s1["nsteps"][n1:] == 0).all()  # padding columns untouched

    _same(got1, _existing(p1, v1, m1, None, 0.004, [150, 77]), "call 1 + 3")
    ref2 = _existing(p2, v2, m2, t2, 0.002, [10 ** 6], **kw2)
    _same(got2, ref2, "call 2")
    assert (got1["nsteps"] == 227).all()
    assert len(np.unique(ref2["status"])) >= 3  # on time, close approach, ejection all occur


def test_static_scratch_entry_point_runs_under_stream_capture():
    """The call made while a stream is being captured into a CUDA graph: cudaMalloc, cudaFree and every synchronising
    call are illegal there (they fail and invalidate the capture), so a graph that instantiates and replays is the
    proof that the entry point only enqueues and allocates nothing.  Each replay advances the caller's arrays in
    place, as a direct call does."""
    n, b = 1000, 10
    p, v, m = _random_systems(n, b, 99)
    s = _to_soa(p, v, m, None, 1024)
    _static(s, n, b, 0.004, 40)  # first call on the device outside capture: one-time set-up (module load, symbol address)
    stream = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    stream.wait_stream(torch.cuda.current_stream())
    with torch.cuda.graph(graph, stream=stream):
        _static(s, n, b, 0.004, 40, stream=torch.cuda.current_stream())
    graph.replay()
    graph.replay()
    torch.cuda.synchronize()
    _same(_from_soa(s, n, b), _existing(p, v, m, None, 0.004, [40, 40, 40]), "captured")
    assert (s["nsteps"][:n] == 120).all()


def test_static_scratch_entry_point_rejects_what_it_cannot_hold():
    t = torch.zeros(64, dtype=torch.float64, device="cuda")
    i32, i64 = torch.zeros(64, dtype=torch.int32, device="cuda"), torch.zeros(64, dtype=torch.int64, device="cuda")
    L = ens.lib()

    def call(n_sys, n_pad, n_body):
        return L.ens_hermite_static(t.data_ptr(), t.data_ptr(), t.data_ptr(), t.data_ptr(), i32.data_ptr(), i64.data_ptr(),
                                    n_sys, n_pad, n_body, 0.01, float("inf"), 10, 0.0, float("inf"), None)

    # sizes beyond the static scratch are refused before anything is touched (the arrays here are 64 elements long)
    for n_body, per_group in ((3, 32), (10, 6), (12, 10), (15, 6)):
        too_many = ens.STATIC_MAX_GROUPS * per_group + 1
        assert call(too_many, too_many, n_body) == ens.ETOOLARGE
    assert b"static scratch" in L.ens_strerror(ens.ETOOLARGE)
    assert call(0, 64, 3) == ens.EINVAL and call(65, 64, 3) == ens.EINVAL and call(8, 64, 17) == ens.EINVAL
    assert L.ens_hermite_static(None, t.data_ptr(), t.data_ptr(), t.data_ptr(), i32.data_ptr(), i64.data_ptr(),
                                8, 64, 3, 0.01, float("inf"), 10, 0.0, float("inf"), None) == ens.EINVAL
    with pytest.raises(ValueError):  # host arrays are not accepted
        ens.hermite_static(np.zeros(9 * 64), t, t, t, i32, i64, 8, 3, 0.01, 10)
    torch.cuda.synchronize()
    assert (t == 0).all() and (i32 == 0).all() and (i64 == 0).all()
