"""Host-side logic of the N > 1 path, covered on CPU with world_size-2 gloo processes.

The data path has no collective (systems are independent): what is checked here is the partition,
the per-rank ranges of the seeded generator, the control-plane reductions (max of a time, sum of counters) and the
gather of results.  The per-rank "integration" is done by the oracle (this is a test), standing in for the CUDA
path that each rank runs on its own GPU.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1208_1157_b200 import shard  # noqa: E402
from paper_1208_1157_b200 import workloads as W  # noqa: E402


@pytest.mark.parametrize("n_sys,world", [(0, 1), (1, 2), (63, 2), (64, 2), (65, 2), (1000, 3), (131072, 8), (100, 8)])
def test_partition_covers_every_system_once(n_sys, world):
    parts = shard.partition(n_sys, world)
    assert len(parts) == world and parts[0][0] == 0 and parts[-1][1] == n_sys
    for (a0, b0), (a1, b1) in zip(parts, parts[1:]):
        assert b0 == a1 and a0 <= b0
    for a, b in parts:
        assert a % shard.GRANULE == 0 or a == n_sys
    sizes = [b - a for a, b in parts]
    assert sum(sizes) == n_sys and max(sizes) - min(sizes) < 2 * shard.GRANULE  # one granule + the ragged tail


def test_partition_rejects_bad_arguments():
    with pytest.raises(ValueError):
        shard.partition(10, 0)
    with pytest.raises(ValueError):
        shard.partition(-1, 2)


def test_generator_ranges_agree_with_the_unsharded_generator():
    full = W.generate(2, n_sys=200)
    for a, b in shard.partition(200, 3):
        part = W.generate(2, n_sys=b - a, offset=a)
        for f, p in zip(full, part):
            assert (f[a:b] == p).all()
    a, b = shard.weak_range(128, 3)
    assert (a, b) == (384, 512)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_sys, outdir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        c = W.CONFIGS[0]
        a, b = shard.my_range(n_sys, rank, world)
        pos, vel, mass = W.generate(0, n_sys=b - a, offset=a)
        o = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=c.dt, max_steps=50, r_close=0.01, r_eject=100.0,
                             nthreads=1)
        t = shard.max_over_ranks(1.0 + rank)
        hist = shard.sum_counters(shard.status_histogram(o["status"]))
        allpos = shard.gather_to_rank0(o["pos"], n_sys, world)
        allsteps = shard.gather_to_rank0(o["nsteps"], n_sys, world)
        if rank == 0:
            np.savez(os.path.join(outdir, "r0.npz"), pos=allpos, nsteps=allsteps, hist=hist, t=t)
        else:
            assert allpos is None and t == float(world)
    finally:
        dist.destroy_process_group()


def test_two_ranks_reproduce_the_single_process_run(tmp_path):
    import oracle
    n_sys, world = 150, 2  # ragged: rank 0 gets 128 systems, rank 1 gets 22
    mp.spawn(_worker, args=(world, _free_port(), n_sys, str(tmp_path)), nprocs=world, join=True)
    got = np.load(os.path.join(tmp_path, "r0.npz"))
    c = W.CONFIGS[0]
    pos, vel, mass = W.generate(0, n_sys=n_sys)
    ref = oracle.integrate(oracle.HERMITE, pos, vel, mass, dt=c.dt, max_steps=50, r_close=0.01, r_eject=100.0, nthreads=1)
    assert (got["pos"] == ref["pos"]).all() and (got["nsteps"] == ref["nsteps"]).all()
    assert got["hist"].sum() == n_sys and got["hist"][oracle.DONE_STEPS] == n_sys
    assert float(got["t"]) == 2.0


def test_reductions_without_a_process_group_are_identity():
    assert shard.max_over_ranks(3.5) == 3.5
    assert (shard.sum_counters([1, 2, 3]) == np.array([1, 2, 3])).all()
    x = np.arange(6).reshape(3, 2)
    assert shard.gather_to_rank0(x, 3, 1) is x
