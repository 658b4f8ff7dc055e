"""N > 1 host logic on CPU (gloo, world_size 2): the path has no exchange step, so what the
ranks share is the slab partition and the max/sum reduction of bench.py's timing scalars."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2411_19617_b200.slabs import weighted_z_slabs, z_slabs  # noqa: E402


def test_z_slabs_cover_the_grid_disjointly():
    for nz in (0, 1, 7, 90, 287):
        for n in (1, 2, 3, 8):
            s = z_slabs(nz, n)
            assert len(s) == n and s[0][0] == 0 and s[-1][1] == nz
            assert all(a[1] == b[0] for a, b in zip(s, s[1:]))
            sizes = [b - a for a, b in s]
            assert max(sizes) - min(sizes) <= 1


def test_weighted_slabs_balance_a_cluster_in_vacuum():
    cost = np.zeros(160)
    cost[60:100] = np.hanning(40) * 1000 + 1
    s = weighted_z_slabs(list(cost), 4)
    assert s[0][0] == 0 and s[-1][1] == 160 and all(a[1] == b[0] for a, b in zip(s, s[1:]))
    per = [cost[a:b].sum() for a, b in s]
    assert max(per) < 1.25 * cost.sum() / 4


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    z0, z1 = z_slabs(90, world)[rank]
    ms = 10.0 + 5.0 * rank                      # the slower rank sets the time
    tmax, pts = bench.reduce_max_sum(ms, (z1 - z0) * 90 * 90, world)
    q.put((rank, z0, z1, tmax, pts))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_ranks_reduce_time_as_max_and_points_as_sum():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=90) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert (res[0][1], res[0][2], res[1][1], res[1][2]) == (0, 45, 45, 90)
    for r in res:
        assert r[3] == 15.0 and r[4] == 90 ** 3
