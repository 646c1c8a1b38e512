"""N > 1 is 'replicas only': the only cross-rank logic is the timing reduction
(max over ranks) and the work sum.  Covered here on CPU with gloo, world size 2."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r pretends to have taken (10 + r) ms for 500 iterations and 1000 launches
    ms, iters, launches = bench.reduce_over_ranks(10.0 + rank, 500.0, 1000.0, world, device="cpu")
    # workloads of different ranks are different problems (seed offset), same shape
    p0 = bench.workload("c1", rank)[0]
    out.put((rank, ms, iters, launches, p0.seed))
    dist.destroy_process_group()


def test_replica_reduction_max_time_sum_work():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, iters, launches, seed in res:
        assert ms == pytest.approx(11.0)        # max over ranks
        assert iters == pytest.approx(1000.0)   # sum over ranks
        assert launches == pytest.approx(2000.0)
    assert res[0][4] != res[1][4]               # different seeds per replica


def test_single_rank_reduction_is_identity():
    import bench
    assert bench.reduce_over_ranks(3.0, 7.0, 9.0, 1, device="cpu") == (3.0, 7.0, 9.0)
