"""N > 1 path of bench.py on CPU: the path does not shard (replicas only), so the only
multi-rank logic is the MAX-over-ranks timing and the whole-job aggregation.  world_size 2, gloo."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    local = [10.0 + rank, 7.0 - rank, 3.0 * (rank + 1)]          # step ms, e2e ms, kernel ms of this "replica"
    mx = bench.reduce_max_over_ranks(local, dist, "cpu")
    val = bench.whole_job_value(world, 1000.0, 5, mx[0])
    dist.barrier()
    q.put((rank, mx, val, bench._dist_env()))
    dist.destroy_process_group()


def test_replicas_max_over_ranks_and_whole_job_value_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, val, env in out:
        assert mx == [11.0, 7.0, 6.0]                          # slowest rank decides, on every rank
        assert val == pytest.approx(2 * 1000.0 * 5 / 11.0e-3)   # both replicas' units over the slowest time
        assert env[0] == rank and env[2] == 2


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max_over_ranks([1.5, 2.5]) == [1.5, 2.5]
    assert bench.whole_job_value(1, 10.0, 2, 4.0) == pytest.approx(5000.0)
