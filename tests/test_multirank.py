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


# ------------------------------------------------------------------------------ sharded pair sum
class _OracleEngine:
    """Stand-in for mopal.Mopal on CPU: the same members ShardedMopal drives, every stage by the oracle.  A rank's
    share = the rows [lo, hi) of the acceleration given by the library's own partition (mo_shard_range)."""

    def __init__(self, w):
        import numpy as np
        import oracle
        self.np, self.oracle, self.w = np, oracle, w
        self.mu, self.gm = w.G * w.m_star, w.G * w.mass
        self.x, self.v = w.x.copy(), w.v.copy()
        self.a = torch.zeros((3, w.nb), dtype=torch.float64)
        self.rank, self.world = 0, 1
        self.pairs = None

    def set_shard(self, rank, world):
        self.rank, self.world = rank, world

    def _partial_accel(self):
        from paper_2601_19654_b200 import mopal as M
        lo, hi = M.shard_range(self.w.nb, self.rank, self.world)
        rows = self.np.arange(lo, hi, dtype=self.np.int32)
        a = self.np.zeros((3, self.w.nb))
        if len(rows):
            a[:, rows] = self.oracle.accel_rows(self.gm, self.x, self.w.rcrit, rows)[0]
        self.a.copy_(torch.from_numpy(a))

    def accel(self):
        self._partial_accel()

    def accel_summed(self):
        pass

    def step_begin(self, dt):
        o, a = self.oracle, self.a.numpy()
        self.v = o.kick(0.5 * dt, self.v, a)
        self.x, _ = o.jump(0.5 * dt, self.mu, self.gm, self.x, self.v)
        x0, v0 = self.x.copy(), self.v.copy()
        self.x, self.v, _ = o.drift(self.mu, dt, self.x, self.v)
        self.pairs = o.encounters(dt, x0, v0, self.x, self.v, self.w.rcrit)["pairs"]
        self.x, _ = o.jump(0.5 * dt, self.mu, self.gm, self.x, self.v)
        self._partial_accel()

    def step_end(self, dt, sync=True):
        self.v = self.oracle.kick(0.5 * dt, self.v, self.a.numpy())
        return None

    def invalidate_accel(self):
        pass


def _shard_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2601_19654_b200 import workloads as W
    from paper_2601_19654_b200.sharded import ShardedMopal
    w = W.shrink(1, 300)
    eng = _OracleEngine(w)
    sm = ShardedMopal(eng, dist, rank, world)
    sm.step(w.dt, 3)
    q.put((rank, eng.x, eng.v, eng.a.numpy().copy(), eng.pairs, sm.allreduces))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_step_driver_gloo_world2_against_the_unsharded_oracle():
    """ShardedMopal's protocol (share of a -> all-reduce -> kick; begin / sum / end per step) with the library's own
    partition, on two gloo ranks: both ranks end bit-identical and equal to the plain oracle steps."""
    import numpy as np
    import oracle
    sys.path.insert(0, ROOT)
    from paper_2601_19654_b200 import workloads as W
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = W.shrink(1, 300)
    mu, gm = w.G * w.m_star, w.G * w.mass
    a, _ = oracle.accel(gm, w.x, w.rcrit)
    x, v = w.x, w.v
    for _ in range(3):
        r = oracle.step(mu, gm, w.rcrit, w.dt, x, v, a)
        x, v, a = r["x"], r["v"], r["a"]
    (r0, x0, v0, a0, p0, n0), (r1, x1, v1, a1, p1, n1) = out
    assert n0 == n1 == 4                                         # one all-reduce for the first a, one per step
    assert np.array_equal(x0, x1) and np.array_equal(v0, v1) and np.array_equal(a0, a1) and np.array_equal(p0, p1)
    # rows are summed whole on one rank and padded with zeros on the other: the all-reduce is exact
    assert np.array_equal(x0, x) and np.array_equal(v0, v) and np.array_equal(a0, a)
    assert np.array_equal(p0, r["pairs"])


def test_shard_range_partitions_without_gaps():
    sys.path.insert(0, ROOT)
    from paper_2601_19654_b200 import mopal as M
    for n in (0, 1, 7, 4455, 65535):
        for world in (1, 2, 3, 8):
            edges = [M.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[k][1] == edges[k + 1][0] for k in range(world - 1))
            sizes = [hi - lo for lo, hi in edges]
            assert max(sizes) - min(sizes) <= 1
    L = M.load()
    import ctypes as C
    lo, hi = C.c_int64(), C.c_int64()
    assert L.mo_shard_range(10, 2, 2, C.byref(lo), C.byref(hi)) == M.MO_EINVAL
    assert L.mo_shard_range(10, 0, 0, C.byref(lo), C.byref(hi)) == M.MO_EINVAL
    assert L.mo_shard_range(-1, 0, 1, C.byref(lo), C.byref(hi)) == M.MO_EINVAL
