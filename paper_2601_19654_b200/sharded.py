"""The hybrid step with the O(N^2) pair sum sharded over several GPUs.

One process per GPU, every rank holds the whole state; only the pair kernel's work units are split
(``mo_set_shard``), and the ranks' partial accelerations are summed with ONE all-reduce of ``a`` (3*ld doubles) per
step - ``torch.distributed`` (NCCL over NVLink on GPUs) is the plumbing, nothing of the method's arithmetic is here.
Every O(N) stage and the encounter pass run replicated on identical data, so x, v, the pair lists and the statistics
are bit-identical on every rank (an all-reduce hands every rank the same sum).

``engine`` is a ``mopal.Mopal`` (or anything with the same ``set_shard / accel / accel_summed / step_begin /
step_end / a`` members - the CPU tests drive this class with a stand-in built on the oracle, under ``gloo``).
"""
from __future__ import annotations


class ShardedMopal:
    def __init__(self, engine, dist=None, rank=0, world=1, group=None):
        self.engine, self.dist, self.rank, self.world, self.group = engine, dist, int(rank), int(world), group
        if self.world > 1 and dist is None:
            raise ValueError("ShardedMopal: world > 1 needs a torch.distributed module")
        engine.set_shard(self.rank, self.world)
        self.allreduces = 0
        self._a_current = False

    def _sum_a(self):
        """a <- sum over the ranks of the partial accelerations (in place, on the engine's stream)."""
        if self.world > 1:
            self.dist.all_reduce(self.engine.a, op=self.dist.ReduceOp.SUM, group=self.group)
            self.allreduces += 1
            self.engine.accel_summed()

    def accel(self):
        self.engine.accel()
        self._sum_a()
        self._a_current = True

    def step(self, dt, nsteps=1, sync=True):
        """nsteps hybrid steps; returns the statistics of the last one (None with sync=False)."""
        if self.world == 1:
            return self.engine.step(dt, nsteps, sync=sync)
        if not self._a_current:
            self.accel()
        st = None
        for k in range(int(nsteps)):
            self.engine.step_begin(dt)
            self._sum_a()
            st = self.engine.step_end(dt, sync=sync and k == nsteps - 1)
        return st

    def invalidate_accel(self):
        self._a_current = False
        self.engine.invalidate_accel()
