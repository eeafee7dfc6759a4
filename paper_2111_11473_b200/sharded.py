"""Sharded evaluation of the residual over several ranks.

One process per GPU.  The Cholesky index is cut into equal contiguous ranges, the rows of the T2^2 terms into equal
row blocks (`thc_shard_range`); every rank computes its packed partial sums with its own kernels, ONE all-reduce over
`torch.distributed` sums them (NCCL over NVLink on GPUs; the only exchange step of the path), and every rank finishes
redundantly.  The orchestration is written against a small backend protocol so that the host logic can be exercised
on CPU ranks (gloo) in the test-suite:

    backend.shard(rank, world)      -> 1-D tensor: this rank's packed partial sums
    backend.finish(packed)          -> R (tensor [NP, NP]) from the rank-summed buffer
    backend.energy_shard(rank, world) -> 1-element tensor: this rank's part of E
"""
from __future__ import annotations


class CudaBackend:
    """The library on this rank's device.  `B_ov`, `B_oo`, `B_vv` are the rank's own L-slices (thc_shard_range)."""

    def __init__(self, handle, Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps):
        self.h = handle
        self.x = (Xo, Xv, Z, B_ov, B_oo, B_vv, Y, V, eps)
        self._packed = None

    def shard(self, rank, world):
        self._packed = self.h.thc_residual_shard(*self.x, rank, world, out=self._packed)
        return self._packed

    def finish(self, packed):
        Xo, Xv, Z, _, _, _, Y, V, eps = self.x
        return self.h.thc_residual_finish(Xo, Xv, Z, Y, V, eps, packed)

    def energy_shard(self, rank, world):
        Xo, Xv, Z, B_ov = self.x[:4]
        return self.h.thc_energy_shard(Xo, Xv, Z, B_ov, rank, world)


def _rank_world(group):
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(group), dist.get_world_size(group)
    return 0, 1


def residual_sharded(backend, group=None):
    """R on every rank: local partial sums -> one all-reduce (sum) -> redundant finish."""
    import torch.distributed as dist
    rank, world = _rank_world(group)
    packed = backend.shard(rank, world)
    if world > 1:
        dist.all_reduce(packed, op=dist.ReduceOp.SUM, group=group)
    return backend.finish(packed)


def energy_sharded(backend, group=None):
    import torch.distributed as dist
    rank, world = _rank_world(group)
    E = backend.energy_shard(rank, world)
    if world > 1:
        dist.all_reduce(E, op=dist.ReduceOp.SUM, group=group)
    return E
