"""H_eff.psi sharded over ranks, one process per GPU.

Every rank holds the whole MPS and both environments; `dmrg_set_shard` deals the psi' blocks to the ranks by
analytic flops and each rank runs only the tasks of the blocks it owns.  The exchange is one all-reduce of the
padded psi' vector per apply (disjoint blocks: a sum with exact zeros), called by the library through the reduce
callback, so `dmrg_davidson` runs in lock-step on all ranks with replicated vectors.  This module is plumbing
only: it hands `torch.distributed.all_reduce` to the library.
"""
from __future__ import annotations


def make_reduce(group=None):
    """The `reduce` callable of `DMRG.set_shard`: in-place sum over the ranks of `group` (NCCL for CUDA tensors)."""
    import torch.distributed as dist

    def _reduce(t):
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)

    return _reduce


def shard_over_ranks(dmrg, group=None):
    """Shard `dmrg`'s apply over the ranks of `group` (default: the world).  Call before `env_build`."""
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    dmrg.set_shard(rank, world, make_reduce(group) if world > 1 else None)
    return rank, world
