"""Multi-GPU host logic: neutrons are independent, so the path shards by
contiguous neutron-id ranges -- one process per GPU, no data-path collective while tracing -- and the
only exchange is the paper's gather/merge of the detector on the master rank:
one sum-reduction of 3 x ny x nx values.  With a counter-based RNG the union of the shards is the
same set of neutrons as a single-GPU run."""
from __future__ import annotations


def shard_ids(n_total: int, rank: int, world: int):
    """Contiguous id range [first, first+n) of `rank`: the first n_total % world ranks get one more."""
    base, rem = divmod(n_total, world)
    n = base + (1 if rank < rem else 0)
    first = rank * base + min(rank, rem)
    return first, n


def weak_shard(n_per_rank: int, rank: int):
    """Weak scaling: every rank traces n_per_rank new ids; rank r owns [r n, (r+1) n)."""
    return rank * n_per_rank, n_per_rank


def merge_detectors(tensors, dst: int = 0, group=None):
    """Sum-reduce the detector arrays (sum_p, sum_p2 as float64; counts as int64) onto rank dst.
    Works on any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests)."""
    import torch.distributed as dist
    if not dist.is_initialized() or dist.get_world_size(group) == 1:
        return tensors
    for t in tensors:
        dist.reduce(t, dst=dst, op=dist.ReduceOp.SUM, group=group)
    return tensors
