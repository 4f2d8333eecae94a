"""q-sharding of the hot path across ranks ("first layer": q-batches -> MPI ranks, one GPU each;
PAPER.md:381: reduction of Sigma_inf and Sigma~ after the local work).

Stages 1-2 are independent per q; stage 3 and stage 4 produce partial sums over the rank's q shard, which one
all-reduce(sum) completes.  torch.distributed (NCCL on GPUs, gloo in the CPU tests) is the plumbing.
"""
import torch
import torch.distributed as dist


def shard_range(nk, world_size, rank):
    """Contiguous q shard [q_begin, q_end) of rank `rank`; shards differ by at most one q-point."""
    base, rem = divmod(nk, world_size)
    q_begin = rank * base + min(rank, rem)
    q_end = q_begin + base + (1 if rank < rem else 0)
    return q_begin, q_end


def allreduce_sum_(tensors, group=None):
    """In-place sum over ranks of complex tensors (viewed as real pairs: NCCL/gloo reduce real dtypes)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return tensors
    for t in tensors:
        dist.all_reduce(torch.view_as_real(t), op=dist.ReduceOp.SUM, group=group)
    return tensors
