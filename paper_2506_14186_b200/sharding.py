"""Multi-GPU plumbing: environments are independent, so ranks take contiguous env ranges and the
data path has no collective.  Only a caller that wants batch-summed parameter gradients reduces dL/dp."""


def shard_range(nenv, rank, world):
    """Contiguous, balanced [lo, hi) of `nenv` environments for `rank` of `world`."""
    base, rem = divmod(int(nenv), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def sum_param_grads(dLdparams, group=None):
    """Batch-sum dL/dp on this rank, then all-reduce over ranks (NCCL on GPUs, gloo on CPU)."""
    import torch.distributed as dist
    g = dLdparams.sum(dim=0)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(g, op=dist.ReduceOp.SUM, group=group)
    return g


def max_over_ranks(value, device="cpu", group=None):
    """Max of a python float over ranks (timing: the slowest rank defines the step)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def sum_over_ranks(value, device="cpu", group=None):
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return float(t.item())
