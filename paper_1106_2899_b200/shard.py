"""Ensemble sharding over ranks.

Chains are independent (eq 54), so an ensemble is split into contiguous
ranges of the GLOBAL chain index, one per rank; Philox is keyed by the global index, so a
shard reproduces its part of the single-GPU run bit for bit.  The only exchange of the
path is the sum over ranks of the fixed-point int64 stress sums (exact and order
independent, so the result does not depend on the number of ranks).

Host logic only: no arithmetic of the method lives here.
"""
import os


def world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process: 0, 0, 1)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def strong_range(n_chains_total, rank, world_size):
    """Contiguous share [k0, k1) of a FIXED total ensemble: the first (total % world) ranks
    hold one chain more."""
    base, extra = divmod(int(n_chains_total), int(world_size))
    k0 = rank * base + min(rank, extra)
    return k0, k0 + base + (1 if rank < extra else 0)


def weak_range(n_chains_per_rank, rank):
    """Contiguous share [k0, k1) when every rank holds the same number of chains."""
    k0 = int(rank) * int(n_chains_per_rank)
    return k0, k0 + int(n_chains_per_rank)


def allreduce_sums(t, group=None, ctx=None):
    """In-place sum over ranks of an int64 tensor of fixed-point sums (stress samples
    [n][12] or correlator sums).  NCCL on device tensors, gloo on CPU tensors.
    ctx: the Ensemble whose workspace t aliases (ssm_stress_sums_device).  torch orders the collective
    with torch's CURRENT stream; when the context runs on a stream of its own, the two are ordered with
    events (ssm_stream_wait_ctx before, ssm_ctx_wait_stream after) -- no host synchronisation."""
    import torch
    import torch.distributed as dist
    assert t.dtype == torch.int64
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        cur = torch.cuda.current_stream(t.device) if (ctx is not None and t.is_cuda) else None
        if cur is not None:
            ctx.stream_wait_ctx(cur)
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        if cur is not None:
            ctx.ctx_wait_stream(cur)
    return t


def stress_means(sums, n_chains_total):
    """Ensemble means (eq 54) from the all-reduced fixed-point sums [n][12]: ssm_stress_from_sums of the C ABI
    (the fixed point and the remaining -1 of eq 16's diagonal are the library's business, not this module's)."""
    from . import stress_from_sums
    return stress_from_sums(sums, n_chains_total)
