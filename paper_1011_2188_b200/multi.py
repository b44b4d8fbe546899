"""Multi-GPU plumbing: histories are independent, so the proton index space is cut
into one contiguous range per rank, each rank fills its own u64 grid, and the grids are summed once
at the end -- the paper's two host threads whose "absorbed dose ... was combined",
here one integer all-reduce over NCCL (NVLink 5 / NVSwitch).  Integer sums are order-independent,
so the N-GPU grid equals the 1-GPU grid bit for bit.  No arithmetic of the method lives here."""
from __future__ import annotations


def shard_range(total: int, rank: int, world: int):
    """(first, count) of rank's contiguous share of [0, total): floor(total*(r+1)/W) - floor(total*r/W)."""
    assert 0 <= rank < world
    lo = (total * rank) // world
    hi = (total * (rank + 1)) // world
    return lo, hi - lo


def allreduce_sum_int64(t):
    """In-place sum over ranks of an int64 tensor (NCCL on CUDA tensors, gloo on CPU tensors).
    The u64 fixed-point grid is carried as int64: two's-complement addition is the same operation."""
    import torch.distributed as dist
    if dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t


def allreduce_edep(ctx, scratch):
    """Replace ctx's grid by the sum over ranks.  scratch: CUDA int64 tensor shaped like the grid."""
    ctx.fdc_get_edep_fixed(scratch)
    allreduce_sum_int64(scratch)
    ctx.fdc_set_edep_fixed(scratch)


def allreduce_squares(ctx, scratch):
    """Same for the sum-of-squares grid (FDC_TALLY_SQUARES): eq. (2)'s sums run over the histories of
    all ranks, and both sums are integers, so the N-GPU uncertainty map equals the 1-GPU one."""
    ctx.fdc_get_sq_fixed(scratch)
    allreduce_sum_int64(scratch)
    ctx.fdc_set_sq_fixed(scratch)

