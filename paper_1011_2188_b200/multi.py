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


def allreduce_edep(ctx, squares=False):
    """Replace ctx's energy grid (and, with squares=True, its sum-of-squares grid: eq. (2)'s sums run over the
    histories of all ranks) by the sum over ranks, IN PLACE on the library's own device arrays
    (fdc_edep_device_ptr): one all-reduce per grid, no staging copies.  The tensors alias the context's memory and
    the collective runs on the stream the context was created on (torch's current stream), after the transport
    kernels queued there."""
    e, q = ctx.fdc_edep_device_ptr()
    allreduce_sum_int64(e)
    if squares and q is not None:
        allreduce_sum_int64(q)


def sharded_step(ctx, beamlets, first, n_mine, seed, flags, dose_out, world):
    """One step of the hot path on this rank: zero, transport this rank's proton range [first, first + n_mine),
    and -- for world > 1 -- sum the grids over ranks in place, then convert to Gy (each GPU unit
    handles its histories; "the absorbed dose from both threads was combined" at the end).  With world == 1 the Gy
    conversion rides on fdc_run itself.  dose_out: CUDA tensor or host array (then the call synchronises)."""
    ctx.fdc_reset()
    if world == 1:
        ctx.fdc_run(beamlets, first, n_mine, 1, seed, flags=flags, dose_gy=dose_out)
        return
    ctx.fdc_run(beamlets, first, n_mine, 1, seed, flags=flags)
    # FDC_SQUARES_BY_HISTORY alone also fills the squares grid (the library implies FDC_TALLY_SQUARES)
    from . import FDC_SQUARES_BY_HISTORY, FDC_TALLY_SQUARES
    allreduce_edep(ctx, squares=bool(flags & (FDC_TALLY_SQUARES | FDC_SQUARES_BY_HISTORY)))
    if dose_out is not None:
        ctx.fdc_to_gy(dose_out)
