"""Column split of a block over ranks: every column of X is an independent unit of H~X, of the shifted
apply (its own eps_j) and of the filter, so B columns are dealt to the ranks in contiguous slices and NO data-path
collective exists.  The only communication is the harness's barrier and the max-over-ranks of the step time."""


def column_slice(B_total, rank, world):
    """Contiguous slice [lo, hi) of the B_total columns owned by `rank`; sizes differ by at most one."""
    if world < 1 or not (0 <= rank < world) or B_total < 0:
        raise ValueError("column_slice: bad (B_total=%r, rank=%r, world=%r)" % (B_total, rank, world))
    q, r = divmod(B_total, world)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise max of a list of floats over all ranks (times are reported as the slowest rank's)."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def job_throughput(units_per_rank, world, seconds):
    """Whole-job units/s under weak scaling: every rank processed units_per_rank in `seconds` (max over ranks)."""
    return units_per_rank * world / seconds
