"""Multi-GPU plumbing: events are independent, so ranks take contiguous ranges of GLOBAL event
indices (whole AOSOA pages) and no data-path collective exists.  The only exchange is agreeing on the
good-helicity mask once (element-wise OR = MAX over ranks).  Philox counters use the global event index, so the
result does not depend on the split.
"""
from .binding import MG_AOSOA_V


def shard_range(nevt_total, rank, world_size, page=MG_AOSOA_V):
    """Contiguous [first, first+count) of global event indices for `rank`; every shard is a whole number of pages
    except possibly the last one."""
    npages = (nevt_total + page - 1) // page
    base, extra = divmod(npages, world_size)
    first_page = rank * base + min(rank, extra)
    count_pages = base + (1 if rank < extra else 0)
    first = min(first_page * page, nevt_total)
    last = min((first_page + count_pages) * page, nevt_total)
    return first, last - first


def merge_good_masks(mask_u8, group=None):
    """All-reduce (MAX == bitwise OR for 0/1 bytes) of the per-rank good-helicity masks; in place, returns the tensor."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(mask_u8, op=dist.ReduceOp.MAX, group=group)
    return mask_u8


def max_over_ranks(value, device=None, group=None):
    """MAX over ranks of a python float (timings)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
