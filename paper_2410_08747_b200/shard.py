"""Host logic of the multi-GPU form of the path: rays are independent and keyed by index
(PAPER.md:73), so the ray-index range is split into contiguous shares, one per rank, each traced by that rank's own
instrument replica with no data-path collective; the paper's scatter-gather "results added at the end" (PAPER.md:77,
110) is one sum-reduce of the tally arrays after the trace.  No arithmetic of the method lives here."""
from __future__ import annotations


def ray_range(rank: int, world_size: int, n_rays: int, scaling: str = "weak"):
    """(first, count) of rank's share.  weak: every rank traces n_rays of its own, consecutive windows of the index
    space (whole job = world_size * n_rays).  strong: n_rays in total, split as evenly as possible, the first
    n_rays % world_size ranks taking one more."""
    if not (0 <= rank < world_size) or n_rays < 0:
        raise ValueError("bad rank / world_size / n_rays")
    if scaling == "weak":
        return rank * n_rays, n_rays
    if scaling != "strong":
        raise ValueError(f"unknown scaling {scaling!r}")
    base, extra = divmod(n_rays, world_size)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def reduce_tallies(tallies, dst=None, group=None):
    """Sums (N, p, p2) tensors over ranks in place with torch.distributed (NCCL on GPUs, gloo on CPU): all-reduce, or a
    reduce to `dst`.  Integer counts are exact; p and p2 are summed in the collective's rank order."""
    import torch.distributed as dist
    for t in tallies:
        if dst is None:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        else:
            dist.reduce(t, dst=dst, op=dist.ReduceOp.SUM, group=group)
    return tallies
