"""Host-side plan for the paper's i-range decomposition: rank k computes the
force vectors of floor(N/P) particles against all N sources, the "main" rank (0) also takes the
mod(N, P) remainder; positions are replicated, one exchange (all-gather of the drifted
positions) per step.  Pure index arithmetic + torch.distributed plumbing, no method arithmetic."""
from __future__ import annotations


def i_range(rank: int, world: int, n: int) -> tuple[int, int]:
    """[begin, end) of the particles whose forces `rank` computes.  Rank 0 holds the remainder."""
    base, rem = divmod(n, world)
    if rank == 0:
        return 0, base + rem
    begin = base + rem + (rank - 1) * base
    return begin, begin + base


def all_ranges(world: int, n: int) -> list[tuple[int, int]]:
    return [i_range(r, world, n) for r in range(world)]


def gather_soa(local, n: int, group=None):
    """All-gather per-rank SoA slices (3, cnt_r) into the replicated SoA array (3, n).
    Slices may differ in length by the remainder, so they are padded to the longest."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    ranges = all_ranges(world, n)
    longest = max(e - b for b, e in ranges)
    pad = torch.zeros((3, longest), dtype=local.dtype, device=local.device)
    pad[:, : local.shape[1]] = local
    buf = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(buf, pad, group=group)
    out = torch.empty((3, n), dtype=local.dtype, device=local.device)
    for (b, e), piece in zip(ranges, buf):
        out[:, b:e] = piece[:, : e - b]
    return out
