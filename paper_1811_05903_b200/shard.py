"""Host-side plan for sharding the force evaluation over ranks: the paper's decomposition (every node
holds all coordinates and masses, node k computes the force vectors of ITS particles against all N sources, one exchange
of positions per step), with the particles dealt to the ranks ROUND-ROBIN in blocks of 2,048: the sets
are radially ordered, so contiguous slabs would give the inner ranks the dense core and the outer ranks the sparse halo;
every P-th block gives each rank the same mix of near and far tile pairs.  (The paper's contiguous floor(N/P) ranges,
remainder to the main rank, are kept as i_range for reference.)  Pure index arithmetic + torch.distributed plumbing, no
method arithmetic."""
from __future__ import annotations

BLOCK = 2048          # steps_block_size(): the i-block of the force kernels


def i_range(rank: int, world: int, n: int) -> tuple[int, int]:
    """The paper's contiguous plan (L139): [begin, end) of rank's particles; rank 0 holds the remainder."""
    base, rem = divmod(n, world)
    if rank == 0:
        return 0, base + rem
    begin = base + rem + (rank - 1) * base
    return begin, begin + base


def all_ranges(world: int, n: int) -> list[tuple[int, int]]:
    return [i_range(r, world, n) for r in range(world)]


def owned_blocks(rank: int, world: int, n: int, block: int = BLOCK) -> list[int]:
    """Blocks rank, rank + world, ... of the ceil(n / block) blocks (possibly none when world > number of blocks)."""
    nb = (n + block - 1) // block
    return list(range(rank, nb, world))


def owned_count(rank: int, world: int, n: int, block: int = BLOCK) -> int:
    return sum(min(block, n - b * block) for b in owned_blocks(rank, world, n, block))


def owned_indices(rank: int, world: int, n: int, block: int = BLOCK):
    """Global particle indices of rank's blocks, ascending (the order of the packed per-rank arrays)."""
    import numpy as np
    blocks = owned_blocks(rank, world, n, block)
    if not blocks:
        return np.empty(0, dtype=np.int64)
    return np.concatenate([np.arange(b * block, min(n, (b + 1) * block), dtype=np.int64) for b in blocks])


class Gather:
    """All-gather of the ranks' packed SoA slices (3, cnt_r) into the replicated SoA array (3, n), with every buffer and
    index tensor allocated ONCE (no allocation per step): ranks' counts differ by at most one block, slices are padded to
    the longest."""

    def __init__(self, world: int, n: int, device, dtype, block: int = BLOCK):
        import torch
        self.world, self.n = world, n
        self.index = [torch.from_numpy(owned_indices(r, world, n, block)).to(device) for r in range(world)]
        self.longest = max(max(len(ix) for ix in self.index), 1)
        self.send = torch.zeros((3, self.longest), dtype=dtype, device=device)
        self.recv = torch.zeros((world, 3, self.longest), dtype=dtype, device=device)
        self.recv_list = list(self.recv.unbind(0))

    def __call__(self, local, out, group=None):
        """out[:, owned_indices(r)] = rank r's `local` for every r; returns out (shape (3, n), preallocated by the caller)."""
        import torch.distributed as dist
        self.send[:, : local.shape[1]].copy_(local)
        if self.world > 1:
            dist.all_gather(self.recv_list, self.send, group=group)
        else:
            self.recv[0].copy_(self.send)
        for r, ix in enumerate(self.index):
            if len(ix):
                out.index_copy_(1, ix, self.recv[r, :, : len(ix)])
        return out


class ShardedStep:
    """One rank's side of the sharded KDK step of bench.py (N > 1 GPUs): kick/drift of the rank's particles, exchange of the
    drifted positions, forces of the rank's blocks against all sources (steps_forces_blocks).  The three phases are
    separate calls so that a single-GPU test can play several ranks one after the other (tests/test_parity_gpu.py)."""

    def __init__(self, S, rank: int, world: int, pos, vel, mass, soft, mixed: bool):
        import torch
        self.S, self.rank, self.world, self.mixed = S, rank, world, mixed
        self.n = mass.numel()
        self.mass, self.soft = mass, soft
        self.x_all = pos.clone()                                        # replicated sources (3, n)
        self.index = torch.from_numpy(owned_indices(rank, world, self.n)).to(pos.device)
        self.cnt = int(self.index.numel())
        self.x = self.x_all.index_select(1, self.index).contiguous()    # the rank's particles, packed (3, cnt)
        self.v = vel.index_select(1, self.index).contiguous()
        self.m = mass.index_select(0, self.index).contiguous()
        self.a = torch.empty((3, max(self.cnt, 1)), dtype=torch.float64, device=pos.device)[:, : self.cnt].contiguous()
        self.gather = Gather(world, self.n, pos.device, pos.dtype)

    def forces(self):
        if self.cnt:
            self.S.steps_forces_blocks(self.x_all, self.mass, self.soft, self.rank, self.world, self.a, mixed=self.mixed)

    def kick_drift(self, coeffs):
        if self.cnt:
            self.S.steps_kick_drift(self.x, self.v, self.a, coeffs)

    def exchange(self, group=None):
        self.gather(self.x, self.x_all, group=group)

    def step(self, coeffs, group=None):
        self.kick_drift(coeffs)
        self.exchange(group)
        self.forces()


class WorkSharedStep:
    """One rank's side of the KDK step with the force evaluation shared by WORK (steps_forces_share): every rank holds and
    advances ALL particles (the O(N) kick/drift is repeated on every rank, bit-identically), evaluates its share of the pair
    evaluations -- the pair-symmetric kernels at their single-GPU rate -- into a partial acceleration of every particle, and
    the one exchange per step is a sum-reduction of those partials (3N doubles).  The phases are separate calls so that a
    single-GPU test can play several ranks one after the other."""

    def __init__(self, S, rank: int, world: int, pos, vel, mass, soft, mixed: bool):
        import torch
        self.S, self.rank, self.world, self.mixed = S, rank, world, mixed
        self.n = mass.numel()
        self.cnt = self.n                                               # every rank advances every particle
        self.mass, self.soft = mass, soft
        self.x, self.v, self.m = pos.clone(), vel.clone(), mass
        self.a = torch.empty_like(self.x)                               # this rank's partial, then the reduced sum

    def forces_part(self):
        self.S.steps_forces_share(self.x, self.mass, self.soft, self.rank, self.world, self.a, mixed=self.mixed)

    def reduce(self, group=None):
        if self.world > 1:
            import torch.distributed as dist
            dist.all_reduce(self.a, op=dist.ReduceOp.SUM, group=group)

    def forces(self, group=None):
        self.forces_part()
        self.reduce(group)

    def kick_drift(self, coeffs):
        self.S.steps_kick_drift(self.x, self.v, self.a, coeffs)

    def step(self, coeffs, group=None):
        self.kick_drift(coeffs)
        self.forces(group)
