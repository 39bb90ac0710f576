"""-m "not gpu": the N > 1 plumbing of bench.py on CPU -- the paper's decomposition (every node
holds all particles, node k computes the force vectors of its share against all of them, one exchange of positions
per step) with the i-blocks of 2,048 dealt round-robin to the ranks.  world_size 2 and 3, `gloo`
backend, 127.0.0.1 rendezvous.  The per-rank force call is played by the oracle's idx-restricted sum (the CUDA path
needs a GPU); what is under test is the host-side plan: the ranks' blocks partition the particles, the all-gather
into preallocated buffers rebuilds the replicated SoA array, and the sharded evaluation equals the unsharded one bit
for bit."""
import os
import socket

import numpy as np
import pytest

from paper_1811_05903_b200 import shard, synth


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world,n", [(1, 7), (2, 4096), (3, 1000), (8, 1048576), (5, 3)])
def test_i_ranges_tile_the_particles(world, n):
    ranges = shard.all_ranges(world, n)
    assert ranges[0][0] == 0 and ranges[-1][1] == n
    for (b0, e0), (b1, e1) in zip(ranges, ranges[1:]):
        assert e0 == b1 and e0 >= b0
    base, rem = divmod(n, world)
    assert ranges[0][1] - ranges[0][0] == base + rem          # the main rank takes mod(N, P) (L139)
    assert all(e - b == base for b, e in ranges[1:])


@pytest.mark.parametrize("world,n", [(1, 7), (2, 4096), (3, 10000), (8, 1048576), (5, 3), (3, 2048 * 7 + 5)])
def test_round_robin_blocks_partition_the_particles(world, n):
    seen = np.concatenate([shard.owned_indices(r, world, n) for r in range(world)])
    assert np.array_equal(np.sort(seen), np.arange(n))
    counts = [shard.owned_count(r, world, n) for r in range(world)]
    assert sum(counts) == n and max(counts) - min(counts) <= shard.BLOCK
    for r in range(world):
        assert all(b % world == r for b in shard.owned_blocks(r, world, n))
        assert len(shard.owned_indices(r, world, n)) == counts[r]


def _worker(rank: int, world: int, port: int, n: int, out_dir: str) -> None:
    import torch
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import steps_oracle as oracle
        ps = synth.g0(n, seed=77)                              # identical on every rank (seeded)
        idx = shard.owned_indices(rank, world, n)
        gather = shard.Gather(world, n, "cpu", torch.float64)
        x_all = torch.from_numpy(ps.pos.copy())
        for step in range(2):                                  # twice: the buffers are reused, nothing is reallocated
            # one "step": every rank moves ITS particles (a stand-in drift), the slices are all-gathered ...
            x_local = x_all[:, idx] * (1.0 + 1e-3 * (rank + 1))
            ptr = gather.recv.data_ptr()
            gather(x_local, x_all)
            assert gather.recv.data_ptr() == ptr
        # ... and every rank evaluates the forces of its blocks against ALL sources
        pos = np.ascontiguousarray(x_all.numpy())
        acc_local = oracle.forces(pos, ps.mass, ps.soft, idx=idx)
        np.save(os.path.join(out_dir, f"pos_{rank}.npy"), pos)
        np.save(os.path.join(out_dir, f"acc_{rank}.npy"), acc_local)
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,n", [(2, 5001), (3, 9000)])
def test_sharded_step_equals_unsharded(world, n, tmp_path, oracle):
    import torch.multiprocessing as mp

    port = _free_port()
    mp.spawn(_worker, args=(world, port, n, str(tmp_path)), nprocs=world, join=True)
    ps = synth.g0(n, seed=77)
    expect_pos = ps.pos.copy()
    for _ in range(2):
        for r in range(world):
            expect_pos[:, shard.owned_indices(r, world, n)] *= 1.0 + 1e-3 * (r + 1)
    full = oracle.forces(expect_pos, ps.mass, ps.soft)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"pos_{r}.npy"), expect_pos), f"rank {r}: gathered positions"
        assert np.array_equal(np.load(tmp_path / f"acc_{r}.npy"), full[:, shard.owned_indices(r, world, n)]), f"rank {r}: forces"


class _FakeSteps:
    """Stand-in for the ctypes binding on CPU: the rank's share of the work is played by the oracle's sum over the
    sources j = rank (mod world) (the other sources' masses set to zero) -- a partition of the pair evaluations whose
    parts add up to the full sum, like steps_forces_share's; the kick/drift is a plain linear update."""

    def __init__(self, oracle):
        self.oracle = oracle

    def steps_forces_share(self, pos, mass, soft, rank, world, acc_part, mixed=False):
        import torch
        m = mass.numpy().copy()
        m[np.arange(m.size) % world != rank] = 0.0
        acc_part.copy_(torch.from_numpy(self.oracle.forces(np.ascontiguousarray(pos.numpy()), m, soft.numpy())))

    def steps_kick_drift(self, x, v, a, coeffs):
        v.add_(a, alpha=coeffs)
        x.add_(v, alpha=coeffs)


def _share_worker(rank: int, world: int, port: int, n: int, out_dir: str) -> None:
    import torch
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import steps_oracle as oracle
        ps = synth.g0(n, seed=78)
        pos, mass, soft = (torch.from_numpy(a.copy()) for a in (ps.pos, ps.mass, ps.soft))
        sh = shard.WorkSharedStep(_FakeSteps(oracle), rank, world, pos, torch.zeros_like(pos), mass, soft, False)
        sh.forces()
        ptr = sh.a.data_ptr()
        for _ in range(2):
            sh.step(1.0e-2)
        assert sh.a.data_ptr() == ptr                          # reduced in place, nothing reallocated
        np.save(os.path.join(out_dir, f"x_{rank}.npy"), sh.x.numpy())
        np.save(os.path.join(out_dir, f"a_{rank}.npy"), sh.a.numpy())
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,n", [(2, 3001), (3, 2500)])
def test_work_shared_step_equals_unsharded(world, n, tmp_path, oracle):
    """shard.WorkSharedStep over gloo: every rank advances all particles, evaluates its share of the pair evaluations and
    the partial accelerations are summed by one all-reduce; all ranks end bit-identical, and equal to the unsharded run to
    the rounding of the sum of the parts."""
    import torch.multiprocessing as mp

    port = _free_port()
    mp.spawn(_share_worker, args=(world, port, n, str(tmp_path)), nprocs=world, join=True)
    ps = synth.g0(n, seed=78)
    x, v = ps.pos.copy(), np.zeros_like(ps.pos)
    a = oracle.forces(x, ps.mass, ps.soft)
    for _ in range(2):
        v += 1.0e-2 * a
        x += 1.0e-2 * v
        a = oracle.forces(x, ps.mass, ps.soft)
    x0, a0 = np.load(tmp_path / "x_0.npy"), np.load(tmp_path / "a_0.npy")
    for r in range(1, world):
        assert np.array_equal(np.load(tmp_path / f"x_{r}.npy"), x0) and np.array_equal(np.load(tmp_path / f"a_{r}.npy"), a0)
    assert np.max(np.abs(x0 - x)) <= 1e-12 * np.max(np.abs(x))
    assert np.max(np.linalg.norm(a0 - a, axis=0) / np.linalg.norm(a, axis=0)) <= 1e-11
