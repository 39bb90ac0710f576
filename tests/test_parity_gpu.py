"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json's north_star:
  fp64 path : max_i |a_gpu - a_ref|_2 / |a_ref|_2 <= 1e-12
  mixed path: RMS <= 2e-6, max <= 1e-4."""
import ctypes as C
import math

import numpy as np
import pytest

from paper_1811_05903_b200 import synth

pytestmark = pytest.mark.gpu

FP64_MAX = 1e-12
MIXED_RMS, MIXED_MAX = 2e-6, 1e-4
LCDM = dict(H0=0.0288675134594813, Omega_m=0.3, Omega_r=0.0, Omega_L=0.7, Omega_k=0.0)


@pytest.fixture(scope="module")
def S():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1811_05903_b200 import steps
    steps.lib()
    return steps


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def gpu_forces(S, ps_or_arrays, mixed, idx=None):
    import torch
    pos, mass, soft = (ps_or_arrays.pos, ps_or_arrays.mass, ps_or_arrays.soft) if hasattr(ps_or_arrays, "pos") else ps_or_arrays
    dpos, dm, dh = dev(pos), dev(mass), dev(soft)
    acc = torch.full_like(dpos, float("nan"))
    (S.steps_forces_mixed if mixed else S.steps_forces)(dpos, dm, dh, acc)
    torch.cuda.synchronize()
    out = acc.cpu().numpy()
    return out if idx is None else out[:, idx]


def rel_err(got, ref):
    return np.linalg.norm(got - ref, axis=0) / np.linalg.norm(ref, axis=0)


def check(got, ref, mixed, label=""):
    assert np.all(np.isfinite(got)), label
    e = rel_err(got, ref)
    print(f"[{label} {'mixed' if mixed else 'fp64'}] rms {math.sqrt(np.mean(e * e)):.3e} max {e.max():.3e}")
    if mixed:
        rms = math.sqrt(np.mean(e * e))
        assert rms <= MIXED_RMS and e.max() <= MIXED_MAX, f"{label}: mixed rms {rms:.3e} max {e.max():.3e}"
    else:
        assert e.max() <= FP64_MAX, f"{label}: fp64 max {e.max():.3e} (rms {math.sqrt(np.mean(e*e)):.3e})"
    return e


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_config0_forces(S, oracle, mixed):
    ps = synth.config(0)
    check(gpu_forces(S, ps, mixed), oracle.forces(ps.pos, ps.mass, ps.soft), mixed, "config0")


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_config1_forces_65536(S, oracle, mixed, request):
    ps = synth.config(1)
    ref = _oracle_cached(oracle, ps, "c1")
    check(gpu_forces(S, ps, mixed), ref, mixed, "config1")


_CACHE = {}


def _oracle_cached(oracle, ps, key, idx=None):
    if key not in _CACHE:
        _CACHE[key] = oracle.forces(ps.pos, ps.mass, ps.soft, idx=idx)
    return _CACHE[key]


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
@pytest.mark.parametrize("eps0", [0.1, 1.0])
def test_softening_stress(S, oracle, mixed, eps0):
    """h_min inflated 10x / 100x: thousands of pairs in both softened branches of Eq. 4."""
    ps = synth.g0(4096, seed=77, eps0=eps0)
    d = ps.pos[:, :, None] - ps.pos[:, None, :512]
    u = np.linalg.norm(d, axis=0) / (ps.soft[:, None] + ps.soft[None, :512])
    assert ((u > 0) & (u < 0.5)).sum() > 50 and ((u >= 0.5) & (u < 1)).sum() > 200
    check(gpu_forces(S, ps, mixed), oracle.forces(ps.pos, ps.mass, ps.soft), mixed, f"stress eps0={eps0}")


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
@pytest.mark.parametrize("n", [1, 2, 3, 31, 255, 256, 257, 1000, 1025, 2049, 5000])
def test_ragged_sizes(S, oracle, mixed, n):
    ps = synth.g0(n, seed=1000 + n, eps0=0.05)
    got = gpu_forces(S, ps, mixed)
    if n == 1:
        assert np.all(got == 0.0)
        return
    check(got, oracle.forces(ps.pos, ps.mass, ps.soft), mixed, f"n={n}")


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_unsorted_input_is_still_correct(S, oracle, mixed):
    ps = synth.g0(6000, seed=5, sort=False)
    perm = np.random.default_rng(3).permutation(ps.n)
    arrays = (np.ascontiguousarray(ps.pos[:, perm]), ps.mass[perm].copy(), ps.soft[perm].copy())
    check(gpu_forces(S, arrays, mixed), oracle.forces(*arrays), mixed, "unsorted")


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_coincident_particles_and_zero_softening(S, oracle, mixed):
    rng = np.random.default_rng(9)
    pos = rng.normal(size=(3, 600))
    pos[:, 100] = pos[:, 7]                     # a coincident distinct pair (reading #4: contributes 0)
    mass = rng.uniform(0.5, 1.5, 600)
    soft = np.full(600, 0.05)
    check(gpu_forces(S, (pos, mass, soft), mixed), oracle.forces(pos, mass, soft), mixed, "coincident")
    soft0 = np.zeros(600)                       # pure Newtonian: h = 0 everywhere, self pair still skipped
    pos2 = rng.normal(size=(3, 600))
    check(gpu_forces(S, (pos2, mass, soft0), mixed), oracle.forces(pos2, mass, soft0), mixed, "h=0")


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_config2_zoom_core_sampled(S, oracle, mixed):
    ps = synth.config(2)
    assert ps.soft.max() / ps.soft.min() >= 100.0
    idx = synth.stratified_sample(ps.n, 2048)
    ref = _oracle_cached(oracle, ps, "c2", idx)
    check(gpu_forces(S, ps, mixed, idx), ref, mixed, "config2")


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_config3_one_million_sampled(S, oracle, mixed):
    """Full BASELINE size, in the launch configuration bench.py times (fp64: band + pair-symmetric items); oracle on the
    stratified sample SURVEY.md 8(d) / BASELINE.md name: 16,384 i-particles (innermost 1,024 + outermost 1,024 + the rest
    uniform in index) x all 1,048,576 sources."""
    ps = synth.config(3)
    idx = synth.stratified_sample(ps.n, 16384, n_edge=1024)
    assert len(idx) >= 16000 and idx[1023] == 1023 and idx[-1024] == ps.n - 1024
    ref = _oracle_cached(oracle, ps, "c3", idx)
    check(gpu_forces(S, ps, mixed, idx), ref, mixed, "config3")


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
@pytest.mark.parametrize("case", ["ragged", "unsorted", "massless", "massless_mid", "stale_order", "one_sided"])
def test_pair_symmetric_path_and_its_fallbacks(S, oracle, mixed, case):
    """N >= 131,072 takes the pair-symmetric route (band + every far block pair once).  Against the oracle on a sample:
    ragged     N = 150,001: the last block holds 497 particles, the rest of its tiles are pads;
    unsorted   a random permutation: no block pair is far, every row's band reaches the last block and everything runs
               one-sided;
    massless   three tracer particles (m = 0): their reaction sums could not be divided by m_j, so their tiles are marked
               and the device falls back in the same way (one of them sits in the first block) -- the tracers still feel
               the others;
    massless_mid one tracer in the middle block: that block is "not far" from any other, so the rows before it have bands
               that reach it (rows of very different widths), the rows after it have no items, and only the block pairs
               (b, c) with b before and c after the tracer's block stay symmetric items;
    stale_order every particle moved radially by up to 3 % (an order several steps old): wider bands, different from row
               to row;
    one_sided  the "sym" option off: the one-sided kernels at this size, same answer to rounding."""
    import torch
    n = 150001 if case == "ragged" else 139264
    ps = synth.g0(n, seed=4242)
    pos, mass, soft = ps.pos.copy(), ps.mass.copy(), ps.soft.copy()
    rng = np.random.default_rng(17)
    if case == "unsorted":
        perm = rng.permutation(n)
        pos, mass, soft = np.ascontiguousarray(pos[:, perm]), mass[perm].copy(), soft[perm].copy()
    elif case == "massless":
        mass[[5, n // 2, n - 3]] = 0.0
    elif case == "massless_mid":
        mass[n // 2] = 0.0
    elif case == "stale_order":
        pos = np.ascontiguousarray(pos * (1.0 + 0.03 * rng.uniform(-1.0, 1.0, size=n)))
    idx = np.unique(np.concatenate([synth.stratified_sample(n, 1536), [5, n // 2, n - 3]]))
    ref = oracle.forces(pos, mass, soft, idx=idx)
    if case == "one_sided":
        S.steps_set_option("sym", 0)
    try:
        got = gpu_forces(S, (pos, mass, soft), mixed, idx)
    finally:
        S.steps_set_option("sym", 1)
    check(got, ref, mixed, f"sym/{case}")


@pytest.mark.parametrize("mixed,n", [(False, 16385), (False, 24577), (True, 30721), (True, 40001), (True, 50001)],
                         ids=["fp64-16385", "fp64-24577", "mixed-30721", "mixed-40001", "mixed-50001"])
def test_pair_symmetric_route_at_its_smallest_sizes(S, oracle, mixed, n):
    """The smallest sizes of the pair-symmetric route, all ragged: fp64 from 9 blocks (items in 16 parts), mixed from 16 blocks
    (4 parts per item up to 23 blocks, whole items from 24); the band of these sizes runs on the split-j driver.  Against
    the oracle on a sample; the same bits on a second run; the one-sided evaluation to summation-order rounding."""
    assert S.steps_pair_symmetric(n, mixed) == 1
    if n in (16385, 30721):                     # the thresholds themselves
        assert S.steps_pair_symmetric(n - 1, mixed) == 0
    ps = synth.g0(n, seed=5150 + n)
    idx = synth.stratified_sample(n, 1024)
    ref = oracle.forces(ps.pos, ps.mass, ps.soft, idx=idx)
    got = gpu_forces(S, ps, mixed)
    check(got[:, idx], ref, mixed, f"sym-min n={n}")
    assert np.array_equal(got, gpu_forces(S, ps, mixed))
    S.steps_set_option("sym", 0)
    try:
        one = gpu_forces(S, ps, mixed)
    finally:
        S.steps_set_option("sym", 1)
    assert rel_err(got, one).max() <= (1e-4 if mixed else 1e-13)


def test_newtons_third_law_and_determinism_on_device(S):
    import torch
    ps = synth.config(1)
    a1 = gpu_forces(S, ps, False)
    a2 = gpu_forces(S, ps, False)
    assert np.array_equal(a1, a2)               # bitwise run-to-run
    m1, m2 = gpu_forces(S, ps, True), gpu_forces(S, ps, True)
    assert np.array_equal(m1, m2)
    net = np.linalg.norm(a1 @ ps.mass) / np.sum(ps.mass * np.linalg.norm(a1, axis=0))
    assert net < 1e-13


def test_sass_reuse_patch_is_bit_identical(S):
    """The post-link operand-reuse pass (sass_reuse.py) only sets hint bits: the product library and a build of the same
    sources without the pass must give bit-identical forces.  Config 1 (both paths, asymmetric kernels) and g0(131,072)
    in fp64 (band + pair-symmetric kernel)."""
    import torch
    from paper_1811_05903_b200 import build
    info = S.build_info()
    assert info["sass_reuse"] == "applied" and info["sass_reuse_patched_instructions"] >= 40, info
    U = S.load_library(build.build_unpatched())
    for n, paths in ((65536, (False, True)), (131072, (False,))):
        ps = synth.g0(n, synth.SEED_BASE + 1)
        dpos, dm, dh = dev(ps.pos), dev(ps.mass), dev(ps.soft)
        st = torch.cuda.current_stream().cuda_stream
        for mixed in paths:
            a, b = torch.empty_like(dpos), torch.empty_like(dpos)
            (S.steps_forces_mixed if mixed else S.steps_forces)(dpos, dm, dh, a)
            fn = U.steps_forces_mixed if mixed else U.steps_forces
            assert fn(dpos.data_ptr(), dm.data_ptr(), dh.data_ptr(), n, b.data_ptr(), st) == 0
            torch.cuda.synchronize()
            assert torch.equal(a, b), f"N={n} mixed={mixed}: patched and unpatched libraries differ"
    # the periodic kernels get the hints too: group ring (N = 20,000), pair-symmetric route (40,001 fp64 / 150,001 mixed)
    L = 1.0
    for n, paths in ((20000, (False, True)), (40001, (False,)), (150001, (True,))):
        pos, mass, soft = synth.periodic_box(n, L, 4400 + n)
        dpos, dm, dh = dev(pos), dev(mass), dev(soft)
        st = torch.cuda.current_stream().cuda_stream
        for mixed in paths:
            a, b = torch.empty_like(dpos), torch.empty_like(dpos)
            S.steps_forces_quasi_periodic(dpos, dm, dh, L, a, mixed=mixed)
            assert U.steps_forces_quasi_periodic(dpos.data_ptr(), dm.data_ptr(), dh.data_ptr(), n, L, b.data_ptr(), int(mixed), st) == 0
            torch.cuda.synchronize()
            assert torch.equal(a, b), f"quasi-periodic N={n} mixed={mixed}: patched and unpatched libraries differ"
    U.steps_shutdown()


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_simple_driver_cross_check(S, oracle, mixed):
    """The one-CTA-per-i-block driver (plain loads) and the persistent TMA stream-K driver share the
    pair bodies; both must meet the bar and agree to summation-order rounding."""
    ps = synth.g0(20000, seed=31, eps0=0.03)
    ref = oracle.forces(ps.pos, ps.mass, ps.soft)
    S.steps_set_option("sym", 0)                # (the fp64 path is pair-symmetric from 16,385 particles: this test is about the ring driver)
    try:
        fast = gpu_forces(S, ps, mixed)
    finally:
        S.steps_set_option("sym", 1)
    check(gpu_forces(S, ps, mixed), ref, mixed, "default route")
    S.steps_set_option("driver", 1)
    try:
        simple = gpu_forces(S, ps, mixed)
    finally:
        S.steps_set_option("driver", 0)
    check(fast, ref, mixed, "persistent")
    check(simple, ref, mixed, "simple")
    assert rel_err(simple, fast).max() <= (1e-6 if mixed else 1e-14)


def test_forces_range_and_host_entry_points(S, oracle):
    import torch
    ps = synth.g0(5000, seed=21)
    full = gpu_forces(S, ps, False)
    dpos, dm, dh = dev(ps.pos), dev(ps.mass), dev(ps.soft)
    # The whole range is bit-identical to steps_forces.  A sub-range is summed in another order (the split-j driver sizes
    # its work units by the number of 128-particle groups, the ring driver cuts the tile stream by the number of
    # i-blocks), and a range that is not aligned to the groups may evaluate a Newtonian pair through the other body
    # (scaled far / plain near): rounding-level differences, far inside the 1e-12 parity bar.
    for (b, e) in [(0, 5000), (1024, 5000), (2048, 4096), (0, 1), (4999, 5000), (1000, 3077), (2048, 2049)]:
        out = torch.empty(3 * (e - b), dtype=torch.float64, device="cuda")
        S.steps_forces_range(dpos, dm, dh, b, e, out, mixed=False)
        torch.cuda.synchronize()
        got = out.cpu().numpy().reshape(3, e - b)
        if (b, e) == (0, ps.n):
            assert np.array_equal(got, full), (b, e)
        else:
            assert rel_err(got, full[:, b:e]).max() <= 1e-13, (b, e)
    acc_h = np.empty((3, ps.n))
    S.steps_forces_host(ps.pos, ps.mass, ps.soft, acc_h, mixed=False)
    assert np.array_equal(acc_h, full)
    acc_m = np.empty((3, ps.n))
    S.steps_forces_host(ps.pos, ps.mass, ps.soft, acc_m, mixed=True)
    check(acc_m, oracle.forces(ps.pos, ps.mass, ps.soft), True, "host mixed")
    L = S.lib()
    assert L.steps_forces(dpos.data_ptr(), dm.data_ptr(), dh.data_ptr(), 0, dpos.data_ptr(), None) == S.EINVAL
    assert L.steps_forces(dpos.data_ptr() + 8, dm.data_ptr(), dh.data_ptr(), 10, dpos.data_ptr(), None) == S.EINVAL
    assert L.steps_forces_range(dpos.data_ptr(), dm.data_ptr(), dh.data_ptr(), 5000, 10, 10, dpos.data_ptr(), 0, None) == S.EINVAL


def test_radial_sort_permute_and_near_fraction(S, oracle):
    """Row a0: steps_sort_radial orders by |x| (checked against numpy, not against itself), steps_permute applies it, the
    forces of the re-ordered set are the permuted forces of the original one (to the oracle bar), and the share of
    (i-group, tile) pairs that need the per-pair softening test collapses with the order (steps_near_fraction)."""
    import torch
    n = 30011
    ps = synth.g0(n, seed=31, sort=False)
    shuffle = np.random.default_rng(5).permutation(n)
    pos, mass, soft = np.ascontiguousarray(ps.pos[:, shuffle]), ps.mass[shuffle].copy(), ps.soft[shuffle].copy()
    dpos, dm, dh = dev(pos), dev(mass), dev(soft)
    perm = torch.empty(n, dtype=torch.int64, device="cuda")
    S.steps_sort_radial(dpos, perm)
    p = perm.cpu().numpy()
    assert np.array_equal(np.sort(p), np.arange(n))
    r = np.linalg.norm(pos, axis=0)
    assert np.all(np.diff(r[p]) >= -4e-16 * r[p][1:])          # ascending up to the rounding of the fp64 keys
    spos, sm, sh = torch.empty_like(dpos), torch.empty_like(dm), torch.empty_like(dh)
    S.steps_permute(dpos, perm, spos); S.steps_permute(dm, perm, sm); S.steps_permute(dh, perm, sh)
    assert np.array_equal(spos.cpu().numpy(), pos[:, p]) and np.array_equal(sm.cpu().numpy(), mass[p])
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    S.steps_near_fraction(dpos, dm, dh, out); unsorted = out.cpu().numpy().copy()
    S.steps_near_fraction(spos, sm, sh, out); ordered = out.cpu().numpy().copy()
    print(f"near (i-group, tile) pairs: unsorted {unsorted[0] / unsorted[1]:.3f}, radially sorted {ordered[0] / ordered[1]:.4f}")
    assert unsorted[1] == ordered[1] == -(-n // 128) * -(-n // 256)
    assert unsorted[0] / unsorted[1] > 0.9 and ordered[0] / ordered[1] < 0.1
    a_un, a_so = torch.empty_like(dpos), torch.empty_like(dpos)
    S.steps_forces(dpos, dm, dh, a_un); S.steps_forces(spos, sm, sh, a_so)
    ref = oracle.forces(pos, mass, soft)
    check(a_un.cpu().numpy(), ref, False, "unsorted")
    check(a_so.cpu().numpy(), ref[:, p], False, "sorted by the library")


@pytest.mark.parametrize("n", [1, 257, 2049, 5000, 20001, 40001, 140001])
def test_outputs_stay_inside_their_buffers(S, n):
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizer.md), so out-of-bounds writes are looked for with
    guard regions: every output buffer sits between two sentinel-filled pads that must come back untouched, for every
    force entry point and the O(N) kernels, at ragged sizes (N not a multiple of the tile / group / block)."""
    import torch
    ps = synth.g0(n, seed=900 + n, eps0=0.05)
    dpos, dm, dh = dev(ps.pos), dev(ps.mass), dev(ps.soft)
    pad, sentinel = 4096, -1.2345e300
    big = torch.full((3 * n + 2 * pad,), sentinel, dtype=torch.float64, device="cuda")
    acc = big[pad:pad + 3 * n]

    def intact():
        torch.cuda.synchronize()
        return bool((big[:pad] == sentinel).all()) and bool((big[pad + 3 * n:] == sentinel).all())

    for call in (lambda: S.steps_forces(dpos, dm, dh, acc), lambda: S.steps_forces_mixed(dpos, dm, dh, acc),
                 lambda: S.steps_forces_quasi_periodic(dpos, dm, dh, 50.0, acc),
                 lambda: S.steps_forces_quasi_periodic(dpos, dm, dh, 50.0, acc, mixed=True),
                 lambda: S.steps_forces_share(dpos, dm, dh, 1, 3, acc), lambda: S.steps_forces_share(dpos, dm, dh, 0, 2, acc, mixed=True)):
        call()
        assert intact() and bool(torch.isfinite(acc).all())
    if n <= 5000:
        S.steps_forces_periodic(dpos, dm, dh, 50.0, acc)
        assert intact() and bool(torch.isfinite(acc).all())
    if n > 1:                                                   # a sub-range and a block-strided set, packed outputs
        b, e = n // 3, n - 1
        big.fill_(sentinel)
        S.steps_forces_range(dpos, dm, dh, b, e, big[pad:pad + 3 * (e - b)], mixed=False)
        torch.cuda.synchronize()
        assert bool((big[:pad] == sentinel).all()) and bool((big[pad + 3 * (e - b):] == sentinel).all())
        from paper_1811_05903_b200 import shard
        cnt = shard.owned_count(1, 2, n)
        if cnt:
            big.fill_(sentinel)
            S.steps_forces_blocks(dpos, dm, dh, 1, 2, big[pad:pad + 3 * cnt], mixed=True)
            torch.cuda.synchronize()
            assert bool((big[:pad] == sentinel).all()) and bool((big[pad + 3 * cnt:] == sentinel).all())
            assert bool(torch.isfinite(big[pad:pad + 3 * cnt]).all())


@pytest.mark.parametrize("world", [2, 3, 8])
@pytest.mark.parametrize("mixed,n", [(False, 65536), (False, 4096), (True, 150001), (True, 40001)],
                         ids=["fp64-65536", "fp64-4096", "mixed-150001", "mixed-40001"])
def test_work_shares_sum_to_the_full_evaluation(S, oracle, mixed, n, world):
    """steps_forces_share: the pair evaluations of one force evaluation cut into `world` equal parts (band visits and
    pair-symmetric items); the sum of the parts' partial accelerations is the full result to rounding (each part is
    rounded to fp64 once; the parts of a particle's acceleration can be much larger than their sum, hence the bound
    relative to sum_j |f_ij|), each part is bit-reproducible, and the sum matches the oracle on a sample."""
    import torch
    ps = synth.g0(n, seed=3100 + n)
    dpos, dm, dh = dev(ps.pos), dev(ps.mass), dev(ps.soft)
    full = torch.empty(3, n, dtype=torch.float64, device="cuda")
    (S.steps_forces_mixed if mixed else S.steps_forces)(dpos, dm, dh, full)
    total = torch.zeros_like(full)
    part, again = torch.empty_like(full), torch.empty_like(full)
    norms = []
    for r in range(world):
        S.steps_forces_share(dpos, dm, dh, r, world, part, mixed=mixed)
        if r == world - 1:
            S.steps_forces_share(dpos, dm, dh, r, world, again, mixed=mixed)
            assert torch.equal(part, again)
        norms.append(float(part.norm()))
        total += part
    scale = full.norm(dim=0)
    d = ((total - full).norm(dim=0) / scale).cpu().numpy()
    print(f"[work shares n={n} world={world} {'mixed' if mixed else 'fp64'}] sum vs full: rms {math.sqrt(np.mean(d ** 2)):.3e} "
          f"max {d.max():.3e}; |part| {['%.3e' % v for v in norms]}")
    assert d.max() <= (2e-6 if mixed else 2e-13)
    if S.steps_pair_symmetric(n, mixed):
        assert min(norms) > 0.0                                   # every rank has work
    idx = synth.stratified_sample(n, 256)
    ref = oracle.forces(ps.pos, ps.mass, ps.soft, idx=idx)
    e = rel_err(total.cpu().numpy()[:, idx], ref)
    assert e.max() <= (1e-4 if mixed else 1e-12)


@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_work_shared_step_on_one_gpu_equals_unsharded(S, mixed):
    """bench.py's N > 1 step with the work-shared force evaluation (shard.WorkSharedStep) played on ONE GPU, rank after
    rank, the all-reduce replaced by adding the ranks' partials: two steps reproduce steps_kdk_step."""
    import torch
    from paper_1811_05903_b200 import shard
    n, world = (150001 if mixed else 40001), 3
    ps = synth.g0(n, seed=3300 + n)
    dpos, dm, dh = dev(ps.pos), dev(ps.mass), dev(ps.soft)
    co = S.KdkCoeffs(1.0, 0.0, 0.98, 1.0e-3, 2.0e-3, 1.0 / ps.r_cut ** 3, int(mixed))
    x, v, a = dpos.clone(), torch.zeros_like(dpos), torch.empty_like(dpos)
    (S.steps_forces_mixed if mixed else S.steps_forces)(x, dm, dh, a)
    ranks = [shard.WorkSharedStep(S, r, world, dpos, torch.zeros_like(dpos), dm, dh, mixed) for r in range(world)]

    def all_forces():
        for sh in ranks:
            sh.forces_part()
        total = sum(sh.a for sh in ranks)
        for sh in ranks:
            sh.a.copy_(total)

    all_forces()
    for _ in range(2):
        S.steps_kdk_step(x, v, a, dm, dh, co)
        for sh in ranks:
            sh.kick_drift(co)
        all_forces()
    for sh in ranks[1:]:
        assert torch.equal(sh.x, ranks[0].x) and torch.equal(sh.v, ranks[0].v)
    da = float(((ranks[0].a - a).norm(dim=0) / a.norm(dim=0)).max())
    dx = float((ranks[0].x - x).abs().max())
    print(f"[work-shared step {'mixed' if mixed else 'fp64'}] acc {da:.3e} x {dx:.3e}")
    assert da <= (5e-6 if mixed else 5e-13) and dx <= 1e-12


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_sharded_step_on_one_gpu_equals_unsharded(S, mixed, world):
    """bench.py's N > 1 step (shard.ShardedStep: kick/drift of the rank's particles, exchange, steps_forces_blocks of the
    rank's round-robin blocks) played on ONE GPU, rank after rank, with the all-gather replaced by copying every rank's
    particles into the replicated array: two steps must reproduce the unsharded steps_kdk_step to the
    summation-order difference of the stream-K split, which cuts the i-blocks' tile ranges differently when a rank holds
    fewer blocks (accelerations after two steps: fp64 < 1e-13, mixed < 1e-12 -- measured 1.2e-14 / 2e-14 --; positions
    and velocities follow the accelerations of the first step)."""
    import torch
    from paper_1811_05903_b200 import shard
    n = 20000                                                   # 10 blocks, the last one ragged
    ps = synth.config4_ics(n, synth.SEED_BASE + 4, vel_factor=0.01)
    pos, vel, m, h = dev(ps.pos), dev(ps.vel), dev(ps.mass), dev(ps.soft)
    cosmo = S.Cosmology(**LCDM)
    sc = S.steps_kdk_schedule(1 / 51, 1e-3, 1.0, cosmo)
    co = S.KdkCoeffs(1.0, 0.0, sc["alpha_open"], sc["beta_open"], sc["gamma"], 1.25e-4, int(mixed))
    # unsharded reference
    x0, v0, a0 = pos.clone(), vel.clone(), torch.empty_like(pos)
    (S.steps_forces_mixed if mixed else S.steps_forces)(x0, m, h, a0)
    for _ in range(2):
        S.steps_kdk_step(x0, v0, a0, m, h, co)
    # the same with `world` ranks played one after the other
    ranks = [shard.ShardedStep(S, r, world, pos, vel, m, h, mixed) for r in range(world)]
    for sh in ranks:
        sh.forces()
    for _ in range(2):
        for sh in ranks:
            sh.kick_drift(co)
        for sh in ranks:                                       # the exchange: every rank receives every rank's particles
            for other in ranks:
                sh.x_all.index_copy_(1, other.index, other.x)
        for sh in ranks:
            sh.forces()
    torch.cuda.synchronize()
    x1, v1, a1 = torch.empty_like(x0), torch.empty_like(x0), torch.empty_like(x0)
    for sh in ranks:
        x1.index_copy_(1, sh.index, sh.x); v1.index_copy_(1, sh.index, sh.v); a1.index_copy_(1, sh.index, sh.a)
        assert torch.equal(sh.x_all, ranks[0].x_all)
    e = rel_err(a1.cpu().numpy(), a0.cpu().numpy())
    print(f"[sharded world={world} {'mixed' if mixed else 'fp64'}] acc vs unsharded: max rel {e.max():.2e}")
    assert e.max() <= (1e-12 if mixed else 1e-13)
    ev = rel_err(v1.cpu().numpy(), v0.cpu().numpy())
    assert np.abs(x1.cpu().numpy() - x0.cpu().numpy()).max() <= 1e-14 * np.abs(ps.pos).max()
    assert ev.max() <= 1e-12


def test_config0_one_kdk_step(S, oracle):
    """Config 0: one force evaluation plus one KDK step (first step of config 4's schedule, v = 0)."""
    import torch
    ps = synth.config(0)
    B = 1.0 / ps.r_cut ** 3
    dt = float(oracle.ln_a_schedule(1 / 51, 1.0, 200, LCDM)[0])
    pos, vel = ps.pos.copy(), ps.vel.copy()
    acc = oracle.forces(pos, ps.mass, ps.soft)
    a1 = oracle.kdk_step(pos, vel, acc, ps.mass, ps.soft, 1 / 51, dt, 1.0, B, LCDM)

    from paper_1811_05903_b200 import integrate
    dpos, dvel, dm, dh = dev(ps.pos), dev(ps.vel), dev(ps.mass), dev(ps.soft)
    dacc = torch.empty_like(dpos)
    S.steps_forces(dpos, dm, dh, dacc)
    a1_gpu = integrate.run_kdk(dpos, dvel, dacc, dm, dh, 1 / 51, [dt], S.Cosmology(**LCDM), 1.0, B)
    torch.cuda.synchronize()
    assert a1_gpu == pytest.approx(a1, rel=1e-14)
    np.testing.assert_allclose(dpos.cpu().numpy(), pos, rtol=1e-13, atol=1e-15)
    assert rel_err(dacc.cpu().numpy(), acc).max() <= FP64_MAX
    assert rel_err(dvel.cpu().numpy(), vel).max() <= 1e-11


def test_momentum_diagnostic(S, oracle):
    import torch
    ps = synth.config4_ics(10000, synth.SEED_BASE + 4, vel_factor=0.7)
    out = torch.empty(4, dtype=torch.float64, device="cuda")
    S.steps_momentum(dev(ps.vel), dev(ps.mass), out)
    want = oracle.momentum(ps.vel, ps.mass)
    got = out.cpu().numpy()
    assert got[3] == pytest.approx(want[3], rel=1e-13)
    assert np.linalg.norm(got[:3] - want[:3]) < 1e-14 * want[3]


def _config4(oracle, n):
    vf = oracle.hubble(1 / 51, LCDM) * oracle.growth_rate(1 / 51, LCDM)
    return synth.config4_ics(n, synth.SEED_BASE + 4, vel_factor=vf)


# ---- Eq. 12 (L113-116): adaptive global time step -----------------------------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("n", [1, 2, 255, 4096, 65536, 100003])
def test_timestep_matches_oracle(S, oracle, n):
    import torch
    ps = synth.config(0, n) if n >= 2 else synth.config(0, 1)
    rng = np.random.default_rng(1200 + n)
    acc = rng.normal(size=(3, n)) * 10.0 ** rng.uniform(-4, 2, n)
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    for coef, B, eps, dt_max in [(1.0, 0.0, 0.025, 1e30), (51.0 ** 3, 1.25e-4, 0.01, 1e30), (1.0, 1.25e-4, 0.025, 1e-6)]:
        S.steps_timestep(dev(ps.pos), dev(acc), dev(ps.soft), coef, B, eps, dt_max, out)
        want = oracle.timestep(ps.pos, acc, ps.soft, coef, B, eps, dt_max)
        # sqrt and divide are IEEE on both sides; the only freedom is FMA contraction inside |A_i| (<= 2 ulp)
        assert out.item() == pytest.approx(want, rel=4e-16), (n, coef, out.item(), want)
    # no acceleration anywhere: dt_max comes back exactly
    S.steps_timestep(dev(ps.pos), dev(0 * acc), dev(ps.soft), 1.0, 0.0, 0.025, 0.75, out)
    assert out.item() == 0.75


@pytest.mark.gpu
def test_adaptive_kdk_run_follows_the_oracle(S, oracle):
    """20 comoving KDK steps whose length is set by Eq. 12 from the forces of the previous step, library vs oracle:
    the step lengths agree to rounding and so do the trajectories."""
    import torch
    from paper_1811_05903_b200 import integrate
    ps = _config4(oracle, 2048)
    B, G, eps, dt_max = 1.0 / ps.r_cut ** 3, 1.0, 0.025, 0.5
    dpos, dvel, dm, dh = dev(ps.pos), dev(ps.vel), dev(ps.mass), dev(ps.soft)
    dacc = torch.empty_like(dpos)
    S.steps_forces(dpos, dm, dh, dacc)
    pos, vel = ps.pos.copy(), ps.vel.copy()
    acc = oracle.forces(pos, ps.mass, ps.soft)
    a_lib = a_ref = 1 / 51
    out = torch.empty(1, dtype=torch.float64, device="cuda")
    cosmo = S.Cosmology(**LCDM)
    for step in range(20):
        S.steps_timestep(dpos, dacc, dh, G / a_lib ** 3, B, eps, dt_max, out)
        dt_lib = out.item()
        dt_ref = oracle.timestep(pos, acc, ps.soft, G / a_ref ** 3, B, eps, dt_max)
        assert dt_lib == pytest.approx(dt_ref, rel=1e-11), step
        a_lib = integrate.run_kdk(dpos, dvel, dacc, dm, dh, a_lib, [dt_lib], cosmo, G, B)
        a_ref = oracle.kdk_step(pos, vel, acc, ps.mass, ps.soft, a_ref, dt_ref, G, B, LCDM)
    assert a_lib == pytest.approx(a_ref, rel=1e-11)
    s = (ps.mass * (4 * np.pi / 3) * ps.r_cut ** 3) ** (1 / 3)
    dx = np.linalg.norm(dpos.cpu().numpy() - pos, axis=0) / s
    print(f"adaptive run, 20 steps: a = {a_ref:.6f}, max |dx|/s library-vs-oracle {dx.max():.3e}")
    assert dx.max() < 1e-9


# ---- glass generation (section 3.1): reversed gravity + net-force residual --------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("n", [1, 3, 257, 65536, 100003])
def test_force_residual_matches_oracle(S, oracle, n):
    import torch
    rng = np.random.default_rng(3100 + n)
    pos = rng.normal(size=(3, n)) * 5.0
    acc = rng.normal(size=(3, n)) * 10.0 ** rng.uniform(-4, 1, n)
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    for B in (0.0, 1.25e-4, 0.37):
        S.steps_force_residual(dev(pos), dev(acc), B, out)
        want = oracle.force_residual(pos, acc, B)
        got = out.cpu().numpy()
        assert got[0] == pytest.approx(want[0], rel=1e-13), (n, B)     # plain fp64 tree sum vs compensated sum
        assert got[1] == pytest.approx(want[1], rel=4e-16), (n, B)


@pytest.mark.gpu
def test_glass_run_reversed_gravity_follows_the_oracle(S, oracle):
    """40 adaptive KDK steps with REVERSED gravity (G = -1) in an EdS background on the compactified g0 set (random on
    S^3, i.e. the starting point of glass making): the library follows the oracle step by step, and the net-force
    residual -- the quantity glass generation minimises -- goes down."""
    import torch
    from paper_1811_05903_b200 import integrate
    ps = synth.config(0, 2048)
    B = 1.0 / ps.r_cut ** 3
    eds = dict(H0=math.sqrt(2 * B), Omega_m=1.0, Omega_r=0.0, Omega_L=0.0, Omega_k=0.0)
    G, eps, dt_max, a0, n_steps = -1.0, 0.025, 1e30, 0.05, 40
    dpos, dvel, dm, dh = dev(ps.pos), dev(np.zeros_like(ps.pos)), dev(ps.mass), dev(ps.soft)
    dacc = torch.empty_like(dpos)
    S.steps_forces(dpos, dm, dh, dacc)
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    S.steps_force_residual(dpos, dacc, B, out)
    res0 = out.cpu().numpy().copy()
    a_lib, dts = integrate.run_adaptive(dpos, dvel, dacc, dm, dh, a0, n_steps, S.Cosmology(**eds), G, B, eps, dt_max)
    S.steps_force_residual(dpos, dacc, B, out)
    res1 = out.cpu().numpy().copy()

    pos, vel = ps.pos.copy(), np.zeros_like(ps.pos)
    acc = oracle.forces(pos, ps.mass, ps.soft)
    want0 = oracle.force_residual(pos, acc, B)
    a = a0
    for k in range(n_steps):
        dt = oracle.timestep(pos, acc, ps.soft, 1.0 / a ** 3, B, eps, dt_max)
        assert dts[k] == pytest.approx(dt, rel=1e-10), k
        a = oracle.kdk_step(pos, vel, acc, ps.mass, ps.soft, a, dt, G, B, eds)
    want1 = oracle.force_residual(pos, acc, B)
    assert a_lib == pytest.approx(a, rel=1e-11)
    assert res0[0] == pytest.approx(want0[0], rel=1e-12) and res1[0] == pytest.approx(want1[0], rel=1e-9)
    s = (ps.mass * (4 * np.pi / 3) * ps.r_cut ** 3) ** (1 / 3)
    dx = np.linalg.norm(dpos.cpu().numpy() - pos, axis=0) / s
    print(f"glass run, {n_steps} steps: a {a0} -> {a:.4f}, residual sum |g|^2 {want0[0]:.4e} -> {want1[0]:.4e}, "
          f"max |dx|/s library-vs-oracle {dx.max():.3e}")
    assert dx.max() < 1e-9
    assert res1[0] < res0[0]


# ---- Eq. 5 (L65-70): quasi-periodic boundary, leading image only ----------------------------------------------------
def _periodic_box(n, L, seed):
    """Constant-resolution periodic box (Eq. 6): equal masses, one softening length for every particle
    (1/30 of the mean spacing), positions uniform in the cube -- the state glass making starts from."""
    rng = np.random.default_rng(seed)
    pos = np.ascontiguousarray(rng.uniform(0, L, size=(3, n)))
    mass = np.full(n, 1.0 / n)
    soft = np.full(n, L / n ** (1 / 3) / 30)
    return pos, mass, soft


@pytest.mark.gpu
@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
@pytest.mark.parametrize("n,ordered", [(2, False), (257, False), (5000, False), (32768, False), (5000, True), (32768, True),
                                       (100003, True), (150001, True), (262144, True)])
def test_quasi_periodic_forces_match_oracle(S, oracle, mixed, n, ordered):
    """ordered: Morton (cell) order -- tile pairs share one image shift and most take the periodic far bodies (uniform
    shift / per-pair conditional wrap); unordered input goes through the general wrapped body for every tile."""
    import torch
    L = 1.7
    pos, mass, soft = _periodic_box(n, L, 5500 + n)
    if ordered:
        pos = np.ascontiguousarray(pos[:, synth.morton_order(pos, L)])
        if not mixed:                                          # positions need not lie inside [0, L) (the fp32 path loses
            pos[:, ::7] += np.array([[L], [-2 * L], [3 * L]])  # coordinate bits outside the box: steps.h)
    if n > 40000:                                              # oracle on a sample
        return _quasi_periodic_sampled(S, oracle, mixed, pos, mass, soft, L)
    if n == 2:                                   # the pair interacts through the boundary
        pos = np.array([[0.05 * L, 0.95 * L], [0.3, 0.3], [0.7, 0.7]])
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    S.steps_forces_quasi_periodic(dev(pos), dev(mass), dev(soft), L, acc, mixed=mixed)
    ref = oracle.forces_quasi_periodic(pos, mass, soft, L)
    e = rel_err(acc.cpu().numpy(), ref)
    rms = math.sqrt(np.mean(e ** 2))
    print(f"[quasi-periodic n={n} {'mixed' if mixed else 'fp64'}] rms {rms:.3e} max {e.max():.3e}")
    if mixed:
        # In a homogeneous periodic box the net force is the small remainder of pulls from all directions: with
        # kappa_i = sum_j |f_ij| / |sum_j f_ij| (10 ... 1e3 here, growing with N) the fp32 rounding of coordinates and
        # pair terms is amplified to ~kappa_i 2^-24 relative to the NET force, whatever the kernel does.  The bars of the
        # compactified configs (rms 2e-6, max 1e-4, BASELINE.json) are therefore applied to the error relative to the
        # pair-force scale sum_j |f_ij| (tolerance of the quasi-periodic row).
        fsum = _pair_force_abs_sum(pos, mass, soft, L)
        e_abs = np.linalg.norm(acc.cpu().numpy() - ref, axis=0) / fsum
        kappa = fsum / np.linalg.norm(ref, axis=0)
        print(f"    relative to sum_j |f_ij|: rms {math.sqrt(np.mean(e_abs ** 2)):.3e} max {e_abs.max():.3e}; kappa median "
              f"{np.median(kappa):.1f} max {kappa.max():.1f}")
        assert math.sqrt(np.mean(e_abs ** 2)) <= 2e-6 and e_abs.max() <= 1e-4
        # ... and the error relative to the NET force is bounded by the same bars times the measured amplification
        assert rms <= 2e-6 * math.sqrt(np.mean(kappa ** 2)) and e.max() <= 1e-4 * kappa.max()
    else:
        assert e.max() <= 1e-12


def _quasi_periodic_sampled(S, oracle, mixed, pos, mass, soft, L):
    import torch
    n = pos.shape[1]
    idx = synth.stratified_sample(n, 1024)
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    S.steps_forces_quasi_periodic(dev(pos), dev(mass), dev(soft), L, acc, mixed=mixed)
    got = acc.cpu().numpy()[:, idx]
    ref = oracle.forces_quasi_periodic(pos, mass, soft, L, idx=idx)
    fsum = _pair_force_abs_sum(pos, mass, soft, L, idx)
    e_abs = np.linalg.norm(got - ref, axis=0) / fsum
    e = rel_err(got, ref)
    print(f"[quasi-periodic n={n} sampled {'mixed' if mixed else 'fp64'}] to net force: max {e.max():.3e}; to sum_j|f_ij|: rms "
          f"{math.sqrt(np.mean(e_abs ** 2)):.3e} max {e_abs.max():.3e}")
    if mixed:
        assert math.sqrt(np.mean(e_abs ** 2)) <= 2e-6 and e_abs.max() <= 1e-4
    else:
        assert e.max() <= 1e-12


def _pair_force_abs_sum(pos, mass, soft, L, idx=None):
    """sum_j m_j |g(r_ij)| r_ij with leading-image separations, Newtonian magnitude (test-side scale only)."""
    n = pos.shape[1]
    sel = np.arange(n) if idx is None else np.asarray(idx)
    out = np.zeros(len(sel))
    for i0 in range(0, len(sel), 256):
        d = pos[:, None, :] - pos[:, sel[i0:i0 + 256], None]
        d -= L * np.rint(d / L)
        r2 = np.sum(d * d, axis=0)
        r2[r2 == 0] = np.inf
        out[i0:i0 + 256] = np.sum(mass[None, :] / np.maximum(r2, (2 * soft[0]) ** 2), axis=1)
    return out


@pytest.mark.gpu
@pytest.mark.parametrize("mixed,n", [(False, 18433), (False, 40001), (False, 150001), (True, 170001)],
                         ids=["fp64-18433", "fp64-40001", "fp64-150001", "mixed-170001"])
def test_quasi_periodic_pair_symmetric_route(S, mixed, n):
    """From 9 (fp64) / 80 (mixed) blocks the far meetings of two different blocks are evaluated once and applied to both
    groups (forces_sym_box_kernel), the possibly-softened units by forces_boxgen_kernel, the own blocks by the group-ring
    kernel.  Every pair must be evaluated by exactly one of them: the result equals the one-sided evaluation (option
    "sym" = 0: group-ring kernel alone) to rounding, is bit-identical run to run, and obeys Newton's third law."""
    import torch
    L = 1.3
    pos, mass, soft = _periodic_box(n, L, 7700 + n)
    rng = np.random.default_rng(n)
    mass = mass * rng.uniform(0.5, 2.0, size=n)                 # unequal masses: a swapped m_i / m_j would show
    mass /= mass.sum()
    soft = soft * rng.uniform(0.5, 3.0, size=n)                 # some groups with larger softening: more general units
    pos = np.ascontiguousarray(pos[:, synth.morton_order(pos, L)])
    dpos, dm, dh = dev(pos), dev(mass), dev(soft)
    a_sym, a_again, a_one = (torch.empty(3, n, dtype=torch.float64, device="cuda") for _ in range(3))
    assert S.steps_pair_symmetric(n, mixed) == 1
    S.steps_forces_quasi_periodic(dpos, dm, dh, L, a_sym, mixed=mixed)
    S.steps_forces_quasi_periodic(dpos, dm, dh, L, a_again, mixed=mixed)
    assert torch.equal(a_sym, a_again)
    try:
        S.steps_set_option("sym", 0)
        S.steps_forces_quasi_periodic(dpos, dm, dh, L, a_one, mixed=mixed)
    finally:
        S.steps_set_option("sym", 1)
    idx = synth.stratified_sample(n, 1024)
    fsum = _pair_force_abs_sum(pos, mass, np.full(n, soft.min()), L, idx)
    d = np.linalg.norm((a_sym - a_one).cpu().numpy()[:, idx], axis=0) / fsum
    print(f"[quasi-periodic sym vs one-sided n={n} {'mixed' if mixed else 'fp64'}] relative to sum_j|f_ij|: rms "
          f"{math.sqrt(np.mean(d ** 2)):.3e} max {d.max():.3e}")
    assert d.max() <= (2e-5 if mixed else 1e-13)
    dmass = torch.from_numpy(mass).cuda()
    p = (dmass * a_sym).sum(dim=1)
    assert float(p.norm()) < (1e-7 if mixed else 1e-13) * float((dmass * a_sym.norm(dim=0)).sum())


@pytest.mark.gpu
@pytest.mark.parametrize("mixed", [False, True], ids=["fp64", "mixed"])
def test_quasi_periodic_pair_symmetric_route_with_tracers_and_a_heavy_softened_group(S, oracle, mixed):
    """Edge cases of the periodic pair-symmetric route against the oracle: massless tracer particles (they feel forces but
    their reaction sums cannot be divided by m_j: their groups must stay out of the symmetric meetings), a block whose
    particles carry a softening of a tenth of the box (softened pairs far beyond the neighbouring cells), particles given
    outside [0, L) by whole periods (fp64), and N not a multiple of the group / tile / block."""
    import torch
    n = 150001 if mixed else 40001
    L = 2.5
    pos, mass, soft = _periodic_box(n, L, 8800 + n)
    pos = np.ascontiguousarray(pos[:, synth.morton_order(pos, L)])
    mass[[5, 2048 * 3 + 17, n - 1]] = 0.0                       # tracers
    soft[2048 * 5: 2048 * 5 + 300] = 0.05 * L                   # pair softening 0.1 L for 300 particles of block 5
    if not mixed:
        pos[:, 2048 * 7: 2048 * 7 + 40] += np.array([[2 * L], [-L], [0.0]])
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    assert S.steps_pair_symmetric(n, mixed) == 1
    S.steps_forces_quasi_periodic(dev(pos), dev(mass), dev(soft), L, acc, mixed=mixed)
    idx = np.unique(np.concatenate([synth.stratified_sample(n, 512), [5, 2048 * 3 + 17, n - 1], np.arange(2048 * 5, 2048 * 5 + 300, 7),
                                    np.arange(2048 * 7, 2048 * 7 + 40, 3)]))
    ref = oracle.forces_quasi_periodic(pos, mass, soft, L, idx=idx)
    got = acc.cpu().numpy()[:, idx]
    fsum = _pair_force_abs_sum(pos, mass, np.full(n, soft.min()), L, idx)
    e_abs = np.linalg.norm(got - ref, axis=0) / fsum
    print(f"[quasi-periodic edge cases n={n} {'mixed' if mixed else 'fp64'}] to sum_j|f_ij|: rms {math.sqrt(np.mean(e_abs ** 2)):.3e} max {e_abs.max():.3e}")
    assert np.isfinite(got).all()
    if mixed:
        assert math.sqrt(np.mean(e_abs ** 2)) <= 2e-6 and e_abs.max() <= 1e-4
    else:
        assert e_abs.max() <= 1e-13 and rel_err(got, ref).max() <= 1e-12


@pytest.mark.gpu
def test_quasi_periodic_translation_invariance_and_unwrapped_positions_on_device(S):
    """Shifting every particle by an arbitrary vector, without wrapping the positions back into [0, L), must leave the
    fp64 forces unchanged to rounding (the wrap acts on separations, not on positions)."""
    import torch
    L, n = 2.0, 20000
    pos, mass, soft = _periodic_box(n, L, 5601)
    a0 = torch.empty(3, n, dtype=torch.float64, device="cuda")
    a1 = torch.empty_like(a0)
    S.steps_forces_quasi_periodic(dev(pos), dev(mass), dev(soft), L, a0)
    moved = np.ascontiguousarray(pos + np.array([[3 * L + 0.37], [-5 * L - 0.11], [0.5 * L]]))
    S.steps_forces_quasi_periodic(dev(moved), dev(mass), dev(soft), L, a1)
    e = rel_err(a1.cpu().numpy(), a0.cpu().numpy())
    assert e.max() < 1e-9, e.max()              # positions carry ~1e-15 L absolute rounding after the shift
    # Newton's third law on the device
    p = (torch.from_numpy(mass).cuda() * a0).sum(dim=1)
    assert float(p.norm()) < 1e-13 * float((torch.from_numpy(mass).cuda() * a0.norm(dim=0)).sum())


# ---- device-resident adaptive stepping (8(f)-1, second half) ---------------------------------------------------------
def _oracle_adaptive(oracle, ps, vel0, cosmo, G, B, eps, dt_max, a0, n_steps):
    pos, vel = ps.pos.copy(), vel0.copy()
    acc = oracle.forces(pos, ps.mass, ps.soft)
    a, dts = a0, []
    for _ in range(n_steps):
        dt = oracle.timestep(pos, acc, ps.soft, abs(G) / a ** 3, B, eps, dt_max)
        a = oracle.kdk_step(pos, vel, acc, ps.mass, ps.soft, a, dt, G, B, cosmo)
        dts.append(dt)
    return pos, vel, a, dts


@pytest.mark.gpu
@pytest.mark.parametrize("mode", ["lcdm", "glass"])
def test_device_resident_adaptive_run_matches_oracle(S, oracle, mode):
    """steps_kdk_step_adaptive computes the step length (Eq. 12), a(t) (RK4) and the kick/drift coefficients on the
    device; 20 steps without any host round trip must land where the oracle's host-driven loop lands."""
    import torch
    n_steps, eps, dt_max = 20, 0.025, 0.5
    if mode == "lcdm":
        ps = _config4(oracle, 2048); vel0 = ps.vel; cosmo = LCDM; G = 1.0; a0 = 1 / 51
    else:
        ps = synth.config(0, 2048); vel0 = np.zeros_like(ps.pos); G = -1.0; a0 = 0.05
        cosmo = dict(H0=math.sqrt(2.0 / ps.r_cut ** 3), Omega_m=1.0, Omega_r=0.0, Omega_L=0.0, Omega_k=0.0)
    B = 1.0 / ps.r_cut ** 3
    dpos, dvel, dm, dh = dev(ps.pos), dev(vel0), dev(ps.mass), dev(ps.soft)
    dacc = torch.empty_like(dpos)
    S.steps_forces(dpos, dm, dh, dacc)
    state = torch.tensor([a0, 0.0, 1.0, 0.0, 0.0], dtype=torch.float64, device="cuda")
    c = S.Cosmology(**cosmo)
    for _ in range(n_steps):
        S.steps_kdk_step_adaptive(dpos, dvel, dacc, dm, dh, state, c, G, B, eps, dt_max)
    S.steps_kick_close_adaptive(dpos, dvel, dacc, state, B)
    st = state.cpu().numpy()
    pos, vel, a, dts = _oracle_adaptive(oracle, ps, vel0, cosmo, G, B, eps, dt_max, a0, n_steps)
    assert st[4] == n_steps and st[2] == 1.0 and st[3] == 0.0
    assert st[0] == pytest.approx(a, rel=1e-11) and st[1] == pytest.approx(dts[-1], rel=1e-9)
    s = (ps.mass * (4 * np.pi / 3) * ps.r_cut ** 3) ** (1 / 3)
    dx = np.linalg.norm(dpos.cpu().numpy() - pos, axis=0) / s
    dv = np.linalg.norm(dvel.cpu().numpy() - vel, axis=0) / np.maximum(np.linalg.norm(vel, axis=0), 1e-300)
    print(f"device-resident adaptive run [{mode}]: a = {a:.6f}, max |dx|/s {dx.max():.3e}, max |dv|/|v| {dv.max():.3e}")
    assert dx.max() < 1e-9 and dv.max() < 1e-8


@pytest.mark.gpu
@pytest.mark.parametrize("n,mixed", [(4096, False), (40000, False), (140000, True)])
def test_device_resident_steps_replay_from_a_cuda_graph(S, oracle, n, mixed):
    """Five adaptive steps captured ONCE in a CUDA graph and replayed four times give bit for bit the state of twenty
    eager calls: the whole step (time-step criterion, coefficients, kick/drift, tile prep, forces, reduce) is
    stream-ordered device work with no host dependence.  N = 4,096: split-j driver; 40,000: fp64 band + pair-symmetric
    sub-items; 140,000 mixed: band + pair-symmetric items -- their plan (band width, item count) is computed on the device
    inside the captured sequence.  Also: a call that would have to allocate workspace under capture is refused."""
    import torch
    ps = _config4(oracle, n)
    B, G, eps, dt_max, a0 = 1.0 / ps.r_cut ** 3, 1.0, 0.025, 0.5, 1 / 51
    c = S.Cosmology(**LCDM)
    dm, dh = dev(ps.mass), dev(ps.soft)

    def fresh():
        dpos, dvel = dev(ps.pos), dev(ps.vel)
        dacc = torch.empty_like(dpos)
        (S.steps_forces_mixed if mixed else S.steps_forces)(dpos, dm, dh, dacc)
        return dpos, dvel, dacc, torch.tensor([a0, 0.0, 1.0, 0.0, 0.0], dtype=torch.float64, device="cuda")

    pos_e, vel_e, acc_e, st_e = fresh()
    for _ in range(20):
        S.steps_kdk_step_adaptive(pos_e, vel_e, acc_e, dm, dh, st_e, c, G, B, eps, dt_max, mixed=mixed)
    torch.cuda.synchronize()

    pos_g, vel_g, acc_g, st_g = fresh()
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            for _ in range(5):
                S.steps_kdk_step_adaptive(pos_g, vel_g, acc_g, dm, dh, st_g, c, G, B, eps, dt_max, mixed=mixed)
            if n == 4096:                         # a larger N than any reserved so far would need cudaMalloc: refused
                big = 3 * 1024 * 1024 + 77
                z = torch.empty(0)                # never dereferenced: the call returns before any launch
                rc = S.lib().steps_forces(pos_g.data_ptr(), dm.data_ptr(), dh.data_ptr(), big, acc_g.data_ptr(), side.cuda_stream)
                assert rc == S.ECAPTURE, rc
    torch.cuda.current_stream().wait_stream(side)
    for _ in range(4):
        g.replay()
    torch.cuda.synchronize()
    assert torch.equal(st_g, st_e) and st_g[4].item() == 20.0
    assert torch.equal(pos_g, pos_e) and torch.equal(vel_g, vel_e) and torch.equal(acc_g, acc_e)


@pytest.mark.gpu
@pytest.mark.parametrize("n", [4096, 20000, 40000, 140000])
def test_fused_timestep_minimum_equals_the_separate_pass(S, oracle, n):
    """Eq. 12's minimum fused into the force evaluation's last kernel (split-j epilogue at 4,096, ring reduce at 20,000,
    pair-symmetric panel reduce at 40,000 / 140,000) against the separate O(N) pass: twelve adaptive steps, bit-identical
    state either way; and the shortcut is dropped when another library call comes between two steps."""
    import torch
    ps = _config4(oracle, n)
    B, G, eps, dt_max, a0 = 1.0 / ps.r_cut ** 3, 1.0, 0.025, 0.5, 1 / 51
    c = S.Cosmology(**LCDM)
    dm, dh = dev(ps.mass), dev(ps.soft)
    out = torch.empty(4, dtype=torch.float64, device="cuda")
    runs = {}
    for fuse in (1, 0):
        S.steps_set_option("fuse_eq12", fuse)
        try:
            dpos, dvel = dev(ps.pos), dev(ps.vel)
            dacc = torch.empty_like(dpos)
            S.steps_forces(dpos, dm, dh, dacc)
            st = torch.tensor([a0, 0.0, 1.0, 0.0, 0.0], dtype=torch.float64, device="cuda")
            l0 = S.steps_kernel_launch_count()
            for k in range(12):
                S.steps_kdk_step_adaptive(dpos, dvel, dacc, dm, dh, st, c, G, B, eps, dt_max)
                if k == 5:
                    S.steps_momentum(dvel, dm, out)          # a foreign call: the next step must not use the shortcut
            torch.cuda.synchronize()
            runs[fuse] = (dpos.clone(), dvel.clone(), dacc.clone(), st.clone(), S.steps_kernel_launch_count() - l0)
        finally:
            S.steps_set_option("fuse_eq12", 1)
    for a, b in zip(runs[1][:4], runs[0][:4]):
        assert torch.equal(a, b)
    assert runs[0][4] - runs[1][4] == 10                     # 12 steps: the first and the one after the foreign call keep the pass


# ---- Eq. 5 (L65-70) with the cut |x - nL| < 2.6 L: periodic image sum (fp64) ------------------------------------------
@pytest.mark.gpu
@pytest.mark.parametrize("n", [2, 27, 300, 1500])
def test_periodic_image_sum_matches_oracle(S, oracle, n):
    import torch
    L = 1.3
    pos, mass, soft = _periodic_box(n, L, 6600 + n)
    if n == 27:                                  # simple-cubic lattice: every site a centre of symmetry, force 0
        g = (np.arange(3) + 0.5) * L / 3
        pos = np.ascontiguousarray(np.array(np.meshgrid(g, g, g, indexing="ij")).reshape(3, -1))
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    S.steps_forces_periodic(dev(pos), dev(mass), dev(soft), L, acc)
    got = acc.cpu().numpy()
    ref = oracle.forces_periodic_images(pos, mass, soft, L)
    if n == 27:
        assert np.abs(got).max() < 1e-12 and np.abs(ref).max() < 1e-12
        return
    # ~80 images per pair cancel to a remainder: the error is measured against the scale of what is summed
    scale = _pair_force_abs_sum(pos, mass, soft, L)
    e_abs = np.linalg.norm(got - ref, axis=0) / scale
    e = rel_err(got, ref)
    print(f"[image sum n={n}] relative to net force: max {e.max():.3e}; relative to sum_j |f_ij|: max {e_abs.max():.3e}")
    assert e_abs.max() <= 1e-12 and e.max() <= 1e-10
    # representative independence on the device: shift a third of the particles by lattice vectors
    moved = pos.copy(); moved[:, ::3] += np.array([[2 * L], [-L], [3 * L]])
    acc2 = torch.empty_like(acc)
    S.steps_forces_periodic(dev(np.ascontiguousarray(moved)), dev(mass), dev(soft), L, acc2)
    assert np.abs(acc2.cpu().numpy() - got).max() <= 1e-10 * np.abs(got).max()


@pytest.mark.gpu
def test_periodic_image_sum_several_i_blocks_sampled(S, oracle):
    """The image sum at N = 9,000: 36 j-tiles, 5 i-blocks (the last one ragged), so the stream-K split of an i-block
    across CTAs and the multi-record reduce are exercised with BOX = 2; oracle on a sample of 96 particles (first and
    last of every i-block + uniform).  Bars: 1e-12 relative to the scale of what is summed, sum_j |f_ij| (the fp64
    path's bar); relative to the NET force the same error appears amplified by kappa_i = sum_j|f_ij| / |sum_j f_ij|
    (the ~80 images per pair cancel), bar 1e-12 x max kappa, asserted."""
    import torch
    n, L = 9000, 1.3
    pos, mass, soft = _periodic_box(n, L, 6600 + n)
    edges = np.concatenate([[b * 2048, min(n, (b + 1) * 2048) - 1] for b in range(5)])
    idx = np.unique(np.concatenate([edges, np.linspace(0, n - 1, 86).astype(np.int64)]))
    acc = torch.empty(3, n, dtype=torch.float64, device="cuda")
    S.steps_forces_periodic(dev(pos), dev(mass), dev(soft), L, acc)
    got = acc.cpu().numpy()[:, idx]
    ref = oracle.forces_periodic_images(pos, mass, soft, L, idx=idx)
    scale = _pair_force_abs_sum(pos, mass, soft, L)[idx]
    kappa = scale / np.linalg.norm(ref, axis=0)
    e_abs = np.linalg.norm(got - ref, axis=0) / scale
    e = rel_err(got, ref)
    print(f"[image sum n={n}, {len(idx)} sampled] relative to sum_j|f_ij|: max {e_abs.max():.3e}; to the net force: max "
          f"{e.max():.3e}; kappa max {kappa.max():.1f}")
    assert e_abs.max() <= 1e-12
    assert e.max() <= 1e-12 * kappa.max()
    # Newton's third law over the whole set, on the device
    dm = dev(mass)
    p = (dm * acc).sum(dim=1)
    assert float(p.norm()) < 1e-12 * float((dm * acc.norm(dim=0)).sum())


@pytest.mark.parametrize("n,ordered", [(18433, True), (32768, True), (40001, True), (32768, False)])
def test_periodic_image_sum_pair_symmetric_route(S, oracle, n, ordered):
    """From 9 blocks (N = 16,385) the image sum evaluates every far meeting of two groups of different blocks once
    (forces_sym_img_kernel), the possibly-softened units through forces_boxgen_kernel<., 2>, the own blocks through the
    group-ring kernel.  Against the oracle on a sample (unequal masses: a swapped m_i / m_j in the reaction would show;
    some larger softenings; unordered input: everything through the unpruned route), equality with the one-sided
    evaluation (option "sym" = 0), bit-identical re-run, Newton's third law."""
    import torch
    L = 1.3
    pos, mass, soft = _periodic_box(n, L, 6700 + n)
    rng = np.random.default_rng(n)
    mass = mass * rng.uniform(0.5, 2.0, size=n)
    mass /= mass.sum()
    soft = soft * rng.uniform(0.5, 3.0, size=n)
    if ordered:
        pos = np.ascontiguousarray(pos[:, synth.morton_order(pos, L)])
    dpos, dm, dh = dev(pos), dev(mass), dev(soft)
    acc, again, one = (torch.empty(3, n, dtype=torch.float64, device="cuda") for _ in range(3))
    S.steps_forces_periodic(dpos, dm, dh, L, acc)
    if not ordered:                                             # (slow route: the oracle comparison is enough)
        idx = np.linspace(0, n - 1, 24).astype(np.int64)
    else:
        S.steps_forces_periodic(dpos, dm, dh, L, again)
        assert torch.equal(acc, again)
        try:
            S.steps_set_option("sym", 0)
            S.steps_forces_periodic(dpos, dm, dh, L, one)
        finally:
            S.steps_set_option("sym", 1)
        edges = np.concatenate([[b * 2048, min(n, (b + 1) * 2048) - 1] for b in range((n + 2047) // 2048)])
        idx = np.unique(np.concatenate([edges, np.linspace(0, n - 1, 40).astype(np.int64)]))
    got = acc.cpu().numpy()[:, idx]
    ref = oracle.forces_periodic_images(pos, mass, soft, L, idx=idx)
    scale = _pair_force_abs_sum(pos, mass, np.full(n, soft.min()), L, idx)
    e_abs = np.linalg.norm(got - ref, axis=0) / scale
    print(f"[image sum, pair-symmetric route n={n} ordered={ordered}, {len(idx)} sampled] relative to sum_j|f_ij|: max {e_abs.max():.3e}")
    assert e_abs.max() <= 1e-12
    if ordered:
        d = np.linalg.norm((acc - one).cpu().numpy()[:, idx], axis=0) / scale
        assert d.max() <= 1e-13, d.max()
    p = (dm * acc).sum(dim=1)
    assert float(p.norm()) < 1e-12 * float((dm * acc.norm(dim=0)).sum())


def test_config4_lockstep_200_steps_8192(S, oracle):
    """Config 4 at N = 8192, every one of the 200 comoving KDK steps (a: 1/51 -> 1): the library steps
    from the ORACLE's state (x_n, v_n, acc_n) and must land on the oracle's (x_{n+1}, v_{n+1},
    acc_{n+1}).  Lock-step shows the per-step error; what accumulates is the free-running test below."""
    import torch
    n = 8192
    ps = _config4(oracle, n)
    B = 1.0 / ps.r_cut ** 3
    dts = oracle.ln_a_schedule(1 / 51, 1.0, 200, LCDM)
    cosmo = S.Cosmology(**LCDM)
    pos, vel = ps.pos.copy(), ps.vel.copy()
    acc = oracle.forces(pos, ps.mass, ps.soft)
    dm, dh = dev(ps.mass), dev(ps.soft)
    a = 1 / 51
    worst = dict(x=0.0, v=0.0, acc=0.0)
    for k, dt in enumerate(dts):
        dpos, dvel, dacc = dev(pos), dev(vel), dev(acc)
        sc = S.steps_kdk_schedule(a, float(dt), 1.0, cosmo)
        S.steps_kdk_step(dpos, dvel, dacc, dm, dh, S.KdkCoeffs(1.0, 0.0, sc["alpha_open"], sc["beta_open"], sc["gamma"], B, 0))
        S.steps_kick_drift(dpos, dvel, dacc, S.KdkCoeffs(sc["alpha_close"], sc["beta_close"], 1.0, 0.0, 0.0, B, 0))
        a_next = oracle.kdk_step(pos, vel, acc, ps.mass, ps.soft, a, float(dt), 1.0, B, LCDM)
        assert sc["a_next"] == pytest.approx(a_next, rel=1e-14)
        a = a_next
        worst["x"] = max(worst["x"], np.max(np.linalg.norm(dpos.cpu().numpy() - pos, axis=0) / ps.spacing))
        worst["acc"] = max(worst["acc"], rel_err(dacc.cpu().numpy(), acc).max())
        worst["v"] = max(worst["v"], rel_err(dvel.cpu().numpy(), vel).max())
    print(f"config4 lockstep N={n}: worst over 200 steps: |dx|/s {worst['x']:.2e}, acc rel {worst['acc']:.2e}, v rel {worst['v']:.2e}")
    assert a == pytest.approx(1.0, rel=1e-8)
    assert worst["x"] <= 1e-13 and worst["acc"] <= FP64_MAX and worst["v"] <= 1e-11


def _chaos_floor():
    """tests/golden/config4_chaos_floor.txt (written by tests/golden/make_config4_chaos_floor.py, oracle only):
    {step: max_i |dx_i|/s_i between the oracle run and oracle runs started 1 ulp away}."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "config4_chaos_floor.txt")
    rows = [line.split() for line in open(path) if not line.startswith("#")]
    return {int(r[0]): float(r[2]) for r in rows}


def test_config4_free_running_vs_oracle_8192(S, oracle):
    """BASELINE.json configs[4]: "final positions compared to the oracle run at N = 8,192".  The library runs free (its own
    state from step 0) next to the free-running oracle.  The run is chaotic, so the comparison is held to the chaos floor
    (SURVEY.md 8(c.5)): the distance between the oracle and the oracle started 1 ulp away, recorded every 10 steps in
    tests/golden/config4_chaos_floor.txt (1e-14 spacings at step 10, 1e-6 at step 130, O(1) from step 175; DESIGN.md
    section 2).  Bar: library-vs-oracle <= 10 x floor at every recorded step up to the LAST one whose floor is still
    <= 1e-6 of the local spacing -- step 130 of 200 -- beyond which no two fp64 implementations agree; the remaining
    70 steps are run for the momentum bound and sanity."""
    import torch
    from paper_1811_05903_b200 import integrate
    n = 8192
    ps = _config4(oracle, n)
    B = 1.0 / ps.r_cut ** 3
    dts = oracle.ln_a_schedule(1 / 51, 1.0, 200, LCDM)
    floor = _chaos_floor()
    last = max(k for k, v in floor.items() if v <= 1e-6)
    assert last == 130, "the chaos-floor table changed: re-read the bar in the docstring"

    pos, vel = ps.pos.copy(), ps.vel.copy()
    acc = oracle.forces(pos, ps.mass, ps.soft)
    a, ref = 1 / 51, {}
    for k, dt in enumerate(dts[:last]):
        a = oracle.kdk_step(pos, vel, acc, ps.mass, ps.soft, a, float(dt), 1.0, B, LCDM)
        if (k + 1) in floor:
            ref[k + 1] = pos.copy()

    dpos, dvel, dm, dh = dev(ps.pos), dev(ps.vel), dev(ps.mass), dev(ps.soft)
    dacc = torch.empty_like(dpos)
    S.steps_forces(dpos, dm, dh, dacc)
    cosmo = S.Cosmology(**LCDM)
    got = {}

    def on_step(k, a_k):                        # positions after step k + 1 are final (the closing kick only touches v)
        if (k + 1) in ref:
            got[k + 1] = dpos.cpu().numpy()

    a_gpu = integrate.run_kdk(dpos, dvel, dacc, dm, dh, 1 / 51, dts, cosmo, 1.0, B, on_step=on_step)
    torch.cuda.synchronize()
    table = []
    for k in sorted(ref):
        d = np.max(np.linalg.norm(got[k] - ref[k], axis=0) / ps.spacing)
        table.append((k, d, floor[k]))
    print("config4 free-running N=8192: step, library-vs-oracle max|dx|/s, chaos floor: " +
          "; ".join(f"{k}: {d:.2e} / {f:.2e}" for k, d, f in table))
    for k, d, f in table:
        assert d <= 10.0 * f, f"step {k}: library-vs-oracle {d:.3e} > 10 x chaos floor {f:.3e}"
    assert a_gpu == pytest.approx(1.0, rel=1e-8)
    assert np.all(np.isfinite(dpos.cpu().numpy()))
    p = oracle.momentum(dvel.cpu().numpy(), ps.mass)
    assert np.linalg.norm(p[:3]) / p[3] <= 1e-10


def test_config4_momentum_drift_262144(S, oracle):
    """Config 4 at its full size: total momentum drift <= 1e-10 relative in fp64 through 200 steps -- once as the
    particles come (no re-sorting), once re-sorted radially at the start and every 20 steps (integrate.resort_radial).
    Also the measurement VERDICT r01 asked for: the share of (i-group, tile) pairs that need the per-pair softening test
    at steps 0 / 100 / 200, and the wall clock of the two runs (DESIGN.md section 5.2 records the numbers)."""
    import time
    import torch
    from paper_1811_05903_b200 import integrate
    ps = _config4(oracle, 262144)
    B = 1.0 / ps.r_cut ** 3
    dts = oracle.ln_a_schedule(1 / 51, 1.0, 200, LCDM)
    out = torch.empty(4, dtype=torch.float64, device="cuda")
    report = {}
    for resort in (0, 20, 2):
        dpos, dvel, dm, dh = dev(ps.pos), dev(ps.vel), dev(ps.mass), dev(ps.soft)
        dacc = torch.empty_like(dpos)
        ids = torch.arange(ps.n, dtype=torch.int64, device="cuda")
        if resort:
            integrate.resort_radial([dpos, dvel], [dm, dh], ids)
        S.steps_forces(dpos, dm, dh, dacc)
        worst, near = [], {}

        def near_fraction(tag):
            S.steps_near_fraction(dpos, dm, dh, out[:2])
            o = out[:2].cpu().numpy()
            near[tag] = round(float(o[0] / o[1]), 4)

        near_fraction("step 0")

        def on_step(k, a):
            if k % 20 == 19:
                S.steps_momentum(dvel, dm, out)
                o = out.cpu().numpy()
                worst.append(np.linalg.norm(o[:3]) / o[3])
            if k + 1 in (100, 200):
                near_fraction(f"step {k + 1}")

        torch.cuda.synchronize()
        t0 = time.perf_counter()
        integrate.run_kdk(dpos, dvel, dacc, dm, dh, 1 / 51, dts, S.Cosmology(**LCDM), 1.0, B, on_step=on_step,
                          resort_every=resort, ids=ids)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        S.steps_momentum(dvel, dm, out)
        o = out.cpu().numpy()
        worst.append(np.linalg.norm(o[:3]) / o[3])
        report[resort] = (near, wall, max(worst))
        assert np.all(np.isfinite(dpos.cpu().numpy()))
        assert max(worst) <= 1e-10
        assert np.array_equal(np.sort(ids.cpu().numpy()), np.arange(ps.n))
    for resort, (near, wall, w) in report.items():
        print(f"config4 N=262144, 200 steps, re-sort every {resort or 'never'}: near (i-group, tile) share {near}, "
              f"wall {wall:.2f} s, worst |P|/sum m|v| {w:.2e}")
    assert report[20][0]["step 200"] < report[0][0]["step 200"] and report[20][1] < report[0][1]
