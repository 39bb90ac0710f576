"""-m gpu: steps_forces_static (include/steps.h) -- the fp64 force evaluation of PAPER.md Eq. 3-4 for callers that cannot
allocate device memory: its scratch is a file-scope __device__ array of the library (STEPS_STATIC_SCRATCH_BYTES), N is
limited to STEPS_STATIC_MAX_N.  Checked against the existing path (steps_forces) within the fp64 bar of the parity tests,
on two calls in a row that share the array (the second smaller and ragged, so it runs over the first call's leftovers).
This file is collected last on purpose (the suite runs with pytest -x) and needs nothing from the other test files: it
passes alone in a fresh process and after the others."""
import numpy as np
import pytest

from paper_1811_05903_b200 import synth

pytestmark = pytest.mark.gpu

FP64_MAX = 1e-12          # north_star's fp64 bar, as in test_parity_gpu.py


@pytest.fixture(scope="module")
def S():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_1811_05903_b200 import steps
    steps.lib()
    return steps


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _rel_err(got, ref):
    return np.linalg.norm(got - ref, axis=0) / np.linalg.norm(ref, axis=0)


def test_static_scratch_forces_match_the_existing_path_on_two_calls_in_a_row(S):
    import torch
    assert S.STATIC_MAX_N == 16384
    sets = [synth.g0(S.STATIC_MAX_N, seed=9101), synth.g0(5001, seed=9102)]      # the maximum, then a ragged smaller set
    inputs = [(_dev(ps.pos), _dev(ps.mass), _dev(ps.soft)) for ps in sets]
    outs = [torch.full_like(x, float("nan")) for x, _, _ in inputs]
    # the two calls in a row, nothing in between, BEFORE the existing path runs (alone in a fresh process this is the
    # library's very first call: no workspace exists yet)
    for (x, m, h), a in zip(inputs, outs):
        S.steps_forces_static(x, m, h, a)
    torch.cuda.synchronize()
    for (x, m, h), a, ps in zip(inputs, outs, sets):
        ref = torch.full_like(x, float("nan"))
        S.steps_forces(x, m, h, ref)
        torch.cuda.synchronize()
        got, want = a.cpu().numpy(), ref.cpu().numpy()
        assert np.all(np.isfinite(got)), f"N={ps.n}"
        e = _rel_err(got, want)
        print(f"[static N={ps.n}] max rel err vs steps_forces {e.max():.3e}, bit-identical: {np.array_equal(got, want)}")
        assert e.max() <= FP64_MAX, f"N={ps.n}: {e.max():.3e}"
    # the first input again, over the second call's leftovers: the same bits as the first time
    again = torch.full_like(inputs[0][0], float("nan"))
    S.steps_forces_static(*inputs[0], again)
    torch.cuda.synchronize()
    assert torch.equal(again, outs[0])


def test_static_scratch_calls_leave_device_memory_alone(S):
    """Steady state: with the tensors in place and one call done (module and kernels loaded), further calls change the
    device's free memory by nothing."""
    import torch
    ps = synth.g0(8192, seed=9103)
    x, m, h = _dev(ps.pos), _dev(ps.mass), _dev(ps.soft)
    a = torch.empty_like(x)
    S.steps_forces_static(x, m, h, a)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        S.steps_forces_static(x, m, h, a)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_static_scratch_rejects_sizes_beyond_the_maximum(S):
    import torch
    n = S.STATIC_MAX_N + 1
    x = torch.zeros(3, n, dtype=torch.float64, device="cuda")
    m = torch.ones(n, dtype=torch.float64, device="cuda")
    h = torch.full((n,), 0.01, dtype=torch.float64, device="cuda")
    a = torch.full_like(x, 7.0)
    with pytest.raises(S.StepsError, match="STEPS_STATIC_MAX_N"):
        S.steps_forces_static(x, m, h, a)
    torch.cuda.synchronize()
    assert bool((a == 7.0).all())                 # nothing was launched
    assert S.lib().steps_forces_static(x.data_ptr(), m.data_ptr(), h.data_ptr(), n, a.data_ptr(), None) == S.ETOOLARGE
