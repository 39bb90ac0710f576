"""Thin ctypes binding of the C ABI in include/steps.h -- same names, argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libsteps_b200.so; PyTorch is used
for device memory and streams.  There is no CPU fallback: if the library is missing it is
built (nvcc, in-tree) or the import of the symbol fails loudly."""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsteps_b200.so")

OK, EINVAL, ECUDA, EUNSUPPORTED, ENOMEM, ECAPTURE, ETOOLARGE = 0, -1, -2, -3, -4, -5, -6
STATIC_MAX_N = 16384    # steps_forces_static (STEPS_STATIC_MAX_N of include/steps.h)

EXPORTS = [
    "steps_forces", "steps_forces_static", "steps_forces_mixed", "steps_forces_range", "steps_forces_blocks", "steps_forces_share", "steps_block_size", "steps_forces_host", "steps_kick_drift",
    "steps_sort_radial", "steps_permute", "steps_near_fraction",
    "steps_kdk_step", "steps_hubble", "steps_scale_factor_rk4", "steps_kdk_schedule", "steps_momentum",
    "steps_timestep", "steps_timestep_coefficient", "steps_force_residual", "steps_forces_quasi_periodic", "steps_forces_periodic",
    "steps_kdk_step_adaptive", "steps_kick_close_adaptive",
    "steps_reserve", "steps_shutdown", "steps_workspace_bytes", "steps_strerror", "steps_last_cuda_error",
    "steps_version", "steps_kernel_launch_count", "steps_set_option", "steps_last_force_kernel_ms",
    "steps_persistent_grid", "steps_pair_symmetric",
]


class KdkCoeffs(C.Structure):
    _fields_ = [("alpha_close", C.c_double), ("beta_close", C.c_double), ("alpha_open", C.c_double),
                ("beta_open", C.c_double), ("gamma", C.c_double), ("B", C.c_double), ("mixed", C.c_int)]


class Cosmology(C.Structure):
    _fields_ = [("H0", C.c_double), ("Omega_m", C.c_double), ("Omega_r", C.c_double),
                ("Omega_L", C.c_double), ("Omega_k", C.c_double)]


class StepsError(RuntimeError):
    pass


_lib = None


def lib() -> C.CDLL:
    """Load (building first if the .so is absent or stale) the C-ABI library."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    _lib = load_library(_build.build())
    return _lib


def build_info() -> dict:
    """What the build did to the loaded library (nvcc command, operand-reuse pass): build.py's buildinfo record."""
    from . import build as _build
    return _build.build_info()


def load_library(path: str) -> C.CDLL:
    """dlopen a build of the C-ABI library and declare its prototypes (lib() does this for the product build; the A/B
    test of the post-link pass loads the unpatched build next to it)."""
    L = C.CDLL(path)
    vp, ll, dbl, i32 = C.c_void_p, C.c_longlong, C.c_double, C.c_int
    L.steps_forces.argtypes = [vp, vp, vp, ll, vp, vp]
    L.steps_forces_mixed.argtypes = [vp, vp, vp, ll, vp, vp]
    L.steps_forces_static.argtypes = [vp, vp, vp, ll, vp, vp]
    L.steps_forces_range.argtypes = [vp, vp, vp, ll, ll, ll, vp, i32, vp]
    L.steps_forces_host.argtypes = [vp, vp, vp, ll, vp, i32, vp]
    L.steps_forces_blocks.argtypes = [vp, vp, vp, ll, ll, ll, vp, i32, vp]
    L.steps_forces_share.argtypes = [vp, vp, vp, ll, i32, i32, vp, i32, vp]
    L.steps_sort_radial.argtypes = [vp, ll, vp, vp]
    L.steps_permute.argtypes = [vp, ll, i32, vp, vp, vp]
    L.steps_near_fraction.argtypes = [vp, vp, vp, ll, vp, vp]
    L.steps_kick_drift.argtypes = [vp, vp, vp, ll, C.POINTER(KdkCoeffs), vp]
    L.steps_kdk_step.argtypes = [vp, vp, vp, vp, vp, ll, C.POINTER(KdkCoeffs), vp]
    L.steps_hubble.argtypes = [dbl, C.POINTER(Cosmology)]
    L.steps_hubble.restype = dbl
    L.steps_scale_factor_rk4.argtypes = [dbl, dbl, C.POINTER(Cosmology)]
    L.steps_scale_factor_rk4.restype = dbl
    L.steps_kdk_schedule.argtypes = [dbl, dbl, dbl, C.POINTER(Cosmology), C.POINTER(dbl)]
    L.steps_momentum.argtypes = [vp, vp, ll, vp, vp]
    L.steps_forces_quasi_periodic.argtypes = [vp, vp, vp, ll, dbl, vp, i32, vp]
    L.steps_forces_periodic.argtypes = [vp, vp, vp, ll, dbl, vp, vp]
    L.steps_kdk_step_adaptive.argtypes = [vp, vp, vp, vp, vp, ll, vp, C.POINTER(Cosmology), dbl, dbl, dbl, dbl, i32, vp]
    L.steps_kick_close_adaptive.argtypes = [vp, vp, vp, ll, vp, dbl, vp]
    L.steps_timestep.argtypes = [vp, vp, vp, ll, dbl, dbl, dbl, dbl, vp, vp]
    L.steps_force_residual.argtypes = [vp, vp, ll, dbl, vp, vp]
    L.steps_timestep_coefficient.argtypes = [dbl, dbl]
    L.steps_timestep_coefficient.restype = dbl
    L.steps_reserve.argtypes = [ll]
    L.steps_shutdown.restype = None
    L.steps_workspace_bytes.argtypes = [ll]
    L.steps_workspace_bytes.restype = ll
    L.steps_strerror.argtypes = [i32]
    L.steps_strerror.restype = C.c_char_p
    L.steps_kernel_launch_count.restype = ll
    L.steps_set_option.argtypes = [C.c_char_p, ll]
    L.steps_last_force_kernel_ms.restype = dbl
    L.steps_persistent_grid.argtypes = [i32]
    L.steps_pair_symmetric.argtypes = [ll, i32]
    return L


def _check(rc: int) -> None:
    if rc != OK:
        L = lib()
        msg = L.steps_strerror(rc).decode()
        if rc == ECUDA:
            msg += f" [cudaError {L.steps_last_cuda_error()}]"
        raise StepsError(f"steps error {rc}: {msg}")


def _stream(stream=None) -> int:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _dev(t, n_elem: int):
    import torch
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n_elem):
        raise StepsError(f"expected a contiguous CUDA float64 tensor with {n_elem} elements, got "
                         f"{tuple(t.shape)} {t.dtype} {t.device}")
    return t.data_ptr()


def _host(a, n_elem: int):
    import numpy as np
    import torch
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != n_elem:
            raise StepsError("expected a contiguous CPU float64 tensor")
        return a.data_ptr()
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous and a.size == n_elem):
        raise StepsError("expected a C-contiguous float64 numpy array")
    return a.ctypes.data


# ---- the calls of include/steps.h, same names -------------------------------------------------

def steps_forces(pos, mass, soft, acc, stream=None) -> None:
    n = mass.numel()
    _check(lib().steps_forces(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, _dev(acc, 3 * n), _stream(stream)))


def steps_forces_static(pos, mass, soft, acc, stream=None) -> None:
    """steps_forces for N <= STATIC_MAX_N with the scratch in a device array of the library: never allocates."""
    n = mass.numel()
    _check(lib().steps_forces_static(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, _dev(acc, 3 * n), _stream(stream)))


def steps_forces_mixed(pos, mass, soft, acc, stream=None) -> None:
    n = mass.numel()
    _check(lib().steps_forces_mixed(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, _dev(acc, 3 * n),
                                    _stream(stream)))


def steps_forces_range(pos, mass, soft, i_begin: int, i_end: int, acc_out, mixed: bool = False, stream=None) -> None:
    n = mass.numel()
    _check(lib().steps_forces_range(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, i_begin, i_end,
                                    _dev(acc_out, 3 * (i_end - i_begin)), int(mixed), _stream(stream)))


def steps_block_size() -> int:
    return int(lib().steps_block_size())


def steps_forces_blocks(pos, mass, soft, first_block: int, block_stride: int, acc_out, mixed: bool = False, stream=None) -> None:
    """Forces on the particles of the blocks first_block, first_block + block_stride, ... (round-robin dealing of the
    i-blocks over ranks); acc_out: SoA over the owned particles, packed (3 * cnt elements)."""
    n = mass.numel()
    _check(lib().steps_forces_blocks(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, first_block, block_stride,
                                     _dev(acc_out, acc_out.numel()), int(mixed), _stream(stream)))


def steps_forces_share(pos, mass, soft, rank: int, world: int, acc_part, mixed: bool = False, stream=None) -> None:
    """acc_part (3N) = the contribution of the rank-th of `world` equal parts of the pair evaluations to every particle's
    acceleration; the sum over the ranks is the result of steps_forces / steps_forces_mixed to rounding."""
    n = mass.numel()
    _check(lib().steps_forces_share(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, int(rank), int(world),
                                    _dev(acc_part, 3 * n), int(mixed), _stream(stream)))


def steps_sort_radial(pos, perm, stream=None) -> None:
    """perm (int64 device tensor, N) = particle indices by ascending |x|."""
    import torch
    n = pos.numel() // 3
    if not (perm.is_cuda and perm.dtype == torch.int64 and perm.is_contiguous() and perm.numel() == n):
        raise StepsError("perm must be a contiguous CUDA int64 tensor with N elements")
    _check(lib().steps_sort_radial(_dev(pos, 3 * n), n, perm.data_ptr(), _stream(stream)))


def steps_permute(src, perm, dst, stream=None) -> None:
    """dst[c][k] = src[c][perm[k]] (SoA with src.numel() / N components)."""
    n = perm.numel()
    ncomp = src.numel() // n
    _check(lib().steps_permute(_dev(src, ncomp * n), n, ncomp, perm.data_ptr(), _dev(dst, ncomp * n), _stream(stream)))


def steps_near_fraction(pos, mass, soft, out2, stream=None) -> None:
    n = mass.numel()
    _check(lib().steps_near_fraction(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, _dev(out2, 2), _stream(stream)))


def steps_forces_host(pos_host, mass_host, soft_host, acc_host, mixed: bool = False, stream=None) -> None:
    n = int(mass_host.size if hasattr(mass_host, "size") and not callable(mass_host.size) else mass_host.numel())
    _check(lib().steps_forces_host(_host(pos_host, 3 * n), _host(mass_host, n), _host(soft_host, n), n,
                                   _host(acc_host, 3 * n), int(mixed), _stream(stream)))


def steps_kick_drift(pos, vel, acc, coeffs: KdkCoeffs, stream=None) -> None:
    n = pos.numel() // 3
    _check(lib().steps_kick_drift(_dev(pos, 3 * n), _dev(vel, 3 * n), _dev(acc, 3 * n), n, C.byref(coeffs),
                                  _stream(stream)))


def steps_kdk_step(pos, vel, acc, mass, soft, coeffs: KdkCoeffs, stream=None) -> None:
    n = mass.numel()
    _check(lib().steps_kdk_step(_dev(pos, 3 * n), _dev(vel, 3 * n), _dev(acc, 3 * n), _dev(mass, n), _dev(soft, n),
                                n, C.byref(coeffs), _stream(stream)))


def steps_hubble(a: float, cosmo: Cosmology) -> float:
    return lib().steps_hubble(a, C.byref(cosmo))


def steps_scale_factor_rk4(a: float, dt: float, cosmo: Cosmology) -> float:
    return lib().steps_scale_factor_rk4(a, dt, C.byref(cosmo))


def steps_kdk_schedule(a_n: float, dt: float, G: float, cosmo: Cosmology) -> dict:
    out = (C.c_double * 6)()
    _check(lib().steps_kdk_schedule(a_n, dt, G, C.byref(cosmo), out))
    return dict(alpha_open=out[0], beta_open=out[1], gamma=out[2], alpha_close=out[3], beta_close=out[4],
                a_next=out[5])


def steps_momentum(vec, mass, out4, stream=None) -> None:
    n = mass.numel()
    _check(lib().steps_momentum(_dev(vec, 3 * n), _dev(mass, n), n, _dev(out4, 4), _stream(stream)))


def steps_forces_quasi_periodic(pos, mass, soft, L: float, acc, mixed: bool = False, stream=None) -> None:
    """Eq. 5 leading term (nearest image in a cubic box of side L); otherwise as steps_forces / steps_forces_mixed."""
    n = mass.numel()
    _check(lib().steps_forces_quasi_periodic(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, float(L), _dev(acc, 3 * n),
                                             int(mixed), _stream(stream)))


def steps_forces_periodic(pos, mass, soft, L: float, acc, stream=None) -> None:
    """Eq. 5 image sum with the cut |x - nL| < 2.6 L in a cubic box of side L (fp64 path)."""
    n = mass.numel()
    _check(lib().steps_forces_periodic(_dev(pos, 3 * n), _dev(mass, n), _dev(soft, n), n, float(L), _dev(acc, 3 * n),
                                       _stream(stream)))


def steps_kdk_step_adaptive(pos, vel, acc, mass, soft, state5, cosmo: "Cosmology", G: float, B: float, eps: float,
                            dt_max: float, mixed: bool = False, stream=None) -> None:
    """One device-resident adaptive KDK step (Eq. 12 step length, coefficients computed on the device); state5 is a
    5-element device tensor {a, dt, alpha_close, beta_close, steps}."""
    n = mass.numel()
    _check(lib().steps_kdk_step_adaptive(_dev(pos, 3 * n), _dev(vel, 3 * n), _dev(acc, 3 * n), _dev(mass, n), _dev(soft, n), n,
                                         _dev(state5, 5), C.byref(cosmo), G, B, eps, dt_max, int(mixed), _stream(stream)))


def steps_kick_close_adaptive(pos, vel, acc, state5, B: float, stream=None) -> None:
    n = pos.numel() // 3
    _check(lib().steps_kick_close_adaptive(_dev(pos, 3 * n), _dev(vel, 3 * n), _dev(acc, 3 * n), n, _dev(state5, 5), B,
                                           _stream(stream)))


def steps_timestep(pos, acc, soft, coef: float, B: float, eps: float, dt_max: float, dt_out, stream=None) -> None:
    """Eq. 12 global adaptive time step into the 1-element device tensor dt_out (stream-ordered)."""
    n = soft.numel()
    _check(lib().steps_timestep(_dev(pos, 3 * n), _dev(acc, 3 * n), _dev(soft, n), n, coef, B, eps, dt_max,
                                _dev(dt_out, 1), _stream(stream)))


def steps_timestep_coefficient(G: float, a: float) -> float:
    return float(lib().steps_timestep_coefficient(G, a))


def steps_force_residual(pos, acc, B: float, out2, stream=None) -> None:
    """Glass-generation monitor: out2 = [sum_i |acc_i + B x_i|^2, max_i |acc_i + B x_i|] (2-element device tensor)."""
    n = pos.numel() // 3
    _check(lib().steps_force_residual(_dev(pos, 3 * n), _dev(acc, 3 * n), n, B, _dev(out2, 2), _stream(stream)))


def steps_reserve(n: int) -> None:
    _check(lib().steps_reserve(n))


def steps_shutdown() -> None:
    lib().steps_shutdown()


def steps_workspace_bytes(n: int) -> int:
    return int(lib().steps_workspace_bytes(n))


def steps_version() -> int:
    return int(lib().steps_version())


def steps_kernel_launch_count() -> int:
    return int(lib().steps_kernel_launch_count())


def steps_set_option(key: str, value: int) -> None:
    _check(lib().steps_set_option(key.encode(), value))


def steps_last_force_kernel_ms() -> float:
    return float(lib().steps_last_force_kernel_ms())


def steps_persistent_grid(mixed: bool) -> int:
    return int(lib().steps_persistent_grid(int(mixed)))


def steps_pair_symmetric(n: int, mixed: bool = False) -> bool:
    return bool(lib().steps_pair_symmetric(n, int(mixed)))
