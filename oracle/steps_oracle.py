"""ctypes binding of oracle/steps_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this.  It imports nothing from paper_1811_05903_b200 and vice versa.  All
arithmetic lives in the C file (each function there cites the PAPER.md passage it
follows); this file only marshals numpy arrays.  The few pure-Python scalars at the
bottom (closed-form t(a), growth rate by quadrature) are used for input schedules and pins."""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

from . import build as _build

_lib = None


class Cosmo(C.Structure):
    """PAPER.md Eq. 1 (L37-39) parameters, present-day values, code units."""
    _fields_ = [("H0", C.c_double), ("Omega_m", C.c_double), ("Omega_r", C.c_double),
                ("Omega_L", C.c_double), ("Omega_k", C.c_double)]


STATIC = dict(H0=0.0, Omega_m=0.0, Omega_r=0.0, Omega_L=0.0, Omega_k=0.0)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp, llp = C.POINTER(C.c_double), C.POINTER(C.c_longlong)
        L.oracle_spline_F.restype = C.c_double
        L.oracle_spline_F.argtypes = [C.c_double, C.c_double]
        L.oracle_forces.restype = None
        L.oracle_forces.argtypes = [dp, dp, dp, C.c_longlong, llp, C.c_longlong, dp, C.c_int]
        L.oracle_forces_quasi_periodic.restype = None
        L.oracle_forces_quasi_periodic.argtypes = [dp, dp, dp, C.c_longlong, C.c_double, llp, C.c_longlong, dp]
        L.oracle_forces_periodic_images.restype = None
        L.oracle_forces_periodic_images.argtypes = [dp, dp, dp, C.c_longlong, C.c_double, llp, C.c_longlong, dp]
        L.oracle_hubble.restype = C.c_double
        L.oracle_hubble.argtypes = [C.c_double, C.POINTER(Cosmo)]
        L.oracle_rk4_scale_factor.restype = C.c_double
        L.oracle_rk4_scale_factor.argtypes = [C.c_double, C.c_double, C.POINTER(Cosmo)]
        for name in ("oracle_kdk_step", "oracle_kdk_step_explicit_drag"):
            f = getattr(L, name)
            f.restype = None
            f.argtypes = [dp, dp, dp, dp, dp, C.c_longlong, dp, C.c_double, C.c_double, C.c_double,
                          C.POINTER(Cosmo)]
        L.oracle_kdk_coeffs.restype = None
        L.oracle_kdk_coeffs.argtypes = [C.c_double, C.c_double, C.c_double, C.POINTER(Cosmo), dp]
        L.oracle_momentum.restype = None
        L.oracle_momentum.argtypes = [dp, dp, C.c_longlong, dp]
        L.oracle_timestep.restype = C.c_double
        L.oracle_timestep.argtypes = [dp, dp, dp, C.c_longlong, C.c_double, C.c_double, C.c_double, C.c_double]
        L.oracle_force_residual.restype = None
        L.oracle_force_residual.argtypes = [dp, dp, C.c_longlong, C.c_double, dp]
        L.oracle_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def spline_F(r: float, h: float) -> float:
    return lib().oracle_spline_F(float(r), float(h))


def forces(pos, mass, soft, idx=None, reverse_j: bool = False) -> np.ndarray:
    """acc (3, count) for all particles or for the index list `idx` (G = 1, no a^-3)."""
    pos, mass, soft = _f64(pos), _f64(mass), _f64(soft)
    n = mass.shape[0]
    assert pos.shape == (3, n) and soft.shape == (n,)
    if idx is None:
        acc = np.empty((3, n))
        lib().oracle_forces(_dp(pos), _dp(mass), _dp(soft), n, None, 0, _dp(acc), int(reverse_j))
    else:
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        acc = np.empty((3, idx.shape[0]))
        lib().oracle_forces(_dp(pos), _dp(mass), _dp(soft), n,
                            idx.ctypes.data_as(C.POINTER(C.c_longlong)), idx.shape[0], _dp(acc),
                            int(reverse_j))
    return acc


def _periodic(fn, pos, mass, soft, L, idx):
    pos, mass, soft = _f64(pos), _f64(mass), _f64(soft)
    n = mass.shape[0]
    assert pos.shape == (3, n) and soft.shape == (n,)
    if idx is None:
        acc = np.empty((3, n))
        fn(_dp(pos), _dp(mass), _dp(soft), n, float(L), None, 0, _dp(acc))
    else:
        idx = np.ascontiguousarray(idx, dtype=np.int64)
        assert idx.ndim == 1 and (idx >= 0).all() and (idx < n).all()
        acc = np.empty((3, idx.shape[0]))
        fn(_dp(pos), _dp(mass), _dp(soft), n, float(L), idx.ctypes.data_as(C.POINTER(C.c_longlong)), idx.shape[0], _dp(acc))
    return acc


def forces_quasi_periodic(pos, mass, soft, L: float, idx=None) -> np.ndarray:
    """Eq. 5 (L65-70) leading term only: nearest-image pair forces in a cubic box of side L; acc (3, N), G = 1.
    idx: evaluate only these particles (against all N sources); acc is then (3, len(idx))."""
    return _periodic(lib().oracle_forces_quasi_periodic, pos, mass, soft, L, idx)


def forces_periodic_images(pos, mass, soft, L: float, idx=None) -> np.ndarray:
    """Eq. 5 (L65-70) with the paper's cut |x - nL| < 2.6 L over the periodic images; acc (3, N), G = 1.
    idx: evaluate only these particles (against all N sources); acc is then (3, len(idx))."""
    return _periodic(lib().oracle_forces_periodic_images, pos, mass, soft, L, idx)


def hubble(a: float, cosmo: dict) -> float:
    c = Cosmo(**cosmo)
    return lib().oracle_hubble(float(a), C.byref(c))


def rk4_scale_factor(a: float, dt: float, cosmo: dict) -> float:
    c = Cosmo(**cosmo)
    return lib().oracle_rk4_scale_factor(float(a), float(dt), C.byref(c))


def kdk_step(pos, vel, acc, mass, soft, a: float, dt: float, G: float, B: float, cosmo: dict,
             explicit_drag: bool = False) -> float:
    """In-place KDK step on fp64 C-contiguous (3, N) arrays; returns a_{n+1}."""
    for arr in (pos, vel, acc):
        assert arr.dtype == np.float64 and arr.flags.c_contiguous and arr.shape == pos.shape
    mass, soft = _f64(mass), _f64(soft)
    c = Cosmo(**cosmo)
    a_box = C.c_double(a)
    fn = lib().oracle_kdk_step_explicit_drag if explicit_drag else lib().oracle_kdk_step
    fn(_dp(pos), _dp(vel), _dp(acc), _dp(mass), _dp(soft), mass.shape[0], C.byref(a_box),
       float(dt), float(G), float(B), C.byref(c))
    return a_box.value


def kdk_coeffs(a: float, dt: float, G: float, cosmo: dict) -> dict:
    c = Cosmo(**cosmo)
    out = np.empty(6)
    lib().oracle_kdk_coeffs(float(a), float(dt), float(G), C.byref(c), _dp(out))
    return dict(alpha_open=out[0], beta_open=out[1], gamma=out[2], alpha_close=out[3],
                beta_close=out[4], a_next=out[5])


def momentum(vel, mass) -> np.ndarray:
    vel, mass = _f64(vel), _f64(mass)
    out = np.empty(4)
    lib().oracle_momentum(_dp(vel), _dp(mass), mass.shape[0], _dp(out))
    return out


def timestep(pos, acc, soft, coef: float, B: float, eps: float, dt_max: float) -> float:
    """PAPER.md Eq. 12 (L113-116): global adaptive step min[dt_max, min_i sqrt(2 * 2.8 h_i * eps / |A_i|)],
    A_i = coef (acc_i + B x_i)."""
    pos, acc, soft = _f64(pos), _f64(acc), _f64(soft)
    n = soft.shape[0]
    assert pos.shape == (3, n) and acc.shape == (3, n)
    return float(lib().oracle_timestep(_dp(pos), _dp(acc), _dp(soft), n, coef, B, eps, dt_max))


def force_residual(pos, acc, B: float) -> np.ndarray:
    """Glass-generation monitor: [sum_i |acc_i + B x_i|^2, max_i |acc_i + B x_i|]."""
    pos, acc = _f64(pos), _f64(acc)
    assert pos.shape == acc.shape and pos.shape[0] == 3
    out = np.zeros(2)
    lib().oracle_force_residual(_dp(pos), _dp(acc), pos.shape[1], B, _dp(out))
    return out


def num_threads() -> int:
    return int(lib().oracle_num_threads())


# ---------------------------------------------------------------- schedule scalars (pure Python)

def cosmic_time_flat_lcdm(a: float, cosmo: dict) -> float:
    """Closed form of Eq. 1 for Omega_r = Omega_k = 0, Omega_L > 0 (reading #10):
    t(a) = 2/(3 H0 sqrt(OL)) asinh( sqrt(OL/Om) a^{3/2} )."""
    om, ol, h0 = cosmo["Omega_m"], cosmo["Omega_L"], cosmo["H0"]
    return 2.0 / (3.0 * h0 * math.sqrt(ol)) * math.asinh(math.sqrt(ol / om) * a ** 1.5)


def ln_a_schedule(a0: float, a1: float, n_steps: int, cosmo: dict) -> np.ndarray:
    """dt_n = t(a_{n+1}) - t(a_n) for a_n = a0 (a1/a0)^{n/n_steps} (config 4, reading #10)."""
    a = a0 * (a1 / a0) ** (np.arange(n_steps + 1) / n_steps)
    t = np.array([cosmic_time_flat_lcdm(x, cosmo) for x in a])
    return np.diff(t)


def growth_rate(a: float, cosmo: dict, n: int = 20001) -> float:
    """f = dlnD/dlna with D(a) of PAPER.md Eq. 19 (L255), D ~ H(a) int_0^a da'/(a' H(a'))^3
    (reading #12: the normalisation cancels).  Composite Simpson in u = a'^{3/2}-free form."""
    # integrand 1/(a' H)^3 ~ a'^{3/2} near 0 for matter domination; substitute a' = s^2
    s = np.linspace(0.0, math.sqrt(a), n)
    ap = s * s
    with np.errstate(divide="ignore", invalid="ignore"):
        H = np.array([hubble(x, cosmo) if x > 0 else np.inf for x in ap])
        g = 2.0 * s / (ap * H) ** 3
    g[0] = 0.0
    hstep = s[1] - s[0]
    integral = hstep / 3.0 * (g[0] + g[-1] + 4.0 * g[1:-1:2].sum() + 2.0 * g[2:-1:2].sum())
    Ha = hubble(a, cosmo)
    eps = 1e-6 * a
    dlnH = (math.log(hubble(a + eps, cosmo)) - math.log(hubble(a - eps, cosmo))) / (
        math.log(a + eps) - math.log(a - eps))
    return dlnH + a / ((a * Ha) ** 3 * integral)
