"""-m "not gpu": the C-ABI library builds/loads, exports every symbol include/steps.h declares,
and its host-side scalar logic (Friedmann H(a), RK4 a(t), the KDK coefficient schedule)
agrees with the oracle's independently written versions.  No device compute here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1811_05903_b200 import steps as S

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
LCDM = dict(H0=0.0288675134594813, Omega_m=0.3, Omega_r=0.0, Omega_L=0.7, Omega_k=0.0)
GEN = dict(H0=0.05, Omega_m=0.27, Omega_r=1e-4, Omega_L=0.7, Omega_k=0.0299)


def declared_functions():
    text = open(os.path.join(ROOT, "include", "steps.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(steps_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = S.lib()
    names = declared_functions()
    assert len(names) >= 18 and "steps_forces" in names and "steps_kdk_step" in names
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/steps.h but not exported"
    assert sorted(S.EXPORTS) == names, "binding's EXPORTS list and the header disagree"


def test_binding_has_the_same_names():
    for n in declared_functions():
        if n in ("steps_strerror", "steps_last_cuda_error"):
            continue
        assert callable(getattr(S, n)), n


def test_strerror_version_workspace():
    L = S.lib()
    assert L.steps_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4, -99):
        assert len(L.steps_strerror(code)) > 0
    assert S.steps_version() >= 100
    assert S.steps_workspace_bytes(0) == 0
    assert S.steps_workspace_bytes(1 << 20) >= (1 << 20) * 40
    assert S.steps_kernel_launch_count() >= 0
    with pytest.raises(S.StepsError):
        S.steps_set_option("no-such-key", 1)


def test_argument_checks_without_a_device():
    L = S.lib()
    assert L.steps_forces(None, None, None, 4, None, None) == S.EINVAL
    assert L.steps_forces_mixed(None, None, None, 4, None, None) == S.EINVAL
    assert L.steps_forces_range(None, None, None, 4, 0, 4, None, 0, None) == S.EINVAL
    assert L.steps_forces_host(None, None, None, 4, None, 0, None) == S.EINVAL
    assert L.steps_kick_drift(None, None, None, 4, None, None) == S.EINVAL
    assert L.steps_momentum(None, None, 4, None, None) == S.EINVAL
    assert L.steps_forces_periodic(None, None, None, 4, 1.0, None, None) == S.EINVAL
    assert L.steps_forces_quasi_periodic(None, None, None, 4, 1.0, None, 0, None) == S.EINVAL
    assert L.steps_kdk_step_adaptive(None, None, None, None, None, 4, None, None, 1.0, 0.0, 0.025, 1.0, 0, None) == S.EINVAL
    assert L.steps_kick_close_adaptive(None, None, None, 4, None, 0.0, None) == S.EINVAL
    assert L.steps_force_residual(None, None, 4, 0.0, None, None) == S.EINVAL
    assert L.steps_timestep(None, None, None, 4, 1.0, 0.0, 0.025, 1.0, None, None) == S.EINVAL
    assert L.steps_reserve(0) == S.EINVAL
    assert L.steps_kdk_schedule(1.0, 0.1, 1.0, None, None) == S.EINVAL


@pytest.mark.parametrize("cosmo", [LCDM, GEN])
def test_host_scalars_match_oracle(oracle, cosmo):
    c = S.Cosmology(**cosmo)
    for a in (1 / 51, 0.1, 0.5, 1.0):
        assert S.steps_hubble(a, c) == pytest.approx(oracle.hubble(a, cosmo), rel=1e-15)
        for dt in (1e-3, 0.05, 0.4):
            assert S.steps_scale_factor_rk4(a, dt, c) == pytest.approx(oracle.rk4_scale_factor(a, dt, cosmo), rel=1e-14)
            lib_c = S.steps_kdk_schedule(a, dt, 1.7, c)
            ora_c = oracle.kdk_coeffs(a, dt, 1.7, cosmo)
            for k in lib_c:
                assert lib_c[k] == pytest.approx(ora_c[k], rel=1e-13), k


def test_static_mode_schedule(oracle):
    c = S.Cosmology(0, 0, 0, 0, 0)
    s = S.steps_kdk_schedule(1.0, 0.25, 2.0, c)
    assert s == dict(alpha_open=1.0, beta_open=0.25, gamma=0.25, alpha_close=1.0, beta_close=0.25, a_next=1.0)
    o = oracle.kdk_coeffs(1.0, 0.25, 2.0, oracle.STATIC)
    assert all(s[k] == o[k] for k in s)


def test_full_ln_a_schedule_lands_on_a_equals_one(oracle):
    """Config 4's schedule (reading #10): 200 ln-a-uniform steps, a advanced by the LIBRARY's RK4."""
    c = S.Cosmology(**LCDM)
    a = 1 / 51
    for dt in oracle.ln_a_schedule(1 / 51, 1.0, 200, LCDM):
        a = S.steps_kdk_schedule(a, float(dt), 1.0, c)["a_next"]
    assert a == pytest.approx(1.0, rel=1e-8)
