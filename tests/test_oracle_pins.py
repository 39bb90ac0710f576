"""Pins for the CPU oracle (oracle/steps_oracle.c) against what the paper and the physics fix.

None of these re-types the oracle's formula or re-calls its routine as the expected value:
the pair law is pinned by Gauss's law on the cubic-spline density kernel the paper cites
([1, 15] at PAPER.md L51), exact rational hand values of Eq. 4, continuity and exactness
properties; the force sum by two-body closed forms, the shell theorem, Newton's third law,
symmetries and an independent numpy-longdouble brute force; the integrator by closed-form
solutions and convergence orders.  A dropped term, wrong sign, wrong index or transposed
operand in the oracle fails at least one of them."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy import integrate

from paper_1811_05903_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------ independent ingredients

def ml_kernel_density(r, h):
    """Monaghan-Lattanzio cubic spline with support h (GADGET-2 normalisation), the kernel the
    paper cites for its softening (refs [1, 15]).  NOT Eq. 4: this is the density."""
    u = r / h
    if u < 0.5:
        return 8.0 / (math.pi * h ** 3) * (1.0 - 6.0 * u * u + 6.0 * u ** 3)
    if u < 1.0:
        return 8.0 / (math.pi * h ** 3) * 2.0 * (1.0 - u) ** 3
    return 0.0


def gauss_law_F(r, h):
    """Force magnitude per unit mass from the kernel by Gauss's law: M(<r)/r^2, M by quadrature."""
    pts = [p for p in (0.5 * h, h) if p < r]
    m, _ = integrate.quad(lambda s: 4.0 * math.pi * s * s * ml_kernel_density(s, h), 0.0, min(r, h),
                          points=pts or None, epsabs=0, epsrel=1e-13, limit=200)
    return m / (r * r)


def enclosed_mass_ld(u):
    """Enclosed kernel mass M(u), u = r/h, from integrating the kernel analytically in numpy
    longdouble (derivation in the module docstring of this test; not Eq. 4's coefficients)."""
    u = np.longdouble(u)
    if u < 0.5:
        return 32 * (u ** 3 / 3 - 6 * u ** 5 / 5 + u ** 6)
    if u < 1:
        P = u ** 3 / 3 - 3 * u ** 4 / 4 + 3 * u ** 5 / 5 - u ** 6 / 6
        return 1 - 64 * (np.longdouble(1) / 60 - P)
    return np.longdouble(1)


def brute_force_ld(pos, mass, soft):
    """Term-by-term longdouble force sum via Gauss's law on the kernel (tiny N only)."""
    n = mass.shape[0]
    p = pos.astype(np.longdouble)
    acc = np.zeros((3, n), dtype=np.longdouble)
    for i in range(n):
        for j in range(n):
            if i == j:
                continue
            d = p[:, j] - p[:, i]
            r = np.sqrt(np.sum(d * d))
            if r == 0:
                continue
            h = np.longdouble(soft[i]) + np.longdouble(soft[j])
            acc[:, i] += np.longdouble(mass[j]) * enclosed_mass_ld(r / h) / (r * r) * d / r
    return acc


def rel_err(a, b):
    return np.linalg.norm(a - b, axis=0) / np.linalg.norm(b, axis=0)


# ------------------------------------------------------------------ pair law (Eq. 3-4)

def test_eq4_exact_rational_values(oracle):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "eq4_exact_values.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 8
    for r_s, branch, frac_s, dec_s in rows:
        r, want = float(Fraction(r_s)), float(Fraction(frac_s))
        assert abs(want - float(dec_s)) < 1e-15
        # evaluate on the requested side of a branch point
        eps = {"1": -1, "2": (+1 if r == 0.5 else -1), "3": +1}[branch] * 1e-13 if r in (0.5, 1.0) else 0.0
        got = oracle.spline_F(r * (1 + eps), 1.0)
        assert got == pytest.approx(want, rel=2e-12), (r_s, branch)


@pytest.mark.parametrize("h", [0.02, 1.0, 3.7])
def test_pair_law_is_gauss_law_of_cubic_spline_kernel(oracle, h):
    for u in [1e-3, 0.05, 0.2, 0.41415, 0.49999, 0.5, 0.50001, 0.6, 0.75, 0.9, 0.99999, 1.0, 1.5, 7.0]:
        r = u * h
        assert oracle.spline_F(r, h) == pytest.approx(gauss_law_F(r, h), rel=5e-12), u


def test_pair_law_continuity_scaling_maximum(oracle):
    F = oracle.spline_F
    for h in (0.3, 1.0, 5.0):
        for rb in (0.5 * h, h):                         # C0 and C1 at both branch points
            d = 1e-7 * h
            assert F(rb - 1e-14 * h, h) == pytest.approx(F(rb + 1e-14 * h, h), rel=1e-11)
            dl = (F(rb - d, h) - F(rb - 2 * d, h)) / d
            dr = (F(rb + 2 * d, h) - F(rb + d, h)) / d
            assert dl == pytest.approx(dr, rel=1e-4)
        assert F(0.37 * h, h) == pytest.approx(F(0.37, 1.0) / h ** 2, rel=1e-14)   # F(r,h) = F(r/h,1)/h^2
    # derivative values quoted in SURVEY.md 8(c.4)#1: dF/dr = -32/15/h^3 at h/2, -2/h^3 at h
    d = 1e-6
    assert (F(0.5 + d, 1) - F(0.5 - d, 1)) / (2 * d) == pytest.approx(-32.0 / 15.0, rel=1e-6)
    assert (F(1 + d, 1) - F(1 - d, 1)) / (2 * d) == pytest.approx(-2.0, rel=1e-5)
    # single maximum 2.63127/h^2 at r = 0.41415 h
    rs = np.linspace(1e-4, 1.2, 120001)
    fs = np.array([F(r, 1.0) for r in rs])
    k = int(np.argmax(fs))
    assert rs[k] == pytest.approx(0.41415, abs=2e-5) and fs[k] == pytest.approx(2.63127, abs=1e-5)
    assert np.all(np.diff(fs[:k]) > 0) and np.all(np.diff(fs[k + 1:]) < 0)
    # centre of a uniform-density core: F -> (4 pi/3) rho(0) r, rho(0) = 8/(pi h^3)
    assert F(1e-6, 1.0) / 1e-6 == pytest.approx(32.0 / 3.0, rel=1e-5)


def test_pair_law_exactly_newtonian_outside_h(oracle):
    rng = np.random.default_rng(1)
    for _ in range(200):
        h = 10 ** rng.uniform(-3, 1)
        r = h * (1.0 + 10 ** rng.uniform(-12, 3))
        assert oracle.spline_F(r, h) == 1.0 / (r * r)     # bitwise: same expression, no spline term


# ------------------------------------------------------------------ force sum (Eq. 8, first term)

@pytest.mark.parametrize("u", [0.05, 0.3, 0.5, 0.8, 1.0, 4.0, 1e4])
def test_two_body_closed_form(oracle, u):
    m = np.array([0.7, 0.05])
    soft = np.array([0.11, 0.023])
    h = soft.sum()
    n = np.array([0.36, -0.48, 0.8])                      # unit vector from 1 to 2
    x1 = np.array([0.3, -1.2, 2.5])
    pos = np.stack([x1, x1 + u * h * n], axis=1)
    acc = oracle.forces(pos, m, soft)
    F = gauss_law_F(u * h, h)
    np.testing.assert_allclose(acc[:, 0], +m[1] * F * n, rtol=2e-11, atol=0)   # 1 pulled toward 2
    np.testing.assert_allclose(acc[:, 1], -m[0] * F * n, rtol=2e-11, atol=0)
    np.testing.assert_allclose(m[0] * acc[:, 0] + m[1] * acc[:, 1], 0, atol=1e-15 * m[0] * m[1] * F)
    if u > 1.0:                                           # exactly GM/r^2 beyond the softening
        r_act = np.linalg.norm(pos[:, 1] - pos[:, 0])     # the separation as stored (x1 + u h n rounds)
        np.testing.assert_allclose(np.linalg.norm(acc[:, 0]), m[1] / r_act ** 2, rtol=4e-16)


def test_pair_softening_is_the_sum_of_both(oracle):
    """Reading #3 (Eq. 2, Eq. 8): the spline argument is h_i + h_j -- not max, not mean."""
    pos = np.array([[0.0, 1.0], [0, 0], [0, 0]])
    m = np.array([1.0, 1.0])
    a_sum = oracle.forces(pos, m, np.array([0.9, 0.6]))[0, 0]       # h = 1.5 > r: softened
    assert a_sum == pytest.approx(gauss_law_F(1.0, 1.5), rel=1e-11)
    assert a_sum < 0.999                                            # max(0.9,0.6)<1 would give exactly 1
    assert oracle.forces(pos, m, np.array([0.5, 0.5]))[0, 0] == 1.0  # h = 1.0 = r: Newtonian


def test_self_pair_and_coincident_particles(oracle):
    """Reading #4: j = i skipped; distinct coincident particles contribute 0 (F(0, h) = 0)."""
    pos = np.zeros((3, 1))
    assert np.all(oracle.forces(pos, np.ones(1), np.full(1, 0.1)) == 0.0)
    pos = np.array([[0.0, 0.0, 3.0], [0, 0, 0], [0, 0, 0]])
    acc = oracle.forces(pos, np.array([1.0, 2.0, 4.0]), np.full(3, 0.1))
    assert np.all(np.isfinite(acc))
    np.testing.assert_allclose(acc[0], [4.0 / 9, 4.0 / 9, -3.0 / 9], rtol=1e-15)


def _polyhedra():
    phi = (1 + 5 ** 0.5) / 2
    tetra = [(1, 1, 1), (1, -1, -1), (-1, 1, -1), (-1, -1, 1)]
    octa = [(1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)]
    cube = [(i, j, k) for i in (-1, 1) for j in (-1, 1) for k in (-1, 1)]
    icosa = [p for a in (-1, 1) for b in (-phi, phi) for p in ((0, a, b), (a, b, 0), (b, 0, a))]
    dodeca = cube + [p for a in (-1 / phi, 1 / phi) for b in (-phi, phi) for p in ((0, a, b), (a, b, 0), (b, 0, a))]
    return dict(tetra=tetra, octa=octa, cube=cube, icosa=icosa, dodeca=dodeca)


@pytest.mark.parametrize("name", list(_polyhedra()))
@pytest.mark.parametrize("h", [0.01, 0.8])
def test_shell_theorem_regular_polyhedra_centre(oracle, name, h):
    v = np.array(_polyhedra()[name], dtype=float)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    pos = np.concatenate([np.zeros((1, 3)), v], axis=0).T.copy()
    n = pos.shape[1]
    acc = oracle.forces(pos, np.full(n, 1.0 / n), np.full(n, h))
    assert np.linalg.norm(acc[:, 0]) < 1e-15              # centre particle feels nothing
    radial = np.sum(acc[:, 1:] * pos[:, 1:], axis=0)      # vertices: purely radial, all equal
    assert np.allclose(radial, radial[0], rtol=1e-13) and radial[0] < 0
    assert np.max(np.linalg.norm(acc[:, 1:] - radial * pos[:, 1:], axis=0)) < 1e-14


def test_shell_theorem_fibonacci_shell(oracle):
    ns = 20000
    k = np.arange(ns) + 0.5
    ct = 1 - 2 * k / ns
    st = np.sqrt(1 - ct * ct)
    ph = math.pi * (1 + 5 ** 0.5) * k
    shell = np.stack([st * np.cos(ph), st * np.sin(ph), ct])
    probes = np.array([[0.0, 0.3, 0.0, 2.0, 0.0], [0.0, 0.1, -0.5, 0.0, 0.0], [0.0, 0.2, 0.2, 0.0, 5.0]])
    pos = np.concatenate([shell, probes], axis=1).copy()
    mass = np.concatenate([np.full(ns, 1.0 / ns), np.zeros(5)])
    acc = oracle.forces(pos, mass, np.full(ns + 5, 1e-4), idx=np.arange(ns, ns + 5))
    assert np.max(np.linalg.norm(acc[:, :3], axis=0)) < 2e-3          # inside: ~0 (sampling noise)
    for c in (3, 4):                                                  # outside: -M x/r^3
        r = np.linalg.norm(probes[:, c])
        np.testing.assert_allclose(acc[:, c], -probes[:, c] / r ** 3, rtol=0, atol=2e-3 / r ** 2)


def test_uniform_sphere_pair_sum_cancels_background_term(oracle):
    """Eq. 8 is 'derived from Newton's shell theorem' (L86): for a (statistically) uniform
    sphere the pair sum is -(M/R_sim^3) x, i.e. it cancels +B x with
    B = (4 pi/3) rho_bar = M/R_sim^3 (readings #6, #7).  Statistical pin (discreteness noise)."""
    rng = np.random.default_rng(11)
    n, R = 8192, 20.0
    d = rng.normal(size=(3, n))
    pos = np.ascontiguousarray(d / np.linalg.norm(d, axis=0) * R * rng.random(n) ** (1 / 3))
    idx = np.arange(0, n, 4)
    acc = oracle.forces(pos, np.full(n, 1.0 / n), np.full(n, 0.5), idx=idx)
    x = pos[:, idx]
    inner = np.linalg.norm(x, axis=0) < 0.8 * R
    slope = np.sum(acc[:, inner] * x[:, inner]) / np.sum(x[:, inner] ** 2)
    assert slope == pytest.approx(-1.0 / R ** 3, rel=0.03)


@pytest.mark.parametrize("n", [64, 1024, 4096])
def test_newtons_third_law(oracle, n):
    ps = synth.g0(n, seed=5, eps0=0.05)
    acc = oracle.forces(ps.pos, ps.mass, ps.soft)
    net = np.linalg.norm(acc @ ps.mass)
    scale = np.sum(ps.mass * np.linalg.norm(acc, axis=0))
    assert net / scale < 1e-15 * math.sqrt(n)


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_brute_force_longdouble_tiny_n(oracle, seed):
    rng = np.random.default_rng(seed)
    n = 8
    pos = rng.normal(size=(3, n))
    mass = rng.uniform(0.1, 1.0, n)
    soft = rng.uniform(0.05, 1.2, n)            # large: every branch of the spline is exercised
    u = np.array([np.linalg.norm(pos[:, i] - pos[:, j]) / (soft[i] + soft[j]) for i in range(n) for j in range(i)])
    assert (u < 0.5).any() and ((u >= 0.5) & (u < 1)).any() and (u >= 1).any()
    want = brute_force_ld(pos, mass, soft).astype(np.float64)
    got = oracle.forces(pos, mass, soft)
    assert np.max(rel_err(got, want)) < 1e-13


def test_symmetries(oracle):
    ps = synth.g0(512, seed=3, eps0=0.2)       # eps0 inflated: many softened pairs
    pos, m, h = ps.pos, ps.mass, ps.soft
    base = oracle.forces(pos, m, h)
    perm = np.random.default_rng(0).permutation(512)
    np.testing.assert_allclose(oracle.forces(pos[:, perm].copy(), m[perm], h[perm]), base[:, perm], rtol=1e-13, atol=1e-18)
    shift = np.array([[3.0], [-7.0], [11.0]])
    assert np.max(rel_err(oracle.forces(pos + shift, m, h), base)) < 1e-11
    q, _ = np.linalg.qr(np.random.default_rng(1).normal(size=(3, 3)))
    assert np.max(rel_err(oracle.forces(np.ascontiguousarray(q @ pos), m, h), q @ base)) < 1e-12
    lam = 3.0
    assert np.max(rel_err(oracle.forces(lam * pos, m, lam * h), base / lam ** 2)) < 1e-13
    assert np.max(rel_err(oracle.forces(pos, 2.0 * m, h), 2.0 * base)) == 0.0   # power of two: exact
    sub = np.array([0, 17, 511])
    assert np.array_equal(oracle.forces(pos, m, h, idx=sub), base[:, sub])


def test_summation_order_independence(oracle):
    ps = synth.g0(4096, seed=9)
    fwd = oracle.forces(ps.pos, ps.mass, ps.soft)
    rev = oracle.forces(ps.pos, ps.mass, ps.soft, reverse_j=True)
    assert np.max(rel_err(fwd, rev)) < 1e-15


# ------------------------------------------------------------------ background a(t) (Eq. 1)

EDS = dict(H0=0.7, Omega_m=1.0, Omega_r=0.0, Omega_L=0.0, Omega_k=0.0)
LCDM = dict(H0=0.0288675134594813, Omega_m=0.3, Omega_r=0.0, Omega_L=0.7, Omega_k=0.0)


def test_hubble_parameter_eq1(oracle):
    c = dict(H0=2.0, Omega_m=0.3, Omega_r=0.05, Omega_L=0.6, Omega_k=0.05)
    assert oracle.hubble(1.0, c) == pytest.approx(2.0, rel=1e-15)
    assert oracle.hubble(0.5, c) == pytest.approx(2.0 * math.sqrt(0.3 * 8 + 0.05 * 16 + 0.6 + 0.05 * 4), rel=1e-15)


def test_rk4_scale_factor_vs_closed_forms(oracle):
    # EdS: a = (3 H0 t/2)^(2/3)
    t0 = 2.0 / (3 * EDS["H0"]) * (1 / 51) ** 1.5
    t1 = 2.0 / (3 * EDS["H0"])
    errs = []
    for n in (100, 200, 400):
        a, dt = 1 / 51, (t1 - t0) / n
        for _ in range(n):
            a = oracle.rk4_scale_factor(a, dt, EDS)
        errs.append(abs(a - 1.0))
    assert errs[2] < 1e-5 and errs[0] / errs[1] > 8 and errs[1] / errs[2] > 8       # ~4th order (first steps >> t0)
    # flat LCDM: asinh closed form (reading #10), ln-a-uniform schedule of config 4
    dts = oracle.ln_a_schedule(1 / 51, 1.0, 200, LCDM)
    a = 1 / 51
    for k, dt in enumerate(dts):
        a = oracle.rk4_scale_factor(a, dt, LCDM)
        assert a == pytest.approx((1 / 51) * 51 ** ((k + 1) / 200), rel=1e-8)
    assert oracle.cosmic_time_flat_lcdm(1 / 51, LCDM) == pytest.approx(0.11577, rel=1e-4)
    assert oracle.cosmic_time_flat_lcdm(1.0, LCDM) == pytest.approx(33.3974, rel=1e-5)


def test_growth_rate_limits(oracle):
    assert oracle.growth_rate(0.3, EDS) == pytest.approx(1.0, abs=1e-6)             # D = a in EdS
    assert oracle.growth_rate(1.0, LCDM) == pytest.approx(0.3 ** 0.55, abs=5e-3)    # textbook fit


def test_growth_rate_flat_lcdm_closed_form(oracle):
    """Flat LCDM (Omega_r = Omega_k = 0): the growing mode of PAPER.md Eq. 19 (L255) has the closed form
    D(a) ~ a 2F1(1/3, 1; 11/6; x), x = -a^3 Omega_L/Omega_m, hence
    f = dlnD/dlna = 1 + 3 x F'(x)/F(x) with F' = (1/3 * 1 / (11/6)) 2F1(4/3, 2; 17/6; x).
    scipy's hypergeometric routine is independent of the oracle's quadrature of Eq. 19 (a wrong power of a'H, a wrong
    dlnH/dlna term or a sloppy quadrature fails at 1e-7).  f sets the initial velocities of config 4."""
    from scipy.special import hyp2f1
    for a in (1 / 51, 0.1, 0.3, 0.6, 1.0):
        x = -a ** 3 * LCDM["Omega_L"] / LCDM["Omega_m"]
        F = hyp2f1(1 / 3, 1.0, 11 / 6, x)
        dF = (1 / 3) / (11 / 6) * hyp2f1(4 / 3, 2.0, 17 / 6, x)
        f = 1.0 + 3.0 * x * dF / F
        assert oracle.growth_rate(a, LCDM) == pytest.approx(f, rel=2e-7), a


# ------------------------------------------------------------------ KDK integrator (Eq. 8-11)

def _one_particle(x0, v0):
    return (np.array([[x0], [0.0], [0.0]]), np.array([[v0], [0.0], [0.0]]), np.zeros((3, 1)),
            np.ones(1), np.full(1, 0.01))


def _run(oracle, pos, vel, acc, m, h, cosmo, a0, a1, n, G, B, explicit=False):
    eds_t = lambda a: 2.0 / (3 * cosmo["H0"]) * a ** 1.5
    a_grid = a0 * (a1 / a0) ** (np.arange(n + 1) / n)
    a = a0
    for k in range(n):
        a = oracle.kdk_step(pos, vel, acc, m, h, a, eds_t(a_grid[k + 1]) - eds_t(a_grid[k]), G, B, cosmo,
                            explicit_drag=explicit)
    return a


def test_drag_conserves_a2v_second_order(oracle):
    """G = 0, B = 0:  x'' = -2 H x'  =>  a^2 v conserved.  Reading #8's scheme is 2nd order
    (L96 'second order'); drag explicit in both half kicks is only 1st order."""
    def err(n, explicit):
        pos, vel, acc, m, h = _one_particle(0.0, 1.0)
        a = _run(oracle, pos, vel, acc, m, h, EDS, 1 / 51, 1.0, n, 0.0, 0.0, explicit)
        return a * a * vel[0, 0] / (1 / 51) ** 2 - 1.0
    e = [err(n, False) for n in (100, 200, 400)]
    assert abs(e[1]) < 1e-2 and 3.5 < e[0] / e[1] < 4.5 and 3.5 < e[1] / e[2] < 4.5
    assert e[0] == pytest.approx(-1.8e-2, rel=0.1)       # value quoted in SURVEY.md 8(c.5)
    x = [err(n, True) for n in (100, 200, 400)]
    assert 1.7 < x[0] / x[1] < 2.3 and abs(x[1]) > 10 * abs(e[1])


def test_background_term_closed_form(oracle):
    """N = 1, EdS:  x'' + 2 H x' = (H0^2/2) a^-3 x  has the exact solutions x ~ a^(1/2) and
    x ~ a^-1 (readings #6, #7): B = (4 pi/3) rho_bar = H0^2/2 in G = 1 units, carrying a^-3."""
    B = 0.5 * EDS["H0"] ** 2
    a0 = 1 / 51
    H_init = EDS["H0"] * a0 ** -1.5
    e = []
    for n in (100, 200, 400):
        pos, vel, acc, m, h = _one_particle(1.0, 0.5 * H_init * 1.0)
        _run(oracle, pos, vel, acc, m, h, EDS, a0, 1.0, n, 1.0, B)
        e.append(pos[0, 0] / math.sqrt(51.0) - 1.0)
    assert abs(e[1]) < 1e-3 and 3.5 < e[0] / e[1] < 4.5 and 3.5 < e[1] / e[2] < 4.5
    pos, vel, acc, m, h = _one_particle(1.0, -H_init * 1.0)           # decaying solution x ~ 1/a
    _run(oracle, pos, vel, acc, m, h, EDS, a0, 4 * a0, 400, 1.0, B)
    assert pos[0, 0] == pytest.approx(0.25, rel=2e-3)


def test_kepler_orbit_static_newtonian(oracle):
    """a = 1, H = 0, B = 0 (L92): two-body orbit.  Angular momentum to rounding, energy error
    bounded and ~ dt^2, time reversible."""
    m = np.array([1.0, 0.25])
    h = np.array([0.01, 0.01])

    def setup():
        pos = np.array([[-0.2, 0.8], [0.0, 0.0], [0.0, 0.0]])
        vy = math.sqrt(m.sum() / 1.0) * 1.1            # slightly eccentric
        vel = np.array([[0.0, 0.0], [-0.2 * vy, 0.8 * vy], [0.0, 0.0]])
        return pos, vel, oracle.forces(pos, m, h)

    def energy(pos, vel):
        r = np.linalg.norm(pos[:, 0] - pos[:, 1])
        return 0.5 * np.sum(m * np.sum(vel * vel, axis=0)) - m[0] * m[1] / r

    def angmom(pos, vel):
        return np.sum(m * (pos[0] * vel[1] - pos[1] * vel[0]))

    drift = []
    for n in (400, 800):
        pos, vel, acc = setup()
        e0, l0 = energy(pos, vel), angmom(pos, vel)
        worst = 0.0
        for _ in range(n):
            oracle.kdk_step(pos, vel, acc, m, h, 1.0, 8.0 / n, 1.0, 0.0, oracle.STATIC)
            worst = max(worst, abs(energy(pos, vel) / e0 - 1))
        assert abs(angmom(pos, vel) / l0 - 1) < 1e-13
        drift.append(worst)
    assert drift[1] < 1e-3 and 3.3 < drift[0] / drift[1] < 4.7
    pos, vel, acc = setup()
    p0, v0 = pos.copy(), vel.copy()
    for _ in range(200):
        oracle.kdk_step(pos, vel, acc, m, h, 1.0, 0.01, 1.0, 0.0, oracle.STATIC)
    vel *= -1
    for _ in range(200):
        oracle.kdk_step(pos, vel, acc, m, h, 1.0, 0.01, 1.0, 0.0, oracle.STATIC)
    np.testing.assert_allclose(pos, p0, atol=1e-12)
    np.testing.assert_allclose(-vel, v0, atol=1e-12)


def test_kdk_coefficient_form_equals_literal_step(oracle):
    """The (alpha, beta, gamma) form the library's fused kernel consumes reproduces the literal step."""
    ps = synth.config4_ics(256, synth.SEED_BASE + 4, vel_factor=0.3)
    B = 1.0 / ps.r_cut ** 3
    a0, dt = 1 / 51, 0.02
    pos, vel = ps.pos.copy(), ps.vel.copy()
    acc = oracle.forces(pos, ps.mass, ps.soft)
    c = oracle.kdk_coeffs(a0, dt, 1.0, LCDM)
    v1 = c["alpha_open"] * vel + c["beta_open"] * (acc + B * pos)
    x1 = pos + c["gamma"] * v1
    acc1 = oracle.forces(x1, ps.mass, ps.soft)
    v2 = c["alpha_close"] * v1 + c["beta_close"] * (acc1 + B * x1)
    a1 = oracle.kdk_step(pos, vel, acc, ps.mass, ps.soft, a0, dt, 1.0, B, LCDM)
    assert a1 == c["a_next"]
    np.testing.assert_allclose(pos, x1, rtol=1e-14)
    np.testing.assert_allclose(vel, v2, rtol=1e-12, atol=1e-18)
    p = oracle.momentum(vel, ps.mass)
    assert np.linalg.norm(p[:3]) / p[3] < 1e-12


# ---- diagnostics: P = sum m v, sum m |v| -----------------------------------------------------
def test_periodic_oracles_sampled_equals_full(oracle):
    """The idx argument of the two periodic oracles only selects which particles are evaluated."""
    rng = np.random.default_rng(11)
    n, L = 40, 1.1
    pos, mass, soft = rng.uniform(0, L, (3, n)), rng.uniform(0.5, 1.5, n), np.full(n, 0.02)
    idx = np.array([3, 17, 39, 0])
    for fn in (oracle.forces_quasi_periodic, oracle.forces_periodic_images):
        np.testing.assert_array_equal(fn(pos, mass, soft, L, idx=idx), fn(pos, mass, soft, L)[:, idx])


def test_momentum_hand_values_and_brute_force(oracle):
    """Three particles with hand-typed values: m = (1, 2, 4), v_1 = (3, 4, 0), v_2 = (0, -6, 8), v_3 = (-2, 1, 2),
    |v| = (5, 10, 3):  sum m v = (3 - 8, 4 - 12 + 4, 16 + 8) = (-5, -4, 24),  sum m |v| = 5 + 20 + 12 = 37.
    All four outputs differ, the components differ from each other, and sum m v^2 = 261 != 37, so a swapped index,
    a missing square root or a missing mass fails.  Then a numpy-longdouble brute force on random data."""
    vel = np.array([[3.0, 0.0, -2.0], [4.0, -6.0, 1.0], [0.0, 8.0, 2.0]])
    mass = np.array([1.0, 2.0, 4.0])
    np.testing.assert_array_equal(oracle.momentum(vel, mass), [-5.0, -4.0, 24.0, 37.0])
    rng = np.random.default_rng(7)
    n = 1000
    vel = rng.normal(size=(3, n)) * np.array([[1.0], [10.0], [100.0]])
    mass = rng.uniform(0.1, 5.0, size=n) * 10.0 ** rng.integers(-6, 3, size=n)
    vl, ml = vel.astype(np.longdouble), mass.astype(np.longdouble)
    want = np.array([*(ml * vl).sum(axis=1), (ml * np.sqrt((vl * vl).sum(axis=0))).sum()], dtype=np.longdouble)
    got = oracle.momentum(vel, mass)
    scale = (ml * np.abs(vl)).sum(axis=1)
    assert np.all(np.abs(got[:3] - want[:3]) <= 4e-16 * scale)          # compensated: error ~ 1 ulp of sum |m v|
    assert abs(got[3] - want[3]) <= 4e-16 * want[3]


# ---- Eq. 12 (L113-116): adaptive global time step --------------------------------------------------------------
def _two_body(d, m1, m2, h1, h2):
    pos = np.array([[0.0, d], [0.0, 0.0], [0.0, 0.0]])
    return pos, np.array([m1, m2]), np.array([h1, h2])


def test_timestep_two_body_closed_form(oracle):
    """Two bodies at separation d >= h1 + h2: |A_1| = G m_2 / d^2, |A_2| = G m_1 / d^2 (Eq. 4 third case), so
    dt = min_i sqrt(2 * 2.8 h_i * eps * d^2 / (G m_other)) -- typed out here from Eq. 12, not from the oracle."""
    d, m1, m2, h1, h2, G, eps = 3.0, 2.0, 5.0, 0.3, 0.1, 1.7, 0.025
    pos, mass, soft = _two_body(d, m1, m2, h1, h2)
    acc = oracle.forces(pos, mass, soft)
    dt = oracle.timestep(pos, acc, soft, G, 0.0, eps, 1e30)
    dt1 = math.sqrt(2 * 2.8 * h1 * eps * d * d / (G * m2))
    dt2 = math.sqrt(2 * 2.8 * h2 * eps * d * d / (G * m1))
    assert dt == pytest.approx(min(dt1, dt2), rel=1e-14)
    assert min(dt1, dt2) == dt2 and dt1 / dt2 > 1.05          # the pin would notice the wrong particle being picked


def test_timestep_scalings_clamp_and_zero_acceleration(oracle):
    rng = np.random.default_rng(12)
    n = 200
    pos = rng.normal(size=(3, n)); acc = rng.normal(size=(3, n)); soft = rng.uniform(0.01, 0.1, n)
    base = oracle.timestep(pos, acc, soft, 1.0, 0.0, 0.01, 1e30)
    # dt ~ sqrt(eps), ~ sqrt(h), ~ |A|^-1/2 (Eq. 12)
    assert oracle.timestep(pos, acc, soft, 1.0, 0.0, 0.04, 1e30) == pytest.approx(2 * base, rel=1e-14)
    assert oracle.timestep(pos, acc, 4 * soft, 1.0, 0.0, 0.01, 1e30) == pytest.approx(2 * base, rel=1e-14)
    assert oracle.timestep(pos, acc, soft, 4.0, 0.0, 0.01, 1e30) == pytest.approx(base / 2, rel=1e-14)
    assert oracle.timestep(pos, 4 * acc, soft, 1.0, 0.0, 0.01, 1e30) == pytest.approx(base / 2, rel=1e-14)
    # dt_max clamps; a particle at rest in the force field puts no limit
    assert oracle.timestep(pos, acc, soft, 1.0, 0.0, 0.01, base / 3) == base / 3
    assert oracle.timestep(pos, 0 * acc, soft, 1.0, 0.0, 0.01, 7.5) == 7.5
    # the background term enters A_i = coef (acc_i + B x_i): with acc = -B x the particle feels nothing
    assert oracle.timestep(pos, -0.3 * pos, soft, 2.0, 0.3, 0.01, 7.5) == 7.5


def test_timestep_against_numpy_brute_force(oracle):
    rng = np.random.default_rng(13)
    n = 1000
    pos = rng.normal(size=(3, n)); acc = rng.normal(size=(3, n)) * 10.0 ** rng.uniform(-3, 3, n)
    soft = 10.0 ** rng.uniform(-3, 0, n)
    coef, B, eps = 0.37, 0.011, 0.025
    A = np.linalg.norm(coef * (acc + B * pos), axis=0)
    want = float(np.min(np.sqrt(2 * 2.8 * soft * eps / A)))
    assert oracle.timestep(pos, acc, soft, coef, B, eps, 1e30) == pytest.approx(want, rel=1e-14)


# ---- glass generation monitor (section 3.1): net force residual g_i = acc_i + B x_i -------------------
def test_force_residual_closed_forms_and_brute_force(oracle):
    rng = np.random.default_rng(31)
    n, B = 500, 0.37
    pos = rng.normal(size=(3, n))
    # a particle alone in the background (pair sum 0): g = B x exactly; a particle in exact balance: g = 0
    r = oracle.force_residual(pos, np.zeros((3, n)), B)
    assert r[0] == pytest.approx(B * B * np.sum(pos ** 2), rel=1e-14)
    assert r[1] == pytest.approx(B * np.max(np.linalg.norm(pos, axis=0)), rel=1e-15)
    assert np.all(oracle.force_residual(pos, -B * pos, B) == 0.0)
    acc = rng.normal(size=(3, n))
    g = np.linalg.norm(acc.astype(np.longdouble) + np.longdouble(B) * pos.astype(np.longdouble), axis=0)
    r = oracle.force_residual(pos, acc, B)
    assert r[0] == pytest.approx(float(np.sum(g * g)), rel=1e-15)
    assert r[1] == pytest.approx(float(np.max(g)), rel=1e-15)


def test_force_residual_of_a_uniform_ball_is_small_and_reversed_gravity_lowers_it(oracle):
    """Shell theorem (L86): inside a uniform ball of total mass M and radius R the pair sum is -(M/R^3) x, so with
    B = M/R^3 (reading #7) the residual of a dense random sampling is only its Poisson noise.  Evolving that sampling
    with REVERSED gravity in EdS (L245: G < 0 in the kick, nothing else changes) must lower the rms residual."""
    rng = np.random.default_rng(32)
    n, R = 1500, 1.0
    u = rng.normal(size=(3, n)); u /= np.linalg.norm(u, axis=0)
    pos = np.ascontiguousarray(u * R * rng.uniform(0, 1, n) ** (1 / 3))
    mass = np.full(n, 1.0 / n); soft = np.full(n, 0.5 * (4 * np.pi / 3 / n) ** (1 / 3) * R)
    B = 1.0 / R ** 3
    acc = oracle.forces(pos, mass, soft)
    inner = np.linalg.norm(pos, axis=0) < 0.6 * R
    rms_pair = np.sqrt(np.mean(np.sum(acc[:, inner] ** 2, axis=0)))
    g = acc + B * pos
    rms0 = np.sqrt(np.mean(np.sum(g[:, inner] ** 2, axis=0)))
    assert rms0 < 0.5 * rms_pair                      # background term cancels the mean pull (sign and size of B)
    cosmo = dict(H0=math.sqrt(2 * B), Omega_m=1.0, Omega_r=0.0, Omega_L=0.0, Omega_k=0.0)
    vel = np.zeros_like(pos); a = 0.05
    r_start = oracle.force_residual(pos, acc, B)[0]
    for _ in range(40):
        dt = oracle.timestep(pos, acc, soft, 1.0 / a ** 3, B, 0.025, 1e30)
        a = oracle.kdk_step(pos, vel, acc, mass, soft, a, dt, -1.0, B, cosmo)        # G = -1: reversed gravity
    r_end = oracle.force_residual(pos, acc, B)[0]
    assert r_end < 0.5 * r_start, (r_start, r_end)


# ---- Eq. 5 (L65-70), quasi-periodic boundary: only the leading (nearest) image of each pair --------------------------
def _box(rng, n, L):
    pos = rng.uniform(0, L, size=(3, n))
    mass = rng.uniform(0.5, 1.5, n) / n
    soft = np.full(n, 0.02 * L)
    return np.ascontiguousarray(pos), mass, soft


def test_quasi_periodic_two_body_across_the_boundary(oracle):
    """x_1 = 0.05 L, x_2 = 0.95 L: the leading image of the separation has length 0.1 L and points THROUGH the boundary,
    so particle 1 is pulled towards -x with m_2 / (0.1 L)^2 (Eq. 4 third case), not towards +x with m_2 / (0.9 L)^2."""
    L, m1, m2 = 2.0, 3.0, 5.0
    pos = np.array([[0.05 * L, 0.95 * L], [0.3, 0.3], [0.7, 0.7]])
    acc = oracle.forces_quasi_periodic(pos, np.array([m1, m2]), np.array([0.01, 0.01]), L)
    assert acc[0, 0] == pytest.approx(-m2 / (0.1 * L) ** 2, rel=1e-13)
    assert acc[0, 1] == pytest.approx(+m1 / (0.1 * L) ** 2, rel=1e-13)
    assert np.all(acc[1:] == 0.0)


def test_quasi_periodic_lattice_translation_newton3_and_open_limit(oracle):
    rng = np.random.default_rng(55)
    L = 1.7
    # odd simple-cubic lattice (no separation component of exactly L/2): every particle sits at a centre of symmetry
    g = (np.arange(5) + 0.5) * L / 5
    lat = np.ascontiguousarray(np.array(np.meshgrid(g, g, g, indexing="ij")).reshape(3, -1))
    acc = oracle.forces_quasi_periodic(lat, np.full(125, 1 / 125), np.full(125, 0.01), L)
    assert np.abs(acc).max() < 1e-13 * (1 / 125) / (L / 5) ** 2 * 125
    pos, mass, soft = _box(rng, 300, L)
    ref = oracle.forces_quasi_periodic(pos, mass, soft, L)
    # translation by any vector, positions wrapped back into the box: same forces (this is what the wrap is for)
    shift = np.array([[0.61 * L], [-2.3 * L], [0.123]])
    moved = np.ascontiguousarray(np.mod(pos + shift, L))
    err = np.linalg.norm(oracle.forces_quasi_periodic(moved, mass, soft, L) - ref, axis=0) / np.linalg.norm(ref, axis=0)
    assert err.max() < 1e-11
    # Newton's third law survives the wrap (the leading image of x_i - x_j is minus that of x_j - x_i)
    assert np.linalg.norm((mass * ref).sum(axis=1)) < 1e-14 * np.sum(mass * np.linalg.norm(ref, axis=0))
    # all particles within a region smaller than L/2: no wrap is active, result = the open-boundary oracle
    small = np.ascontiguousarray(0.3 * L + pos * 0.45)
    assert np.array_equal(oracle.forces_quasi_periodic(small, mass, soft, L), oracle.forces(small, mass, soft))
    # brute force with numpy longdouble on a few particles
    p8, m8, h8 = pos[:, :8].astype(np.longdouble), mass[:8], soft[:8]
    want = np.zeros((3, 8), dtype=np.longdouble)
    for i in range(8):
        for j in range(8):
            if i != j:
                d = p8[:, j] - p8[:, i]
                d = d - L * np.rint(d / L)
                r = np.sqrt(np.sum(d * d))
                want[:, i] += m8[j] * oracle.spline_F(float(r), h8[i] + h8[j]) * d / r
    got = oracle.forces_quasi_periodic(np.ascontiguousarray(pos[:, :8]), m8, h8, L)
    assert np.abs(got - want.astype(np.float64)).max() < 1e-13 * np.abs(got).max()


# ---- Eq. 5 (L65-70) with the cut |x - nL| < 2.6 L: periodic image sum ------------------------------------------------
def test_periodic_images_count_and_two_body_sum(oracle):
    """One source at the origin, one test particle at x: the force is the sum over the images inside the 2.6 L sphere
    around x, typed out here with numpy; at x -> 0+ there are 81 such triplets minus the coincident one."""
    L = 1.0
    n = np.array([(a, b, c) for a in range(-4, 5) for b in range(-4, 5) for c in range(-4, 5)], dtype=float)
    assert int(np.sum(np.sum(n * n, axis=1) < 2.6 ** 2)) == 81
    xt = np.array([0.21, -0.13, 0.34])
    v = xt[None, :] - n * L                                     # x_i - x_j - nL with x_j = 0
    r = np.linalg.norm(v, axis=1)
    keep = r < 2.6 * L
    want = -(2.0 * v[keep] / r[keep, None] ** 3).sum(axis=0)    # m_j = 2, calF = 1/r^2 beyond the softening
    pos = np.ascontiguousarray(np.array([xt, [0.0, 0.0, 0.0]]).T)
    acc = oracle.forces_periodic_images(pos, np.array([1.0, 2.0]), np.array([0.01, 0.01]), L)
    assert np.allclose(acc[:, 0], want, rtol=1e-13, atol=1e-15)


def test_periodic_images_symmetries(oracle):
    rng = np.random.default_rng(66)
    L = 1.3
    g = (np.arange(3) + 0.5) * L / 3
    lat = np.ascontiguousarray(np.array(np.meshgrid(g, g, g, indexing="ij")).reshape(3, -1))
    acc = oracle.forces_periodic_images(lat, np.full(27, 1 / 27), np.full(27, 0.01), L)
    assert np.abs(acc).max() < 1e-12                            # every lattice site is a centre of symmetry
    pos, mass, soft = _box(rng, 60, L)
    ref = oracle.forces_periodic_images(pos, mass, soft, L)
    # the image set of a separation does not depend on its representative: shifting particles by lattice vectors or
    # translating the whole set (without wrapping) leaves the forces unchanged
    moved = pos.copy(); moved[:, ::3] += np.array([[2 * L], [-L], [3 * L]])
    assert np.abs(oracle.forces_periodic_images(np.ascontiguousarray(moved), mass, soft, L) - ref).max() < 1e-11 * np.abs(ref).max()
    shifted = np.ascontiguousarray(pos + np.array([[0.37], [-1.9], [0.05]]))
    assert np.abs(oracle.forces_periodic_images(shifted, mass, soft, L) - ref).max() < 1e-11 * np.abs(ref).max()
    # Newton III
    assert np.linalg.norm((mass * ref).sum(axis=1)) < 1e-13 * np.sum(mass * np.linalg.norm(ref, axis=0))
    # the nearest image is one of the terms: removing the cut's other images gives back the quasi-periodic force
    qp = oracle.forces_quasi_periodic(pos, mass, soft, L)
    assert np.abs(ref - qp).max() > 1e-3 * np.abs(qp).max()     # the other images do contribute
