"""Seeded synthetic particle sets shaped like the paper's compactified runs.

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench, and
therefore holds none of the method's arithmetic (no pair law, no force sum, no
integrator, no Friedmann equation): it only draws inputs.  Everything is numpy fp64
on the host, `numpy.random.Generator(PCG64(seed))`, seed = SEED_BASE + config index.

Recipe (stated again in DESIGN.md §"Input recipe"; shapes follow PAPER.md §3.1):

* points uniform on S^3 (radius R) are mapped to R^3 by the stereographic
  projection of PAPER.md Eq. 15 (L208-213) with D_s = 2R, i.e. r = 2R tan(chi/2);
  draws with r > r_cut = 20R are rejected;
* masses follow the real-space volume per unit S^3 volume, the continuum limit of
  PAPER.md Eq. 16 (L219):  w = (1 + r^2/(4R^2))^3,  m = w / sum(w)   (Eq. 25);
* softening follows PAPER.md Eq. 7 (L82):  h_i = eps0 * (m_i/m_min)^(1/3);
* each position gets a Gaussian jitter of `jitter` times the local mean spacing
  s_i = (m_i V)^(1/3), V = (4 pi/3) r_cut^3;
* the set is finally sorted by |x| ascending (the radial order the force kernel's
  far/near tile classification profits from; correctness never depends on it).

Arrays are returned in the library's layout: `pos` is SoA, shape (3, N), C-contiguous
(`[x_0..x_{N-1} | y_0.. | z_0..]`), `mass` and `soft` have shape (N,).
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

SEED_BASE = 181105903  # + config index (BASELINE.json `configs`)


@dataclass
class ParticleSet:
    pos: np.ndarray      # (3, N) float64, SoA
    vel: np.ndarray      # (3, N) float64, SoA (zeros unless a config sets them)
    mass: np.ndarray     # (N,)   float64, sum = 1
    soft: np.ndarray     # (N,)   float64, the paper's h_i (Eq. 7)
    spacing: np.ndarray  # (N,)   float64, local mean interparticle spacing s_i
    volume: float        # V = (4 pi/3) r_cut^3
    r_cut: float

    @property
    def n(self) -> int:
        return int(self.mass.shape[0])


def _s3_stereographic(rng: np.random.Generator, n: int, R: float, r_lo: float, r_hi: float) -> np.ndarray:
    """n points: uniform on S^3, projected to R^3, kept when r_lo < r <= r_hi.  Returns (n, 3)."""
    out = np.empty((0, 3))
    while out.shape[0] < n:
        need = n - out.shape[0]
        u = rng.standard_normal((int(need * 1.25) + 64, 4))
        u /= np.linalg.norm(u, axis=1, keepdims=True)
        denom = 1.0 + u[:, 3]
        ok = denom > 1e-12
        x = 2.0 * R * u[ok, :3] / denom[ok, None]
        r = np.linalg.norm(x, axis=1)
        keep = (r > r_lo) & (r <= r_hi)
        out = np.concatenate([out, x[keep]], axis=0)
    return out[:n]


def _uniform_ball(rng: np.random.Generator, n: int, radius: float) -> np.ndarray:
    d = rng.standard_normal((n, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    rr = radius * rng.random(n) ** (1.0 / 3.0)
    return d * rr[:, None]


def _finish(rng, x, w, eps0, jitter, r_cut, sort) -> ParticleSet:
    n = x.shape[0]
    mass = w / np.sum(w)
    soft = eps0 * np.cbrt(mass / mass.min())
    volume = 4.0 * math.pi / 3.0 * r_cut ** 3
    spacing = np.cbrt(mass * volume)
    x = x + jitter * spacing[:, None] * rng.standard_normal((n, 3))
    if sort:
        order = np.argsort(np.linalg.norm(x, axis=1), kind="stable")
        x, mass, soft, spacing = x[order], mass[order], soft[order], spacing[order]
    pos = np.ascontiguousarray(x.T)
    return ParticleSet(pos=pos, vel=np.zeros_like(pos), mass=np.ascontiguousarray(mass),
                       soft=np.ascontiguousarray(soft), spacing=np.ascontiguousarray(spacing),
                       volume=volume, r_cut=r_cut)


def g0(n: int, seed: int, R: float = 1.0, r_cut_over_R: float = 20.0, eps0: float = 0.01,
       jitter: float = 0.01, sort: bool = True) -> ParticleSet:
    """Compactified set of configs 0, 1, 3 (and the unperturbed set of config 4)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    r_cut = r_cut_over_R * R
    x = _s3_stereographic(rng, n, R, -1.0, r_cut)
    r2 = np.sum(x * x, axis=1)
    w = (1.0 + r2 / (4.0 * R * R)) ** 3
    return _finish(rng, x, w, eps0, jitter, r_cut, sort)


def g2(n: int, seed: int, R: float = 1.0, r_cut_over_R: float = 20.0, core_frac_radius: float = 0.1,
       eps0: float = 0.01, jitter: float = 0.01, sort: bool = True) -> ParticleSet:
    """Config 2: the inner 10 % of the radius holds 50 % of the particles at uniform (minimum)
    mass, like the equal-mass core of the paper's constant-Delta-omega scheme (Eq. 17);
    the outer half follows g0's law.  Softening ratio across the set ~ 101."""
    rng = np.random.Generator(np.random.PCG64(seed))
    r_cut = r_cut_over_R * R
    r_core = core_frac_radius * r_cut
    n_core = n // 2
    xc = _uniform_ball(rng, n_core, r_core)
    xo = _s3_stereographic(rng, n - n_core, R, r_core, r_cut)
    wo = (1.0 + np.sum(xo * xo, axis=1) / (4.0 * R * R)) ** 3
    x = np.concatenate([xc, xo], axis=0)
    w = np.concatenate([np.ones(n_core), wo])
    return _finish(rng, x, w, eps0, jitter, r_cut, sort)


def config4_ics(n: int, seed: int, vel_factor: float, amp: float = 0.005) -> ParticleSet:
    """Config 4 initial conditions: g0(n), then a
    Zel'dovich-like displacement (Eq. 23-24) with i.i.d. Gaussian
    Psi_i = amp * s_i * N(0, I_3):  x = q + Psi,  v = vel_factor * Psi  (the caller supplies
    vel_factor = H(a_init) * dlnD/dlna(a_init) in code units; this module does no cosmology),
    the mass-weighted centre of mass and the net momentum removed."""
    ps = g0(n, seed)
    rng = np.random.Generator(np.random.PCG64(seed + 7919))
    m = ps.mass
    psi = amp * ps.spacing[None, :] * rng.standard_normal((3, n))
    pos = ps.pos + psi
    # zero centre of mass AFTER the displacement: the background term B x of Eq. 8 is a force
    # field centred on the origin, so total momentum is conserved only for x_com = 0
    pos = pos - (pos @ m)[:, None] / m.sum()
    vel = vel_factor * psi
    vel = vel - (vel @ m)[:, None] / m.sum()
    return ParticleSet(pos=np.ascontiguousarray(pos), vel=np.ascontiguousarray(vel), mass=m,
                       soft=ps.soft, spacing=ps.spacing, volume=ps.volume, r_cut=ps.r_cut)


def morton_order(pos: np.ndarray, L: float, bits: int = 7) -> np.ndarray:
    """Permutation that sorts the particles of a periodic box of side L along the Morton (Z-order) curve of a
    2^bits-per-side grid: consecutive particles then fill compact cells, the order the periodic-box kernels profit from
    (the counterpart of the radial order of the compactified sets; correctness never depends on it)."""
    g = np.floor(np.mod(pos, L) / L * (1 << bits)).astype(np.int64).clip(0, (1 << bits) - 1)
    code = np.zeros(pos.shape[1], dtype=np.int64)
    for b in range(bits):
        for c in range(3):
            code |= ((g[c] >> b) & 1) << (3 * b + c)
    return np.argsort(code, kind="stable")


def periodic_box(n: int, L: float, seed: int, cell_ordered: bool = True):
    """Uniform random particles of equal mass in a periodic cube of side L, softening 1/30 of the mean spacing (the
    state glass making starts from, section 3.1); Morton-ordered unless cell_ordered is False.
    Returns (pos (3, n), mass (n,), soft (n,))."""
    rng = np.random.default_rng(seed)
    pos = np.ascontiguousarray(rng.uniform(0.0, L, size=(3, n)))
    if cell_ordered:
        pos = np.ascontiguousarray(pos[:, morton_order(pos, L)])
    return pos, np.full(n, 1.0 / n), np.full(n, L / n ** (1 / 3) / 30)


def stratified_sample(n: int, n_sample: int, n_edge: int | None = None) -> np.ndarray:
    """Indices for sampled parity at large N: the innermost and outermost `n_edge` particles
    plus the rest uniform in index.  Sorted, unique, int64."""
    n_sample = min(n_sample, n)
    if n_edge is None:
        n_edge = max(1, n_sample // 16)
    n_edge = min(n_edge, n // 2)
    mid = np.linspace(n_edge, n - n_edge - 1, max(n_sample - 2 * n_edge, 0)).astype(np.int64)
    idx = np.concatenate([np.arange(n_edge), mid, np.arange(n - n_edge, n)])
    return np.unique(idx).astype(np.int64)


def config(index: int, n: int | None = None) -> ParticleSet:
    """The force-evaluation particle sets of BASELINE.json configs 0-3 (config 4: config4_ics)."""
    sizes = {0: 4096, 1: 65536, 2: 262144, 3: 1048576}
    if index not in sizes:
        raise ValueError("config index must be 0..3 (use config4_ics for config 4)")
    n = sizes[index] if n is None else n
    seed = SEED_BASE + index
    return g2(n, seed) if index == 2 else g0(n, seed)
