"""Writes tests/golden/config4_chaos_floor.txt: how fast config 4 (N = 8,192, 200 comoving KDK steps, a: 1/51 -> 1)
forgets a rounding-size perturbation.  Calls ONLY the CPU oracle (oracle/) and the seeded input generator.

The run is repeated from initial positions perturbed by +-1 ulp (three realisations); the table lists, every 10 steps,
max_i |x_i(perturbed) - x_i| / s_i (s_i = local mean spacing), the largest of the three.  This is the floor below which
no two fp64 implementations of the same step can be expected to agree (SURVEY.md 8(c.5) "chaos floor"); DESIGN.md
section 2 quotes the table and tests/test_parity_gpu.py::test_config4_free_running_vs_oracle_8192 re-measures the part it
uses.

Usage: python tests/golden/make_config4_chaos_floor.py      (about a minute on 8 cores)"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import steps_oracle as oracle  # noqa: E402
from paper_1811_05903_b200 import synth  # noqa: E402

LCDM = dict(H0=0.0288675134594813, Omega_m=0.3, Omega_r=0.0, Omega_L=0.7, Omega_k=0.0)
N, STEPS, EVERY, REALISATIONS = 8192, 200, 10, 3


def main():
    vf = oracle.hubble(1 / 51, LCDM) * oracle.growth_rate(1 / 51, LCDM)
    ps = synth.config4_ics(N, synth.SEED_BASE + 4, vel_factor=vf)
    B = 1.0 / ps.r_cut ** 3
    dts = oracle.ln_a_schedule(1 / 51, 1.0, STEPS, LCDM)

    def run(pos0):
        pos, vel = pos0.copy(), ps.vel.copy()
        acc = oracle.forces(pos, ps.mass, ps.soft)
        a, snaps = 1 / 51, []
        for k, dt in enumerate(dts):
            a = oracle.kdk_step(pos, vel, acc, ps.mass, ps.soft, a, float(dt), 1.0, B, LCDM)
            if (k + 1) % EVERY == 0:
                snaps.append(pos.copy())
        return snaps

    base = run(ps.pos)
    floor = np.zeros(len(base))
    for r in range(REALISATIONS):
        sign = np.random.default_rng(r).choice([-1.0, 1.0], size=ps.pos.shape)
        pert = run(ps.pos * (1.0 + 1.1e-16 * sign))
        floor = np.maximum(floor, [np.max(np.linalg.norm(p - b, axis=0) / ps.spacing) for p, b in zip(pert, base)])
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config4_chaos_floor.txt")
    with open(out, "w") as f:
        f.write("# config 4, N = 8192, seed 181105907: max_i |dx_i| / s_i between the oracle run and the oracle run started from\n"
                "# positions perturbed by +-1 ulp (largest of 3 realisations).  Written by make_config4_chaos_floor.py (oracle only).\n"
                "# step  a  max|dx|/s\n")
        for j, v in enumerate(floor):
            k = (j + 1) * EVERY
            f.write(f"{k:4d}  {(1 / 51) * 51 ** (k / STEPS):.5f}  {v:.3e}\n")
    print(open(out).read())


if __name__ == "__main__":
    main()
