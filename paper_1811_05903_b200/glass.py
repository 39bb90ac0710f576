"""Glass generation (section 3.1): "integrating Eq. 8 with reversed gravity" in an Einstein-de Sitter
background until the net force on every particle is as small as it gets -- the paper notes it costs as much as a
simulation, so it is the long, purely N^2-bound run of the hot path.  Everything runs through the C ABI: device-resident
adaptive steps (Eq. 12; steps_kdk_step_adaptive, no host round trip between steps), the residual monitor
steps_force_residual every `report` steps, and a re-sort into radial order (steps_sort_radial) every `resort` steps.

    python -m paper_1811_05903_b200.glass --n 262144 --steps 400 [--mixed] [--report 50] [--resort 100]

Start: the compactified set g0(N) (seeded; Poisson-sampled in compact space, the state the paper's glass making starts from),
zero velocities.  Prints one JSON line per report and a final summary with the sustained interactions/s of the run."""
from __future__ import annotations

import argparse
import json
import time


def run(n: int, steps: int, mixed: bool = False, report: int = 50, resort: int = 100, seed: int = 181105903 + 5,
        eps: float = 0.025, a0: float = 0.05, log=print) -> dict:
    import torch

    from . import steps as S
    from . import synth

    ps = synth.g0(n, seed)
    pos, vel = torch.from_numpy(ps.pos).cuda(), torch.zeros((3, n), dtype=torch.float64, device="cuda")
    mass, soft = torch.from_numpy(ps.mass).cuda(), torch.from_numpy(ps.soft).cuda()
    acc = torch.empty_like(pos)
    B = 1.0 / ps.r_cut ** 3                                   # (4 pi / 3) rho_bar in G = 1, sum m = 1 units (reading #7)
    H0 = (2.0 * B) ** 0.5                                     # Einstein-de Sitter: Omega_m = 1
    cosmo = S.Cosmology(H0=H0, Omega_m=1.0, Omega_r=0.0, Omega_L=0.0, Omega_k=0.0)
    G = -1.0                                                  # reversed gravity
    state = torch.tensor([a0, 0.0, 1.0, 0.0, 0.0], dtype=torch.float64, device="cuda")
    out2 = torch.empty(2, dtype=torch.float64, device="cuda")
    perm = torch.empty(n, dtype=torch.int64, device="cuda")
    scratch3, scratch1 = torch.empty_like(pos), torch.empty_like(mass)
    S.steps_reserve(n)
    force = S.steps_forces_mixed if mixed else S.steps_forces
    force(pos, mass, soft, acc)
    dt_max = 0.05 / H0

    def residual():
        S.steps_force_residual(pos, acc, B, out2)
        s2, mx = out2.tolist()
        return (s2 / n) ** 0.5, mx

    rms0, max0 = residual()
    log(json.dumps({"step": 0, "a": a0, "rms_net_force": rms0, "max_net_force": max0}))
    torch.cuda.synchronize()
    t0, history = time.perf_counter(), []
    for k in range(1, steps + 1):
        S.steps_kdk_step_adaptive(pos, vel, acc, mass, soft, state, cosmo, G, B, eps, dt_max, mixed=mixed)
        if resort and k % resort == 0 and k < steps:
            # re-sort into radial order: the pending closing kick is applied first so that (pos, vel) are a consistent state
            S.steps_kick_close_adaptive(pos, vel, acc, state, B)
            S.steps_sort_radial(pos, perm)
            for arr, tmp in ((pos, scratch3), (vel, scratch3), (acc, scratch3), (mass, scratch1), (soft, scratch1)):
                S.steps_permute(arr, perm, tmp)
                arr.copy_(tmp)
        if k % report == 0 or k == steps:
            rms, mx = residual()
            history.append((k, rms))
            log(json.dumps({"step": k, "a": state[0].item(), "dt": state[1].item(), "rms_net_force": rms, "max_net_force": mx}))
    S.steps_kick_close_adaptive(pos, vel, acc, state, B)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    rms1, max1 = residual()
    summary = {"n": n, "steps": steps, "path": "mixed" if mixed else "fp64", "wall_s": wall,
               "interactions_per_s": steps * n * (n - 1.0) / wall, "rms_net_force_start": rms0, "rms_net_force_end": rms1,
               "max_net_force_start": max0, "max_net_force_end": max1, "a_end": state[0].item()}
    log(json.dumps(summary))
    return summary


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=262144)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--mixed", action="store_true")
    ap.add_argument("--report", type=int, default=50)
    ap.add_argument("--resort", type=int, default=100)
    a = ap.parse_args()
    run(a.n, a.steps, mixed=a.mixed, report=a.report, resort=a.resort)
