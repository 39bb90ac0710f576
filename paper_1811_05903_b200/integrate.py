"""Host-side driver of the KDK run (row a6: the O(1) scalar bookkeeping; all O(N) and O(N^2)
work is in the kernels).  Follows the driver pattern documented at steps_kdk_step in
include/steps.h: forces once, then one fused kick/drift + force evaluation per step, the
closing half kick of step n fused with the opening half kick of step n+1."""
from __future__ import annotations

from . import steps as S


def resort_radial(arrays3, arrays1, ids=None) -> None:
    """Re-order the particle state into radial order in place (row a0: steps_sort_radial + steps_permute).  arrays3: SoA
    (3, N) tensors, the FIRST of which is the positions; arrays1: (N,) tensors (mass, soft); ids: optional int64 tensor of
    particle labels that follows the permutation (so that the caller can find a particle again)."""
    import torch
    pos = arrays3[0]
    n = pos.shape[1]
    perm = torch.empty(n, dtype=torch.int64, device=pos.device)
    S.steps_sort_radial(pos, perm)
    tmp3, tmp1 = torch.empty_like(pos), torch.empty(n, dtype=torch.float64, device=pos.device)
    for a in arrays3:
        S.steps_permute(a, perm, tmp3)
        a.copy_(tmp3)
    for a in arrays1:
        S.steps_permute(a, perm, tmp1)
        a.copy_(tmp1)
    if ids is not None:
        ids.copy_(ids.index_select(0, perm))


def run_kdk(pos, vel, acc, mass, soft, a0: float, dts, cosmo: S.Cosmology, G: float, B: float,
            mixed: bool = False, on_step=None, resort_every: int = 0, ids=None) -> float:
    """Integrate in place over the time steps `dts` starting at scale factor a0.  `acc` must
    hold the forces at the initial positions on entry (steps_forces) and holds the forces at
    the final positions on return.  Returns the final scale factor.  on_step(k, a) is called
    after each step's force evaluation with velocities still lacking the closing half kick.
    resort_every > 0: every that many steps the state (pos, vel, acc, mass, soft and `ids`) is re-ordered radially
    (resort_radial) -- the order the force kernels are fast in decays as the structure grows; the
    pending closing kick is a pair of scalars and needs no attention."""
    a = a0
    alpha_c, beta_c = 1.0, 0.0                      # identity closing kick before the first step
    for k, dt in enumerate(dts):
        sc = S.steps_kdk_schedule(a, float(dt), G, cosmo)
        co = S.KdkCoeffs(alpha_c, beta_c, sc["alpha_open"], sc["beta_open"], sc["gamma"], B, int(mixed))
        S.steps_kdk_step(pos, vel, acc, mass, soft, co)
        alpha_c, beta_c, a = sc["alpha_close"], sc["beta_close"], sc["a_next"]
        if on_step is not None:
            on_step(k, a)
        if resort_every and (k + 1) % resort_every == 0 and k + 1 < len(dts):
            resort_radial([pos, vel, acc], [mass, soft], ids)
    S.steps_kick_drift(pos, vel, acc, S.KdkCoeffs(alpha_c, beta_c, 1.0, 0.0, 0.0, B, int(mixed)))
    return a


def run_adaptive(pos, vel, acc, mass, soft, a0: float, n_steps: int, cosmo: S.Cosmology, G: float, B: float,
                 eps: float, dt_max: float, mixed: bool = False, on_step=None):
    """n_steps KDK steps whose length is the global adaptive step of Eq. 12 (steps_timestep) evaluated on the forces
    at the start of each step.  G < 0 is the reversed gravity of glass generation.  `acc` holds the
    forces at the current positions on entry and on return.  Returns (final scale factor, list of step lengths).
    One device->host read of the step length per step (the next step's coefficients need it)."""
    import torch
    dt_dev = torch.empty(1, dtype=torch.float64, device=pos.device)
    a, dts = a0, []
    for k in range(n_steps):
        S.steps_timestep(pos, acc, soft, S.steps_timestep_coefficient(G, a), B, eps, dt_max, dt_dev)
        dt = float(dt_dev.item())
        a = run_kdk(pos, vel, acc, mass, soft, a, [dt], cosmo, G, B, mixed=mixed)
        dts.append(dt)
        if on_step is not None:
            on_step(k, a)
    return a, dts
