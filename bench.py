#!/usr/bin/env python
"""bench.py -- BASELINE.json's metric: ordered pairwise interactions/s per force evaluation at
N = 1,048,576 (config 3), and the fraction of the FP32 (mixed path) / FP64 (fp64 path) peak.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl native|reference] [--n N_PARTICLES]

A "step" is one pass of the whole hot path through the C ABI: steps_kdk_step (fused kick/drift,
tile prep, the O(N^2) force kernel, the split-j reduce) plus the momentum diagnostic -- rows
a0-a7 of SURVEY.md 8(a); a6 is a handful of host doubles.  Both paths are timed; `value` is the
mixed path (the FP32 target), `paths.fp64` carries the fp64 path.  One JSON line on stdout.

  * inputs resident in HBM for `value`; `e2e` goes through steps_forces_host with pinned HOST
    buffers (H2D of pos/mass/soft and D2H of acc inside the timed region);
  * every step is bracketed by CUDA events on the launch stream, L2 is flushed (256 MiB write)
    between timed steps, >= 3 warm-up steps; the force kernel alone is bracketed by the library
    ("profile" option) for the roofline figure;
  * clocks / throttle reasons are sampled through NVML during the timed region;
  * `cpu_baseline` / `--impl reference`: the CPU oracle as it stands, on a bounded i-sample.
  * N > 1 GPUs (torchrun): the paper's decomposition (L135-139) with the i-blocks dealt round-robin
    (shard.py) -- each rank evaluates the forces of its blocks against all sources
    (steps_forces_blocks), kicks/drifts its particles, and the drifted positions are all-gathered
    (NCCL): total work fixed => "strong" scaling.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

FLOP_PER_INTERACTION = 20.0      # stated convention
SM_COUNT, SM_MAX_MHZ, SM_MHZ_SOURCE = 148, 1965.0, "profiling guide (1965 MHz)"
try:                                   # driver-written per pod; absent -> the guide's B200 boost clock
    with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as _f:
        _mhz = float(json.load(_f).get("sm_max_mhz", 0.0))
    if 1000.0 < _mhz < 3000.0:
        SM_MAX_MHZ, SM_MHZ_SOURCE = _mhz, "MEASURED_PEAKS.json sm_max_mhz"
except (OSError, ValueError):
    pass
PEAK_FP32_TFLOPS = SM_COUNT * 128 * 2 * SM_MAX_MHZ * 1e6 / 1e12     # 74.45
PEAK_FP64_TFLOPS = SM_COUNT * 64 * 2 * SM_MAX_MHZ * 1e6 / 1e12      # 37.22 (64 FP64 lanes/SM, measured)
METRIC = "pairwise interactions/s per force eval at N=1M"
UNIT = "interactions/s"
LCDM = dict(H0=0.0288675134594813, Omega_m=0.3, Omega_r=0.0, Omega_L=0.7, Omega_k=0.0)


def ncu_traffic(path: str, n: int):
    """DRAM bytes per force evaluation (dram__bytes_read.sum + dram__bytes_write.sum of its force kernels) from the newest
    committed `ncu --set full` capture, profiles/r*_dram_traffic.csv: rows `path,N,kernel,read_bytes,write_bytes`.  The
    figure is a record of that capture, not measured in this run: returned only for the captured (path, N), else None."""
    import csv
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_dram_traffic.csv")))
    if not files:
        return None, "no ncu capture committed"
    total, kernels = 0.0, []
    with open(files[-1]) as f:
        for row in csv.DictReader(f):
            if row["path"] == path and int(row["N"]) == n:
                total += float(row["read_bytes"]) + float(row["write_bytes"])
                kernels.append(row["kernel"])
    if not kernels:
        return None, f"{os.path.basename(files[-1])} has no capture of path={path} N={n}"
    return total, f"{os.path.basename(files[-1])}: " + " + ".join(kernels)


class ClockSampler:
    """NVML sampler thread: SM clock and throttle reasons while the timed region runs."""

    def __init__(self, index: int, period: float = 0.1):
        self.samples, self.reasons, self.period, self._stop = [], set(), period, threading.Event()
        self.max_mhz, self.ok = None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            pass
        self.t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.ok:
            self.t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self.ok:
            self.t.join(timeout=2)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def cpu_oracle_rate(ps, budget_s: float = 12.0):
    """The oracle as it stands on this host's cores, on a bounded stratified i-sample x all j."""
    from oracle import steps_oracle as oracle
    from paper_1811_05903_b200 import synth
    n = ps.n
    probe = synth.stratified_sample(n, max(64, min(n, 4 * oracle.num_threads() * 16)))
    t0 = time.perf_counter()
    oracle.forces(ps.pos, ps.mass, ps.soft, idx=probe)
    dt = time.perf_counter() - t0
    rate = len(probe) * (n - 1.0) / dt
    n_idx = int(min(n, max(len(probe), budget_s * rate / (n - 1.0))))
    idx = synth.stratified_sample(n, n_idx)
    t0 = time.perf_counter()
    oracle.forces(ps.pos, ps.mass, ps.soft, idx=idx)
    dt = time.perf_counter() - t0
    return {"value": len(idx) * (n - 1.0) / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{len(idx)} stratified i-particles x all {n} sources of the same workload, {dt:.1f} s"}


def bench_next_rows(S, synth, torch, stream, reps: int = 3):
    """SURVEY.md 8(f) rows, each timed on its own workload (3 warm-up + `reps` timed calls, CUDA events on the launch
    stream, L2 not flushed: these kernels are ALU-bound and their inputs fit L2 anyway).  Periodic boxes: uniform random
    particles of equal mass in a cube of side 1, softening 1/30 of the mean spacing (the state glass making starts from,
    as in the parity tests), in Morton (cell) order -- the periodic counterpart of the radial order.  The roofline fraction uses the same 20 flop per evaluated pair term as the headline."""
    import numpy as np

    def timed(fn):
        for _ in range(3):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        e1.synchronize()
        return e0.elapsed_time(e1) / reps

    def box(n, seed):
        pos, mass, soft = (torch.from_numpy(a).cuda() for a in synth.periodic_box(n, 1.0, seed))
        return pos, mass, soft, torch.empty_like(pos)

    rows = {}
    for n, tag in ((262144, ""), (1048576, "_1M")):
        pos, mass, soft, acc = box(n, 9001)
        for mixed in (False, True):
            ms = timed(lambda: S.steps_forces_quasi_periodic(pos, mass, soft, 1.0, acc, mixed=mixed))
            rate = n * (n - 1.0) / (ms * 1e-3)
            peak = PEAK_FP32_TFLOPS if mixed else PEAK_FP64_TFLOPS
            rows["quasi_periodic_" + ("mixed" if mixed else "fp64") + tag] = {
                "value": rate, "unit": UNIT, "ms": ms, "N": n, "workload": "uniform periodic box in Morton order, leading image (Eq. 5)",
                "roofline": {"bound": "alu", "achieved": FLOP_PER_INTERACTION * rate / 1e12, "peak": peak, "unit": "TFLOP/s",
                             "frac": FLOP_PER_INTERACTION * rate / 1e12 / peak}}
        del pos, mass, soft, acc
    images = 4.0 / 3.0 * math.pi * 2.6 ** 3                        # mean number of images inside the 2.6 L cut per pair
    for n, tag in ((32768, ""), (131072, "_131072")):
        pos, mass, soft, acc = box(n, 9002)
        ms = timed(lambda: S.steps_forces_periodic(pos, mass, soft, 1.0, acc))
        rate = n * (n - 1.0) / (ms * 1e-3)
        rows["periodic_images" + tag] = {
            "value": rate, "unit": "pairs/s (each summed over its images inside |x - nL| < 2.6 L)", "ms": ms, "N": n,
            "images_per_pair_in_cut": images, "image_terms_per_s": rate * images,
            "roofline": {"bound": "alu", "achieved": FLOP_PER_INTERACTION * rate * images / 1e12, "peak": PEAK_FP64_TFLOPS,
                         "unit": "TFLOP/s", "frac": FLOP_PER_INTERACTION * rate * images / 1e12 / PEAK_FP64_TFLOPS}}
    # device-resident adaptive step (Eq. 12 + KDK + force evaluation), config 0 size and 32,768
    for n in (4096, 32768):
        ps = synth.g0(n, synth.SEED_BASE)
        x, m, h = (torch.from_numpy(a).cuda() for a in (ps.pos, ps.mass, ps.soft))
        v, a = torch.zeros_like(x), torch.empty_like(x)
        S.steps_forces(x, m, h, a)
        st = torch.tensor([1.0 / 51.0, 0.0, 1.0, 0.0, 0.0], dtype=torch.float64, device="cuda")
        cosmo = S.Cosmology(**LCDM)
        ms = timed(lambda: S.steps_kdk_step_adaptive(x, v, a, m, h, st, cosmo, 1.0, 1.25e-4, 0.025, 0.05))
        rows[f"adaptive_step_{n}"] = {"value": n * (n - 1.0) / (ms * 1e-3), "unit": UNIT, "us_per_step": 1e3 * ms, "N": n,
                                       "workload": "steps_kdk_step_adaptive, fp64, compactified g0 set"}
    return rows


def run_reference(args):
    """--impl reference: the CPU oracle (fp64 pairwise spline sum), each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import steps_oracle as oracle
    from paper_1811_05903_b200 import synth
    n = args.n or 1048576
    ps = synth.g0(n, synth.SEED_BASE + 3)
    per_step = max(64, min(n, int(args.ref_pairs / n)))
    idx = synth.stratified_sample(n, per_step)
    for _ in range(args.warmup):
        oracle.forces(ps.pos, ps.mass, ps.soft, idx=idx[: max(16, len(idx) // 8)])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.forces(ps.pos, ps.mass, ps.soft, idx=idx)
    dt = time.perf_counter() - t0
    value = args.steps * len(idx) * (n - 1.0) / dt
    sample = f"{len(idx)} stratified i-particles x all {n} sources per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config3: compactified g0 set, N={n}, CPU oracle on a bounded i-sample", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--n", type=int, default=0, help="override the particle count (default: config 3, 1,048,576)")
    ap.add_argument("--paths", default="mixed,fp64")
    ap.add_argument("--ref-pairs", type=float, default=4e9, help="--impl reference: pair budget per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the periodic / adaptive-step rows (SURVEY 8(f))")
    ap.add_argument("--next-rows-only", action="store_true",
                    help="only the periodic / adaptive-step rows (one JSON line with `next_rows`; for profiling them)")
    ap.add_argument("--sharded-step", action="store_true",
                    help="time the N > 1 step (shard.WorkSharedStep / shard.ShardedStep: share of the work + exchange) even with one rank")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_1811_05903_b200 import shard, synth
    from paper_1811_05903_b200 import steps as S

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    if world > 1:
        # NCCL's communicator/topology log (NVLS, rings, ranks) to stderr: stdout carries the one JSON line
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT,ENV")
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    args.warmup = max(args.warmup, 3)

    if args.next_rows_only:
        S.steps_set_option("profile", 0)
        print(json.dumps({"next_rows": bench_next_rows(S, synth, torch, torch.cuda.current_stream(), reps=args.steps), "build": S.build_info()}))
        return

    n = args.n or 1048576
    ps = synth.g0(n, synth.SEED_BASE + 3)          # config 3 (identical on every rank: seeded)
    cnt = shard.owned_count(rank, world, n)        # N > 1: the rank's round-robin blocks (shard.py)
    pos = torch.from_numpy(ps.pos).cuda()           # replicated sources
    mass, soft = torch.from_numpy(ps.mass).cuda(), torch.from_numpy(ps.soft).cuda()
    S.steps_reserve(n)
    S.steps_set_option("profile", 1)
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    mom = torch.empty(4, dtype=torch.float64, device="cuda")
    cosmo = S.Cosmology(**LCDM)
    B = 1.0 / ps.r_cut ** 3
    sched = S.steps_kdk_schedule(1.0 / 51.0, 1.0e-3, 1.0, cosmo)
    stream = torch.cuda.current_stream()
    inter_step = float(n) * (n - 1.0)               # ordered pairs of one whole-job force evaluation
    paths = [p for p in args.paths.split(",") if p in ("mixed", "fp64")]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    results, launches_total, plans = {}, 0, {}
    sampler = ClockSampler(local_rank)
    with sampler:
        for path in paths:
            mixed = path == "mixed"
            x = pos.clone()
            co = S.KdkCoeffs(1.0, 0.0, sched["alpha_open"], sched["beta_open"], sched["gamma"], B, int(mixed))
            if world == 1 and not args.sharded_step:
                v, acc = torch.zeros_like(x), torch.empty_like(x)
                (S.steps_forces_mixed if mixed else S.steps_forces)(x, mass, soft, acc)

                def step():
                    S.steps_kdk_step(x, v, acc, mass, soft, co)
                    S.steps_momentum(v, mass, mom)
            elif S.steps_pair_symmetric(n, mixed):
                # N > 1: the force evaluation shared by WORK (steps_forces_share: each rank an equal part of the band visits
                # and of the pair-symmetric items, at the single-GPU kernels' rate), one all-reduce of the partial
                # accelerations per step, every rank advances all particles
                sh = shard.WorkSharedStep(S, rank, world, x, torch.zeros_like(x), mass, soft, mixed)
                sh.forces()

                def step():
                    sh.step(co)
                    S.steps_momentum(sh.v, sh.m, mom)
            else:
                sh = shard.ShardedStep(S, rank, world, x, torch.zeros_like(x), mass, soft, mixed)
                sh.forces()

                def step():
                    sh.step(co)
                    if sh.cnt:
                        S.steps_momentum(sh.v, sh.m, mom)

            for _ in range(args.warmup):
                step()
            barrier()
            l0 = S.steps_kernel_launch_count()
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
            kernel_ms = []
            for k in range(args.steps):
                flush_buf.fill_(k & 0xFF)                       # L2 flush between timed steps (outside the events)
                ev[k][0].record(stream)
                step()
                ev[k][1].record(stream)
                ev[k][1].synchronize()
                kernel_ms.append(S.steps_last_force_kernel_ms())
            barrier()
            launches = S.steps_kernel_launch_count() - l0
            t_ms = torch.tensor([sum(a.elapsed_time(c) for a, c in ev)], dtype=torch.float64, device="cuda")
            if world > 1:
                dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
            total_ms = float(t_ms.item())
            k_ms = sum(kernel_ms) / len(kernel_ms)
            peak = PEAK_FP32_TFLOPS if mixed else PEAK_FP64_TFLOPS
            sharded = world > 1 or args.sharded_step
            symmetric = bool(S.steps_pair_symmetric(n, mixed))
            # this rank's launches: its blocks against all sources (one-sided plan) or 1 / world of the pair evaluations
            kern_inter = inter_step / world if (sharded and symmetric) else float(cnt) * (n - 1.0)
            achieved = FLOP_PER_INTERACTION * kern_inter / (k_ms * 1e-3) / 1e12
            traffic, traffic_source = ncu_traffic(path, n) if not sharded else (None, "sharded step")
            plans[path] = ("none" if not sharded else
                           f"pair evaluations shared equally among {world} ranks (steps_forces_share), all-reduce of 3N partial accelerations" if symmetric
                           else f"i-blocks of 2048 dealt round-robin to {world} ranks (PAPER L135-139, SURVEY 8(e)), all-gather of positions")
            results[path] = {
                "value": args.steps * inter_step / (total_ms * 1e-3), "unit": UNIT,
                "ms_per_step": total_ms / args.steps, "force_kernel_ms": k_ms, "gpu_launches": int(launches),
                "dtype": "f32 pairs, f64 accumulate" if mixed else "f64",
                "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                             "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source,
                             "flop_per_interaction": FLOP_PER_INTERACTION,
                             "pair_evaluation": ("each far block pair once, applied to both blocks (Newton III, PAPER L131); "
                                                 "band around the diagonal one-sided") if symmetric else "one-sided (every ordered pair)",
                             "peak_source": "148 SM x %d lanes x 2 x %.0f MHz (%s; DESIGN.md section 6; lanes/SM measured)" % (128 if mixed else 64, SM_MAX_MHZ, SM_MHZ_SOURCE),
                             "kernel": (("forces_sym_mixed_kernel" if mixed else "forces_sym_kernel") +
                                        " + band forces_persistent_kernel + reduces (one event pair around all of them)") if symmetric
                                       else "forces_persistent_kernel<%s>" % ("MixedPath" if mixed else "Fp64Path"),
                             "kernel_share_of_step": k_ms * args.steps / total_ms},
            }
            launches_total += launches

        # end to end through the C ABI with HOST buffers (N = 1 process only: the call is single-GPU)
        e2e = None
        if world == 1 and "mixed" in paths:
            hp, hm, hh = (torch.from_numpy(a).pin_memory() for a in (ps.pos, ps.mass, ps.soft))
            ha = torch.empty((3, n), dtype=torch.float64).pin_memory()
            for _ in range(2):
                S.steps_forces_host(hp, hm, hh, ha, mixed=True)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = max(2, min(args.steps, 5))
            e0.record(stream)
            for _ in range(reps):
                S.steps_forces_host(hp, hm, hh, ha, mixed=True)
            e1.record(stream)
            e1.synchronize()
            e2e = {"value": reps * inter_step / (e0.elapsed_time(e1) * 1e-3), "unit": UNIT,
                   "h2d_bytes_per_step": 5 * n * 8, "d2h_bytes_per_step": 3 * n * 8,
                   "call": "steps_forces_host(mixed=1), pinned host buffers"}
        # the section 8(f) NEXT rows (one GPU; their own short repetition, not --steps)
        next_rows = bench_next_rows(S, synth, torch, stream) if world == 1 and not args.no_next_rows else None
    clocks = sampler.summary()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    head = "mixed" if "mixed" in results else paths[0]
    r = results[head]
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_oracle_rate(ps)
    if clocks.get("sm_mhz"):
        for p in results.values():
            p["roofline"]["frac_at_sampled_clock"] = p["roofline"]["frac"] * SM_MAX_MHZ / clocks["sm_mhz"]
    out = {
        "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
        "scaling": "strong", "vs_baseline": None, "dtype": r["dtype"], "data": "synthetic",
        "config": {"workload": f"config3: compactified g0 set (S^3 stereographic, m~(1+r^2/4R^2)^3, eps_i=0.01(m_i/m_min)^(1/3)), N={n}, "
                               f"one steps_kdk_step (kick+drift+prep+force+reduce) + momentum per step",
                   "headline_path": head, "l2": "256 MiB flush write between timed steps (inputs 42 MB fit L2; ALU-bound)",
                   "i_sharding": plans[head],
                   "persistent_grid": {p: S.steps_persistent_grid(p == "mixed") for p in results}},
        "roofline": r["roofline"], "paths": results, "clocks": clocks, "gpu_launches": int(launches_total),
        "e2e": e2e, "cpu_baseline": cpu, "next_rows": next_rows, "build": S.build_info(),
        "context": "paper (other hardware): 9.3 Tflop/s on 4x GTX 1080 Ti, ~24% of peak (L159); K80 ~9.7e9 interactions/s/GPU (Table 1, derived)",
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
