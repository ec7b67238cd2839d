#!/usr/bin/env python
"""bench.py — ray-substep-bin updates/s of the Ray-trax march (BASELINE.json metric) on N B200s.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl reference]

A "step" is one pass of the whole hot path: one rt_march call (zero-fill, ray-order, march, snapshot
prefix) over the full workload.  Default workload = BASELINE.json configs[2] ("C2": 128^3, 4,096 rays,
2,097 sources at the density peaks, 444 substeps), the configuration the metric is quoted on.
One JSON line is printed by rank 0; see DESIGN.md §8 for every field.  Besides the headline (C2) the default
single-GPU run also times, a few steps each, the other large configs (`per_config`: C3, C4, and C2 with its sources
jittered off the cell nodes -- the general-position cost of the headline) and the other entry points on C2
(`modes`: step, trilinear_kappa, adjoint_j, adjoint_kappa, jvp_kappa), each with its own roofline and a checksum
(--no-extras skips them).

N > 1 (under torchrun): weak scaling — rank r marches sources [r*n_src, (r+1)*n_src) of the N*n_src
highest-density cells, then one NCCL sum all-reduce of the field (sharding.py).

--impl reference times the fp64 CPU oracle (oracle/, as it stands) on this box's host cores on a bounded
sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "ray-substep-bin updates/s"
UNIT = "updates/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C2", choices=["C0", "C1", "C2", "C3", "C4"])
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--variant", type=int, default=0, help="RT_VARIANT_* (0 = the product path)")
    ap.add_argument("--mode", default="march", choices=["march", "step", "trilinear_kappa", "adjoint_j", "adjoint_kappa", "jvp_kappa"],
                    help="march: one rt_march call per bench step (the headline); step: the same workload as n_steps "
                         "rt_march_step calls with persistent ray state (DESIGN.md D17); trilinear_kappa: "
                         "rt_march_trilinear_kappa (DESIGN.md D18); adjoint_j: rt_march_adjoint_j, dL/dj for a "
                         "random dL/d out (DESIGN.md D19; `out` then holds nothing useful)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the per_config and modes objects")
    ap.add_argument("--extra-steps", type=int, default=5, help="timed steps of each per_config / modes entry")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target host time of the oracle sample")
    return ap.parse_args()


def make_workload(name, world_size=1):
    """Config `name`; for world_size > 1 the source list is extended to world_size * n_src sources by the
    config's own placement rule (weak scaling: per-GPU work fixed)."""
    import workloads
    w = workloads.make_config(name)
    if world_size > 1:
        n = w.n_src * world_size
        if name in ("C2", "C3"):
            rho = workloads.lognormal_density(128, 938902, 1.5)
            order = np.argsort(-rho.ravel(), kind="stable")[:n]
            w.sources = np.stack(np.unravel_index(order, rho.shape), axis=1).astype(np.float32)
        else:
            seed = {"C0": 939900, "C1": 939901, "C4": 939904}[name]
            hi = w.shape[0] - 1.0
            w.sources = np.random.default_rng(seed).uniform(0.0, hi, (n, 3)).astype(np.float32)
    return w


def describe(w, world_size):
    nx, ny, nz = w.shape
    return {"workload": f"{w.name}: {nx}x{ny}x{nz} fp32 grid x {w.n_bins} bin(s), {w.n_src} sources/GPU, "
                        f"N_Omega={w.n_rays}, ds={w.step_size}, {w.n_steps} step(s) x N_s={w.substeps_per_step}",
            "medium": w.meta.get("medium", ""), "baseline_config_index": int(w.name[1]),
            "ray_substeps_per_gpu": w.ray_substeps, "updates_per_gpu": w.updates,
            "parallelism": f"sources sharded over {world_size} GPU(s)" + (", 1 all-reduce" if world_size > 1 else "")}


# ----------------------------------------------------------------------------------------------------
# the oracle on host cores: cpu_baseline leg and --impl reference
# ----------------------------------------------------------------------------------------------------
def oracle_sample(w, seconds, repeats=1):
    """Time the oracle (as it stands) on a stratified subset of the sources sized for ~`seconds` of host
    time.  Returns (updates/s, cores, description, [seconds per repeat])."""
    import oracle
    cores = oracle.host_threads()
    per_src = w.n_rays * w.n_steps * w.substeps_per_step * w.n_bins
    probe_n = min(w.n_src, cores)
    idx = np.unique(np.linspace(0, w.n_src - 1, probe_n).round().astype(int))
    t0 = time.perf_counter()
    oracle.march(w.j, w.kappa, w.sources[idx], w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
    rate = len(idx) * per_src / (time.perf_counter() - t0)
    n = int(min(w.n_src, max(cores, seconds * rate / per_src)))
    idx = np.unique(np.linspace(0, w.n_src - 1, n).round().astype(int))
    src = np.ascontiguousarray(w.sources[idx])
    times = []
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.march(w.j, w.kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps)
        times.append(time.perf_counter() - t0)
    ups = len(idx) * per_src / min(times)
    what = (f"{len(idx)} of {w.n_src} sources of {w.name} (stratified), all {w.n_rays} rays x "
            f"{w.n_steps * w.substeps_per_step} substeps x {w.n_bins} bin(s); fp64 oracle, {cores} threads")
    return ups, cores, what, times, len(idx) * per_src


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = make_workload(args.config)
    steps = max(1, args.steps)
    for _ in range(min(args.warmup, 1)):
        oracle_sample(w, 1.0)
    budget = max(2.0, min(args.cpu_seconds, 120.0 / steps))
    ups, cores, what, times, units = oracle_sample(w, budget, repeats=steps)
    value = units * len(times) / sum(times)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": describe(w, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
            "note": "each step = the fp64 CPU oracle on the bounded sample described in cpu_baseline.sample"}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------------
# clocks during the timed region
# ----------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), [c.strip() for c in line.split(",")]))

    def wait_first(self, timeout=3.0):
        """Block until nvidia-smi has printed its first row: its start-up holds driver locks for a few hundred ms, which
        would land in a region timed by wall clock."""
        t_end = time.perf_counter() + timeout
        while self.proc and not self.rows and time.perf_counter() < t_end:
            time.sleep(0.01)

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except subprocess.TimeoutExpired:
                self.proc.kill()

    def summary(self, t0, t1):
        rows = [r for t, r in self.rows if t0 <= t <= t1 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_min_mhz": sm[0], "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "power_w_max": max(float(r[2]) for r in rows), "samples": len(rows)}


# ----------------------------------------------------------------------------------------------------
# the CUDA path
# ----------------------------------------------------------------------------------------------------
def measure_ceilings(rt, torch, shape, n_bins, only=None):
    """Reduction-throughput ceilings on a grid of the workload's size, in this process, back to back with
    the march: best of 5 launches of >= 2^28 reductions each, CUDA events.  Greds/s."""
    grid = torch.zeros(shape + (n_bins,), dtype=torch.float32, device="cuda")
    grid64 = None
    res = {}
    for name, mode in rt.binding.RED_MODES.items():
        if only is not None and name not in only:
            continue
        if mode in (6, 7) and grid64 is None:
            grid64 = torch.zeros(shape + (n_bins,), dtype=torch.float64, device="cuda")
        g = grid64 if mode in (6, 7) else grid
        if mode == 1 and grid.numel() % 4:
            continue
        n_red = (1 << 24) if mode in (3, 8) else (1 << 28)
        best = None
        for rep in range(6):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            issued = rt.rt_bench_red_ceiling(mode, g, n_red, seed=rep + 1)
            e1.record()
            e1.synchronize()
            ms = e0.elapsed_time(e1)
            if rep and (best is None or ms < best):
                best = ms
        res[name] = issued / (best * 1e-3) / 1e9
    del grid64
    del grid
    return res


class Case:
    """One workload resident on the device with the buffers of one entry point (`mode`); step() is one pass of the
    whole hot path through the C ABI."""

    def __init__(self, rt, torch, w, sources, mode="march", variant=0):
        self.rt, self.torch, self.w, self.mode, self.variant = rt, torch, w, mode, variant
        nx, ny, nz = w.shape
        nb = w.n_bins
        self.j, self.kappa = torch.from_numpy(w.j).cuda(), torch.from_numpy(w.kappa).cuda()
        self.src = torch.from_numpy(np.ascontiguousarray(sources)).cuda()
        n_src = int(self.src.shape[0])
        self.units = n_src * w.n_rays * w.n_steps * w.substeps_per_step * nb
        u8 = torch.uint8
        if mode in ("adjoint_j", "adjoint_kappa"):
            torch.manual_seed(939913)          # dL/d out of the adjoint modes: seeded, so the checksums repeat
            self.gbar = torch.rand((w.n_steps, nx, ny, nz, nb), dtype=torch.float32, device="cuda")
            self.result = torch.empty((nx, ny, nz, nb), dtype=torch.float32, device="cuda")
            nbytes = (rt.rt_adjoint_workspace_bytes(nx, ny, nz, n_src, w.n_rays, nb, w.n_steps) if mode == "adjoint_j" else
                      rt.rt_adjoint_kappa_workspace_bytes(nx, ny, nz, n_src, w.n_rays, nb, w.step_size, w.c, w.dt, w.n_steps))
        elif mode == "jvp_kappa":          # the paper's "global kappa scale": dkappa = kappa
            self.result = torch.empty((w.n_steps, nx, ny, nz, nb), dtype=torch.float32, device="cuda")
            nbytes = rt.rt_workspace_bytes(nx, ny, nz, n_src, w.n_rays, nb, w.n_steps)
        elif mode == "step":
            self.state = rt.rt_state_reset(n_src, w.n_rays, nb)
            self.result = torch.empty((nx, ny, nz, nb), dtype=torch.float32, device="cuda")
            nbytes = rt.rt_step_workspace_bytes(nx, ny, nz, n_src, w.n_rays, nb)
        else:
            self.result = torch.empty((w.n_steps, nx, ny, nz, nb), dtype=torch.float32, device="cuda")
            nbytes = rt.rt_workspace_bytes(nx, ny, nz, n_src, w.n_rays, nb, w.n_steps)
        self.ws = torch.empty(max(16, nbytes), dtype=u8, device="cuda")

    def step(self):
        rt, w = self.rt, self.w
        a = (w.n_rays, w.step_size, w.c, w.dt)
        if self.mode == "adjoint_kappa":
            rt.rt_march_adjoint_kappa(self.gbar, self.j, self.kappa, self.src, *a, w.n_steps, grad_kappa=self.result,
                                      workspace=self.ws)
        elif self.mode == "adjoint_j":
            rt.rt_march_adjoint_j(self.gbar, self.kappa, self.src, *a, w.n_steps, grad_j=self.result, workspace=self.ws)
        elif self.mode == "step":        # n_steps calls with persistent ray state, the field accumulated in `result`
            rt.rt_state_reset(int(self.src.shape[0]), w.n_rays, w.n_bins, state=self.state)
            for m in range(w.n_steps):
                rt.rt_march_step(self.j, self.kappa, self.src, *a, m * w.substeps_per_step, self.state, out=self.result,
                                 accumulate=bool(m), workspace=self.ws)
        elif self.mode == "jvp_kappa":
            rt.rt_march_jvp_kappa(self.j, self.kappa, self.kappa, self.src, *a, w.n_steps, tangent=self.result, workspace=self.ws)
        elif self.mode == "trilinear_kappa":
            rt.rt_march_trilinear_kappa(self.j, self.kappa, self.src, *a, w.n_steps, out=self.result, workspace=self.ws)
        else:
            rt.rt_march_ex(self.j, self.kappa, self.src, *a, w.n_steps, out=self.result, workspace=self.ws,
                           variant=self.variant)

    def checksum(self):
        return float(self.result.double().sum().item())


def time_steps(torch, flush, fn, steps, warmup, barrier=None):
    """`warmup` untimed then `steps` timed calls of fn(); a 256 MiB memset between calls (outside the event pairs)
    flushes the L2.  Returns the per-step milliseconds (CUDA events on the launch stream)."""
    for _ in range(max(warmup, 0)):
        flush.zero_()
        fn()
    (barrier or torch.cuda.synchronize)()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in ev:
        flush.zero_()
        e0.record()
        fn()
        e1.record()
    (barrier or torch.cuda.synchronize)()
    return [e0.elapsed_time(e1) for e0, e1 in ev]


L2_BYTES = 126e6


def roofline_of(rt, torch, w, n_src, step_s, ceil=None, mode="march"):
    """The roofline object of one measured case.  Grids that stay L2 resident are bounded by the L2
    reduction rate (peak = M3, the stencil-pattern ceiling measured here on a grid of the same size and bin count);
    grids larger than the L2 by HBM traffic (peak = the measured copy bandwidth)."""
    nx, ny, nz = w.shape
    nb = w.n_bins
    cells = nx * ny * nz * nb
    substeps = n_src * w.n_rays * w.n_steps * w.substeps_per_step
    groups = nb // 4 if nb % 4 == 0 else nb
    alg_reds = 8 * groups * substeps
    hbm_bytes = int((2 + 3 * w.n_steps) * cells * 4)        # j, kappa read; fp64 grid zeroed+read (as 2 fp32 units); out written
    resident = cells * 4 <= L2_BYTES / 1.5         # one fp32 grid against the L2 (C3: 64 MiB, the v4 reduction rate bounds it; C4: 256 MiB, HBM)
    if ceil is None:
        ceil = measure_ceilings(rt, torch, (nx, ny, nz), nb, only=("M3_stencil", "M6_stencil_walk"))
    red = {"achieved": alg_reds / step_s / 1e9, "peak": ceil["M3_stencil"], "unit": "Gred/s",
           "frac": alg_reds / step_s / 1e9 / ceil["M3_stencil"], "M6_stencil_walk": ceil.get("M6_stencil_walk")}
    hbm = {"algorithmic_bytes": hbm_bytes, "achieved": hbm_bytes / step_s / 1e9, "peak": _measured_hbm(), "unit": "GB/s",
           "frac": hbm_bytes / step_s / 1e9 / _measured_hbm(), "peak_is": "MEASURED_PEAKS.json hbm_gbs (of measured)"
           if _have_measured_hbm() else "fallback of B200_PROFILING.md (of fallback)"}
    if resident:
        roof = {"bound": "l2_red", **red, "traffic": None, "hbm": hbm}
    else:
        roof = {"bound": "hbm", **{k: hbm[k] for k in ("achieved", "peak", "unit", "frac")}, "traffic": None,
                "algorithmic_bytes": hbm_bytes, "peak_is": hbm["peak_is"], "l2_red": red}
    roof["how"] = ("achieved = ALGORITHMIC units / mean CUDA-event time of the whole call; l2_red: 8 corners x bin groups x "
                   "ray-substeps against M3 measured in this process (frac > 1: the sliding stencil sums a voxel's deposits "
                   "in registers and issues fewer reductions than the method states); hbm: (2 + 3 n_steps) grids of fp32 "
                   "size against the measured copy bandwidth")
    if mode != "march":
        roof["note"] = f"mode {mode}: the same algorithmic count as the forward march of this workload"
    return roof


def run_native(args):
    import torch
    import torch.distributed as dist

    import paper_2511_09389_b200 as rt          # raises on first use if librtmarch.so is missing: no fallback
    from paper_2511_09389_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (use --impl reference for the CPU oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")             # the communicator lines (ranks, NVLS) stay in the log
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if world != args.gpus and rank == 0:
        print(f"warning: --gpus {args.gpus} but WORLD_SIZE={world}", file=sys.stderr)

    w = make_workload(args.config, world)
    n_src_per_gpu = w.n_src // world
    sl = sharding.source_slice(w.n_src, rank, world)
    nx, ny, nz = w.shape
    nb = w.n_bins
    case = Case(rt, torch, w, w.sources[sl], args.mode, args.variant)
    n_src = int(case.src.shape[0])
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    units_per_gpu = case.units

    def step():
        case.step()
        if world > 1:
            sharding.allreduce_field(case.result)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(max(args.warmup, 0)):
        flush.zero_()
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    t0 = time.perf_counter()
    step_ms = time_steps(torch, flush, step, args.steps, 0, barrier)
    t1 = time.perf_counter()
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_s = float(total_ms.item()) * 1e-3
    if rank == 0:
        time.sleep(0.2)
        sampler.stop()
    clocks = sampler.summary(t0, t1) if rank == 0 else None
    value = units_per_gpu * world * args.steps / total_s

    line = None
    if rank == 0:
        launches = rt.rt_launch_count(nx, ny, nz, n_src, w.n_rays, nb, w.n_steps)
        cfg = describe(w, world)
        cfg["workload"] = cfg["workload"].replace(f"{w.n_src} sources/GPU", f"{n_src_per_gpu} sources/GPU")
        cfg.update({"timing": "CUDA events per step on the launch stream; 256 MiB L2 flush (memset) between "
                              "timed steps, outside the event pairs; inputs resident in HBM",
                    "kernel_variant": args.variant, "mode": args.mode, "field_checksum": case.checksum()})
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": 1e3 * total_s / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": cfg,
                "ray_substeps_per_s": value / nb, "step_ms_each": step_ms, "clocks": clocks,
                "gpu_launches": launches * args.steps, "impl": "native", "library": rt.rt_version()}

    # ---- end to end through the host-pointer entry point: pinned host buffers, H2D + D2H inside the call
    if not args.no_e2e:
        hj, hk = torch.from_numpy(w.j).pin_memory(), torch.from_numpy(w.kappa).pin_memory()
        hs = torch.from_numpy(np.ascontiguousarray(w.sources[sl])).pin_memory()
        hout = torch.empty((w.n_steps, nx, ny, nz, nb), dtype=torch.float32).pin_memory()
        dfield = torch.empty_like(hout, device="cuda") if world > 1 else None
        n_e2e = max(1, min(args.steps, 11))

        def e2e_call():
            rt.rt_march_host(hj.numpy(), hk.numpy(), hs.numpy(), w.n_rays, w.step_size, w.c, w.dt, w.n_steps,
                             out=hout.numpy())
            if world > 1:          # the field leaves the call on the host: sum it over the ranks and bring the sum back
                dfield.copy_(hout, non_blocking=True)
                dist.all_reduce(dfield, op=dist.ReduceOp.SUM)
                hout.copy_(dfield, non_blocking=True)
                torch.cuda.synchronize()

        for _ in range(3):             # untimed: pool allocation, page-locking, clocks back up after the idle gap
            e2e_call()
        barrier()
        e2e_sampler = ClockSampler(local)
        if rank == 0:
            e2e_sampler.start()
            e2e_sampler.wait_first()
        for _ in range(2):             # untimed: the sampler's start-up is over, clocks are back up
            e2e_call()
        barrier()
        te0 = time.perf_counter()
        call_s = []
        for _ in range(n_e2e):
            tc = time.perf_counter()
            e2e_call()
            call_s.append(time.perf_counter() - tc)
        te1 = time.perf_counter()
        barrier()
        if rank == 0:
            time.sleep(0.1)
            e2e_sampler.stop()
        # median call (robust against a stray hiccup of a shared box)
        e2e_s = torch.tensor([sorted(call_s)[len(call_s) // 2] * n_e2e], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
        if rank == 0:
            extra = int(hout.numel() * 4) if world > 1 else 0
            line["e2e"] = {"value": units_per_gpu * world * n_e2e / float(e2e_s.item()), "unit": UNIT,
                           "h2d_bytes_per_step": int(hj.numel() * 4 + hk.numel() * 4 + hs.numel() * 4) + extra,
                           "d2h_bytes_per_step": int(hout.numel() * 4) + extra, "steps": n_e2e,
                           "api": "rt_march_host (device buffers from the library's memory pool + H2D + march + D2H inside the call), "
                                  "wall clock around each synchronous call (median call x steps), pinned host buffers"
                                  + ("; N > 1: the host field goes back to the device, one NCCL sum all-reduce, and back" if world > 1 else ""),
                           "call_ms": [1e3 * t for t in call_s],
                           "min_call_ms": 1e3 * min(call_s), "clocks": e2e_sampler.summary(te0, te1)}
        del hj, hk, hs, hout

    # ---- roofline of the dominant kernel (the march kernel) against the measured L2-reduction ceiling
    if rank == 0:
        ceil = measure_ceilings(rt, torch, (nx, ny, nz), nb)
        step_s = total_s / args.steps
        roof = roofline_of(rt, torch, w, n_src, step_s, ceil, args.mode)
        roof["kernel"] = "march kernel of the call"
        roof["ceilings_Gred_per_s"] = ceil
        if world == 1:
            red = roof if roof["bound"] == "l2_red" else roof["l2_red"]
            red["best_step_frac"] = red["frac"] * step_s / (min(step_ms) * 1e-3)
        if args.mode == "march" and world == 1:
            attach_counters(roof, args.config, args.variant, step_s, n_src * w.n_rays * w.n_steps * w.substeps_per_step,
                            ceil.get("M3_f64_stencil") if nb == 1 else ceil["M3_stencil"], (clocks.get("sm_mhz") or 1965.0) * 1e6)
        line["roofline"] = roof

    # ---- the other large configs and the other entry points, a few steps each (single GPU, default run only)
    if rank == 0 and world == 1 and not args.no_extras and args.config == "C2" and args.mode == "march" and args.variant == 0:
        del case
        torch.cuda.empty_cache()
        line["per_config"], line["modes"] = run_extras(rt, torch, w, flush, args.extra_steps)

    if rank == 0:
        if not args.no_cpu_baseline and world == 1:
            ups, cores, what, _, _ = oracle_sample(make_workload(args.config), args.cpu_seconds)
            line["cpu_baseline"] = {"value": ups, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_extras(rt, torch, w_c2, flush, steps):
    """per_config: C3, C4 and C2 with its sources jittered by +-0.5 cell (sources in general position: no shared cell
    fractions, divergent stencil slides); modes: the other entry points on C2.  Each: `steps` timed calls after 3
    warm-ups, CUDA events, L2 flushed between calls; its own roofline; a checksum of the result."""
    import workloads

    def measure(w, sources, mode="march", label=None):
        case = Case(rt, torch, w, sources, mode)
        ms = time_steps(torch, flush, case.step, steps, 3)
        mean_s = sum(ms) / len(ms) * 1e-3
        n_src = int(case.src.shape[0])
        row = {"workload": label or describe(w, 1)["workload"], "mode": mode, "steps": steps, "warmup": 3,
               "ms_per_step": 1e3 * mean_s, "step_ms_each": ms, "updates_per_s": case.units / mean_s,
               "ray_substeps_per_s": case.units / w.n_bins / mean_s, "checksum": case.checksum(),
               "gpu_launches_per_step": rt.rt_launch_count(*w.shape, n_src, w.n_rays, w.n_bins, w.n_steps) if mode == "march" else None,
               "roofline": roofline_of(rt, torch, w, n_src, mean_s, None, mode)}
        if mode == "march" and label is None:
            rf = row["roofline"]
            attach_counters(rf, w.name, 0, mean_s, n_src * w.n_rays * w.n_steps * w.substeps_per_step,
                            rf["peak"] if rf["bound"] == "l2_red" else rf["l2_red"]["peak"], 1965.0e6)
        del case
        torch.cuda.empty_cache()
        return row

    modes = {m: measure(w_c2, w_c2.sources, m) for m in ("step", "trilinear_kappa", "adjoint_j", "adjoint_kappa", "jvp_kappa")}
    per_config = {}
    jit = (w_c2.sources.astype(np.float64) + np.random.default_rng(939912).uniform(-0.5, 0.5, w_c2.sources.shape))
    jit = np.clip(jit, 0.0, w_c2.shape[0] - 1.0).astype(np.float32)
    per_config["C2_jittered"] = measure(w_c2, jit, label=describe(w_c2, 1)["workload"] +
                                        "; sources moved off the cell nodes by uniform(-0.5, 0.5) per axis (seed 939912)")
    for name in ("C3", "C4"):
        w = workloads.make_config(name)
        per_config[name] = measure(w, w.sources)
        del w
    return per_config, modes


def _ncu_counters(config, variant):
    """Per-launch ncu counters of the march kernel (committed text under profiles/, one capture per kernel
    revision).  None if there is no capture of this case for the loaded library."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "march_counters.csv"), newline="") as f:
            for row in csv.DictReader(f):
                if row["case"] == f"{config}:v{variant}" and row["library"] == _lib_version():
                    out = {k: float(row[k]) for k in ("warp_instructions", "red_sectors", "dram_bytes", "issue_active_pct",
                                                      "l1_lsu_wavefronts_pct", "l2_hit_pct", "warps_active_pct", "registers")}
                    out.update(source=row["source"], kernel=row["kernel"])
                    return out
    except (OSError, KeyError, ValueError):
        pass
    return None


def attach_counters(roof, config, variant, step_s, substeps, red_ceiling, sm_hz):
    """`traffic`, `issued`, `alu`, `lsu`: ncu counters of the march kernel of this case REPLAYED from the committed capture
    (profiles/march_counters.csv, same library version string), per launch, divided by the step time measured here."""
    cnt = _ncu_counters(config, variant)
    if not cnt:
        return
    roof["traffic"] = cnt["dram_bytes"]
    roof["issued"] = {"red_sectors_per_launch": cnt["red_sectors"], "red_sectors_per_ray_substep": cnt["red_sectors"] / substeps,
                      "achieved_Gsectors_per_s": cnt["red_sectors"] / step_s / 1e9,
                      "frac_of_M3": cnt["red_sectors"] / step_s / 1e9 / red_ceiling if red_ceiling else None}
    roof["alu"] = {"warp_instructions_per_launch": cnt["warp_instructions"],
                   "warp_instructions_per_warp_substep": cnt["warp_instructions"] / (substeps / 32),
                   "achieved_Ginst_per_s": cnt["warp_instructions"] / step_s / 1e9, "peak_Ginst_per_s": 148 * 4 * sm_hz / 1e9,
                   "frac": cnt["warp_instructions"] / step_s / (148 * 4 * sm_hz), "issue_active_pct_under_ncu": cnt["issue_active_pct"],
                   "peak_how": "148 SMs x 4 schedulers x 1 warp-instruction/clk x SM clock sampled in the run"}
    roof["lsu"] = {"l1_lsu_data_pipe_wavefronts_pct_of_peak_under_ncu": cnt["l1_lsu_wavefronts_pct"], "l2_hit_pct": cnt["l2_hit_pct"],
                   "warps_active_pct": cnt["warps_active_pct"], "registers_per_thread": cnt["registers"],
                   "note": "the busiest unit of the one-bin march: one wavefront per 32-byte sector of a scattered load or "
                           "reduction (DESIGN.md §7)"}
    roof["kernel"] = cnt["kernel"]
    roof["counters_from"] = cnt["source"]
    roof["how"] += ("; `traffic`, `issued`, `alu` and `lsu` are REPLAYED from the committed ncu capture named in "
                    "`counters_from` (same library version string), divided by the step time measured here")


def _lib_version():
    import paper_2511_09389_b200 as rt
    return rt.rt_version()


def _measured_hbm():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except (OSError, KeyError, ValueError):
        return 6650.0      # fallback of B200_PROFILING.md


def _have_measured_hbm():
    return os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json"))


if __name__ == "__main__":
    a = parse()
    sys.exit(run_reference(a) if a.impl == "reference" else run_native(a))
