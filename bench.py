#!/usr/bin/env python
"""bench.py — ray-substep-bin updates/s of the Ray-trax march (BASELINE.json metric) on N B200s.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl reference]

A "step" is one pass of the whole hot path: one rt_march call (zero-fill, ray-order, march, snapshot
prefix) over the full workload.  Default workload = BASELINE.json configs[2] ("C2": 128^3, 4,096 rays,
2,097 sources at the density peaks, 444 substeps), the configuration the metric is quoted on.
One JSON line is printed by rank 0; see DESIGN.md §8 for every field.

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
    ap.add_argument("--mode", default="march", choices=["march", "step", "trilinear_kappa", "adjoint_j", "adjoint_kappa"],
                    help="march: one rt_march call per bench step (the headline); step: the same workload as n_steps "
                         "rt_march_step calls with persistent ray state (DESIGN.md D17); trilinear_kappa: "
                         "rt_march_trilinear_kappa (DESIGN.md D18); adjoint_j: rt_march_adjoint_j, dL/dj for a "
                         "random dL/d out (DESIGN.md D19; `out` then holds nothing useful)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target host time of the oracle sample")
    return ap.parse_args()


def make_workload(name, world_size=1):
    """Config `name`; for world_size > 1 the source list is extended to world_size * n_src sources by the
    config's own placement rule (weak scaling: per-GPU work fixed)."""
    from paper_2511_09389_b200 import workloads
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
def measure_ceilings(rt, torch, shape, n_bins):
    """Reduction-throughput ceilings on a grid of the workload's size, in this process, back to back with
    the march: best of 5 launches of >= 2^28 reductions each, CUDA events.  Greds/s."""
    grid = torch.zeros(shape + (n_bins,), dtype=torch.float32, device="cuda")
    grid64 = torch.zeros(shape + (n_bins,), dtype=torch.float64, device="cuda")
    res = {}
    for name, mode in rt.binding.RED_MODES.items():
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


def run_native(args):
    import torch
    import torch.distributed as dist

    import paper_2511_09389_b200 as rt          # raises if librtmarch.so is missing: no fallback
    from paper_2511_09389_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (use --impl reference for the CPU oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if world != args.gpus and rank == 0:
        print(f"warning: --gpus {args.gpus} but WORLD_SIZE={world}", file=sys.stderr)

    w = make_workload(args.config, world)
    n_src_per_gpu = w.n_src // world
    sl = sharding.source_slice(w.n_src, rank, world)
    nx, ny, nz = w.shape
    nb = w.n_bins
    j, kappa = torch.from_numpy(w.j).cuda(), torch.from_numpy(w.kappa).cuda()
    src = torch.from_numpy(np.ascontiguousarray(w.sources[sl])).cuda()
    out = torch.empty((w.n_steps, nx, ny, nz, nb), dtype=torch.float32, device="cuda")
    ws = rt.alloc_workspace(nx, ny, nz, src.shape[0], w.n_rays, nb, w.n_steps)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2
    units_per_gpu = src.shape[0] * w.n_rays * w.n_steps * w.substeps_per_step * nb

    if args.mode == "step":
        state = rt.rt_state_reset(src.shape[0], w.n_rays, nb)
        ws_step = torch.empty(max(16, rt.rt_step_workspace_bytes(nx, ny, nz, src.shape[0], w.n_rays, nb)),
                              dtype=torch.uint8, device="cuda")

    if args.mode == "adjoint_j":
        gbar = torch.rand((w.n_steps, nx, ny, nz, nb), dtype=torch.float32, device="cuda")
        grad_j = torch.empty((nx, ny, nz, nb), dtype=torch.float32, device="cuda")
        ws_adj = torch.empty(max(16, rt.rt_adjoint_workspace_bytes(nx, ny, nz, src.shape[0], w.n_rays, nb, w.n_steps)),
                             dtype=torch.uint8, device="cuda")

    if args.mode == "adjoint_kappa":
        gbar = torch.rand((w.n_steps, nx, ny, nz, nb), dtype=torch.float32, device="cuda")
        grad_j = torch.empty((nx, ny, nz, nb), dtype=torch.float32, device="cuda")
        ws_adj = torch.empty(max(16, rt.rt_adjoint_kappa_workspace_bytes(nx, ny, nz, src.shape[0], w.n_rays, nb, w.step_size,
                                                                         w.c, w.dt, w.n_steps)),
                             dtype=torch.uint8, device="cuda")

    def step():
        if args.mode == "adjoint_kappa":
            rt.rt_march_adjoint_kappa(gbar, j, kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps, grad_kappa=grad_j,
                                      workspace=ws_adj)
            return
        if args.mode == "adjoint_j":
            rt.rt_march_adjoint_j(gbar, kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps, grad_j=grad_j,
                                  workspace=ws_adj)
            return
        if args.mode == "step":        # n_steps calls, the field of the last snapshot accumulated in out[-1]
            rt.rt_state_reset(src.shape[0], w.n_rays, nb, state=state)
            out[-1].zero_()
            for m in range(w.n_steps):
                rt.rt_march_step(j, kappa, src, w.n_rays, w.step_size, w.c, w.dt, m * w.substeps_per_step, state,
                                 out=out[-1], accumulate=True, workspace=ws_step)
        elif args.mode == "trilinear_kappa":
            rt.rt_march_trilinear_kappa(j, kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps, out=out, workspace=ws)
        else:
            rt.rt_march_ex(j, kappa, src, w.n_rays, w.step_size, w.c, w.dt, w.n_steps, out=out, workspace=ws,
                           variant=args.variant)
        if world > 1:
            sharding.allreduce_field(out)

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
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    t0 = time.perf_counter()
    for e0, e1 in ev:
        flush.zero_()                 # L2 flush between timed iterations (outside the event pair)
        e0.record()
        step()
        e1.record()
    barrier()
    t1 = time.perf_counter()
    step_ms = [e0.elapsed_time(e1) for e0, e1 in ev]
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
        field_sum = float((out[-1] if args.mode == "step" else out).double().sum().item())
        launches = rt.rt_launch_count(nx, ny, nz, int(src.shape[0]), w.n_rays, nb, w.n_steps)
        cfg = describe(w, world)
        cfg["workload"] = cfg["workload"].replace(f"{w.n_src} sources/GPU", f"{n_src_per_gpu} sources/GPU")
        cfg.update({"timing": "CUDA events per step on the launch stream; 256 MiB L2 flush (memset) between "
                              "timed steps, outside the event pairs; inputs resident in HBM",
                    "kernel_variant": args.variant, "mode": args.mode, "field_checksum": field_sum})
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
        n_e2e = max(1, min(args.steps, 11))
        for _ in range(3):             # untimed: pool allocation, page-locking, clocks back up after the idle gap
            rt.rt_march_host(hj.numpy(), hk.numpy(), hs.numpy(), w.n_rays, w.step_size, w.c, w.dt, w.n_steps,
                             out=hout.numpy())
        barrier()
        e2e_sampler = ClockSampler(local)
        if rank == 0:
            e2e_sampler.start()
            time.sleep(0.1)
        te0 = time.perf_counter()
        call_s = []
        for _ in range(n_e2e):
            tc = time.perf_counter()
            rt.rt_march_host(hj.numpy(), hk.numpy(), hs.numpy(), w.n_rays, w.step_size, w.c, w.dt, w.n_steps,
                             out=hout.numpy())
            if world > 1:          # the field leaves the call on the host: reduce it there
                dist.all_reduce(hout.cuda(), op=dist.ReduceOp.SUM)
                torch.cuda.synchronize()
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
            line["e2e"] = {"value": units_per_gpu * world * n_e2e / float(e2e_s.item()), "unit": UNIT,
                           "h2d_bytes_per_step": int(hj.numel() * 4 + hk.numel() * 4 + hs.numel() * 4),
                           "d2h_bytes_per_step": int(hout.numel() * 4), "steps": n_e2e,
                           "api": "rt_march_host (device buffers from the library's memory pool + H2D + march + D2H inside the call), "
                                  "wall clock around each synchronous call (median call x steps), pinned host buffers", "call_ms": [1e3 * t for t in call_s],
                           "min_call_ms": 1e3 * min(call_s), "clocks": e2e_sampler.summary(te0, te1)}

    # ---- roofline of the dominant kernel (the march kernel) against the measured L2-reduction ceiling
    if rank == 0:
        ceil = measure_ceilings(rt, torch, (nx, ny, nz), nb)
        step_s = total_s / args.steps
        reds_per_substep = 8 * (nb // 4 if nb % 4 == 0 else nb)           # algorithmic: 8 corners x bin groups
        alg_reds = reds_per_substep * src.shape[0] * w.n_rays * w.n_steps * w.substeps_per_step
        achieved = alg_reds / step_s / 1e9
        peak = ceil["M3_stencil"]
        hbm_bytes = int((2 + 3 * w.n_steps) * nx * ny * nz * nb * 4)      # j, kappa read; fp64 grid zeroed+read; out written
        roof = {
            "bound": "l2_red", "achieved": achieved, "peak": peak, "unit": "Gred/s", "frac": achieved / peak,
            "traffic": None, "kernel": "march_sliding_kernel",
            "how": "achieved = ALGORITHMIC reductions (8 corners x bin-groups x ray-substeps) / mean CUDA-event "
                   "time of the whole rt_march call (the march kernel is 99% of it at C2, profiles/r01f); peak = "
                   "M3 stencil-pattern red.global.add ceiling measured in this process on a grid of the same "
                   "size (DESIGN.md §8), of measured; frac > 1: the sliding stencil sums a voxel's deposits in "
                   "registers, so fewer reductions are issued than the method states (see `issued`)",
            "best_step_frac": alg_reds / (min(step_ms) * 1e-3) / 1e9 / peak if world == 1 else None,
            "ceilings_Gred_per_s": ceil,
            "hbm": {"algorithmic_bytes": hbm_bytes, "achieved_GBps": hbm_bytes / step_s / 1e9,
                    "peak_GBps": _measured_hbm(), "note": "grids are L2 resident at C0-C2: HBM is not the bound"}}
        cnt = _ncu_counters(args.config, args.variant)
        if cnt and world == 1:
            sm_hz = (clocks.get("sm_mhz") or 1965.0) * 1e6
            roof["traffic"] = cnt["dram_bytes"]
            roof["issued"] = {"red_sectors_per_launch": cnt["red_sectors"],
                              "red_sectors_per_ray_substep": cnt["red_sectors"] / (alg_reds / reds_per_substep),
                              "achieved_Gsectors_per_s": cnt["red_sectors"] / step_s / 1e9,
                              "frac_of_M3": cnt["red_sectors"] / step_s / 1e9 / ceil["M3_f64_stencil"]}
            roof["alu"] = {"warp_instructions_per_launch": cnt["warp_instructions"],
                           "achieved_Ginst_per_s": cnt["warp_instructions"] / step_s / 1e9,
                           "peak_Ginst_per_s": 148 * 4 * sm_hz / 1e9,
                           "frac": cnt["warp_instructions"] / step_s / (148 * 4 * sm_hz),
                           "peak_how": "148 SMs x 4 schedulers x 1 warp-instruction/clk x SM clock sampled in the run"}
            roof["kernel"] = cnt["kernel"]
            roof["counters_from"] = cnt["source"]
        line["roofline"] = roof
        if not args.no_cpu_baseline and world == 1:
            ups, cores, what, _, _ = oracle_sample(make_workload(args.config), args.cpu_seconds)
            line["cpu_baseline"] = {"value": ups, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def _ncu_counters(config, variant):
    """Per-launch ncu counters of the march kernel (committed text under profiles/, one capture per kernel
    revision): instruction count, L2 reduction sectors, DRAM bytes.  None if there is no capture for this case."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "march_counters.csv"), newline="") as f:
            for row in csv.DictReader(f):
                if row["case"] == f"{config}:v{variant}" and row["library"] == _lib_version():
                    return {"warp_instructions": float(row["warp_instructions"]), "red_sectors": float(row["red_sectors"]),
                            "dram_bytes": float(row["dram_bytes"]), "source": row["source"], "kernel": row["kernel"]}
    except (OSError, KeyError, ValueError):
        pass
    return None


def _lib_version():
    import paper_2511_09389_b200 as rt
    return rt.rt_version()


def _measured_hbm():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except (OSError, KeyError, ValueError):
        return 6650.0      # fallback of B200_PROFILING.md


if __name__ == "__main__":
    a = parse()
    sys.exit(run_reference(a) if a.impl == "reference" else run_native(a))
