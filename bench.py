#!/usr/bin/env python
"""bench.py -- throughput of the RTS hot path on B200 (one JSON line on stdout).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one pass of the whole hot path (stage A + all sweep passes + J/Q reduction +
I_top) over one synthetic atmosphere, i.e. one rts_solve.  Default workload: BASELINE.json
configs[2] (4-band RTS on 288^3, the configuration the metric is quoted on).

  value       whole-job cell*band*ray updates/s (U = N*nb*24*P per solve), inputs resident in
              HBM, device-timed with CUDA events, max over ranks
  e2e         same metric through rts_solve_host: pinned HOST buffers in and out, copies timed
  roofline    dominant kernel (rts_sweep_kernel): algorithmic bytes of SURVEY.md 8(d)'s
              compulsory-byte model / its event-timed duration, against MEASURED_PEAKS.json
  cpu_baseline the fp64 oracle, as it stands, on the box's host cores, bounded sample

N > 1 (torchrun): by default the path is run as N independent replicas (one atmosphere per rank, no
data-path collective) -> "scaling": "weak".  --scaling strong shards ONE box by band x octant (rts_set_shard):
every rank sweeps its units, one NCCL sum all-reduce completes Q_rad and I_top inside the timed region.
--impl reference times the oracle (rank 0 only).
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

METRIC = "rts_cell_band_ray_updates_per_s"
UNIT = "updates/s"


def compulsory_bytes(nx, ny, nz, nb, P, n_up=12):
    """SURVEY.md 8(d) compulsory-byte model (fp32 kaprho, S; 8 (octant) traversals per pass)."""
    N = nx * ny * nz
    stage_a = N * (12 + 8 * nb)
    sweep = 8 * P * N * 8 * nb + N * 4 * (8 + 7) + nb * n_up * nx * ny * 4
    return stage_a, sweep


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(inp, sample_bands=1):
    """Time the oracle on a bounded sample: the first `sample_bands` bands of the workload."""
    import copy
    import oracle
    sub = copy.copy(inp)
    sub.nbands = sample_bands
    sub.logkappa = np.ascontiguousarray(inp.logkappa[:sample_bands])
    sub.bandfrac = np.ascontiguousarray(inp.bandfrac[:sample_bands])
    oracle.build()
    t0 = time.perf_counter()
    oracle.solve(sub)
    dt = time.perf_counter() - t0
    return sub.updates / dt, dt, oracle.num_threads(), sub.updates


def run_reference(args, inputs_mod):
    """--impl reference: the oracle on host cores (rank 0 only)."""
    from paper_2107_08145_b200 import multi
    if not multi.reference_arm_runs_here(multi.env_ranks()[0]):
        return 0
    inp = inputs_mod.make_config(args.config)
    sample_bands = 1
    # warm-up steps are a smaller sample (first band of a 1/8 sub-volume would change the
    # workload; instead warm-up = build + one coefficient evaluation)
    import oracle
    oracle.build()
    for _ in range(args.warmup):
        oracle.coefficients(inputs_mod.make_config(1))
    vals, times = [], []
    cores = oracle.num_threads()
    upd = 0
    for _ in range(args.steps):
        v, dt, cores, upd = oracle_sample(inp, sample_bands)
        vals.append(v); times.append(dt)
    value = upd * len(times) / sum(times)
    sample = (f"band 0 of {inp.nbands} on the full {inp.nx}x{inp.ny}x{inp.nz} grid, 24 rays, "
              f"{inp.npasses} passes = {upd:.3e} updates per step")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(times) / len(times),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": workload_name(args.config, inp), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_name(cfg, inp):
    return (f"BASELINE.json configs[{cfg - 1}]: {inp.nbands}-band RTS on {inp.nx}x{inp.ny}x{inp.nz}, "
            f"24 rays, {inp.npasses} passes")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one atmosphere per rank; strong = one box sharded by band x octant")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    from paper_2107_08145_b200 import inputs as inputs_mod
    if args.impl == "reference":
        return run_reference(args, inputs_mod)

    import torch
    import torch.distributed as dist
    from paper_2107_08145_b200 import multi, rts

    rank, local_rank, world = multi.env_ranks()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (no CPU fallback exists)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    # weak: one independent atmosphere per rank (replicas; no data-path collective)
    # strong: the same box on every rank, sweep units dealt round robin, one sum all-reduce of Q and I_top
    strong = (args.scaling == "strong" and world > 1)
    inp = inputs_mod.make_config(args.config, seed_offset=0 if strong else multi.rank_seed_offset(rank))
    solver = rts.from_inputs(inp, shard=(rank, world) if strong else None)
    plan = solver.plan_info()
    solver.enable_timing(True)
    rho, T, P = (torch.from_numpy(a).cuda() for a in (inp.rho, inp.T, inp.P))
    Q = torch.empty(inp.shape, dtype=torch.float32, device="cuda")
    Itop = torch.empty((inp.nbands, inp.n_up, inp.ny, inp.nx), dtype=torch.float32, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def reduce_max(x):
        return multi.max_over_ranks(x, world, "cuda")

    def step():
        solver.solve(rho, T, P, Q, Itop)
        if strong:
            multi.allreduce_sum(world, Q, Itop)

    # ---- device-resident timing
    for _ in range(args.warmup):
        step()
    solver.sync_check()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sweep_ms, stage_a_ms = [], []
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    solver.sync_check()
    local_ms = ev0.elapsed_time(ev1) / args.steps
    # per-stage durations of the kernels (CUDA events recorded on the solve stream inside rts_solve): the same
    # number of solves again, read back one by one (the events belong to the context, so each read waits)
    for _ in range(args.steps):
        solver.solve(rho, T, P, Q, Itop)
        tm = solver.last_timing()
        sweep_ms.append(tm["sweep_ms"]); stage_a_ms.append(tm["stage_a_ms"])
    solver.sync_check()
    clocks = sampler.stop() if rank == 0 else None
    agg = multi.aggregate(local_ms, float(inp.updates), world, "cuda")
    if strong:                         # one box: the job's units are the box's, not world x
        agg["value"] = float(inp.updates) / (agg["ms"] * 1e-3)

    # ---- end to end through the host-buffer entry point (pinned buffers, copies timed)
    e2e = None
    if not args.no_e2e:
        hr, hT, hP = (torch.from_numpy(a).pin_memory() for a in (inp.rho, inp.T, inp.P))
        hQ = torch.empty(inp.shape, dtype=torch.float32).pin_memory()
        hI = torch.empty((inp.nbands, inp.n_up, inp.ny, inp.nx), dtype=torch.float32).pin_memory()
        solver.solve_host(hr, hT, hP, hQ, hI)
        barrier()
        ke = max(3, min(args.steps, 5))
        t0 = time.perf_counter()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(ke):
            solver.solve_host(hr, hT, hP, hQ, hI)
        e1.record()
        barrier()
        e2e_ms = e0.elapsed_time(e1) / ke
        e2e_ms = max(e2e_ms, (time.perf_counter() - t0) * 1e3 / ke) if world == 1 else e2e_ms
        e2e_ms = reduce_max(e2e_ms)
        N = inp.ncells
        e2e = {"value": world * inp.updates / (e2e_ms * 1e-3), "unit": UNIT, "ms_per_step": e2e_ms,
               "h2d_bytes_per_step": 3 * N * 4, "d2h_bytes_per_step": (N + inp.nbands * inp.n_up * inp.ny * inp.nx) * 4,
               "checksum_Q": float(np.abs(hQ.numpy()).max())}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel
    peak, peak_src = measured_peaks()
    a_bytes, s_bytes = compulsory_bytes(inp.nx, inp.ny, inp.nz, inp.nbands, inp.npasses, inp.n_up)
    rounds = 1          # the whole sweep is one persistent launch
    sweep_launch_ms = float(np.mean(sweep_ms)) / rounds
    achieved = (s_bytes / rounds) / (sweep_launch_ms * 1e-3) / 1e9
    roofline = {
        "bound": "hbm", "kernel": "rts_sweep_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
        "algorithmic_bytes_per_launch": s_bytes / rounds, "launches_per_step": rounds,
        "avg_launch_ms": sweep_launch_ms, "min_launch_ms": float(np.min(sweep_ms)) / rounds, "launches_timed": len(sweep_ms),
        "note": "bound 'hbm' is north_star's reporting convention; the kernel is bound by shared-memory bandwidth "
                "and issue latency inside a step and by inter-CTA exchange latency between blocks (DESIGN.md 8, profiles/)",
        "solve_frac_of_compulsory_byte_roofline": ((a_bytes + s_bytes) / (local_ms * 1e-3) / 1e9) / peak,
        "stage_a_ms": float(np.mean(stage_a_ms)),
    }
    # measured DRAM bytes per launch (ncu --set full capture): only when the stored capture is of this workload and plan
    prof = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(prof) and world == 1:
        try:
            with open(prof) as fh:
                tj = json.load(fh)
            if tj.get("config") == args.config and tj.get("tile_u_z") == plan.get("tile_u_z") and tj.get("tile_v_z") == plan.get("tile_v_z"):
                roofline["traffic"] = tj.get("rts_sweep_kernel_dram_bytes_per_launch")
        except Exception:
            pass

    # ---- thick-plane shortcut: updates stay nominal, the skipped share is reported
    thick = None
    if world == 1:
        levels = solver.thick_levels()
        n_zrays = plan["z_march_rays"]                                       # as the library grouped the rays
        skipped = sum(levels) * inp.nx * inp.ny * n_zrays * (inp.npasses - 1)
        thick = {"levels_per_band": levels, "z_march_rays": n_zrays,
                 "skipped_fraction_of_updates": skipped / float(inp.updates)}

    # ---- grid staggering: its two HBM-bound kernels against the same peak
    stag = None
    if world == 1:
        N = inp.ncells
        Nc = (inp.nz - 1) * inp.ny * inp.nx
        cell = torch.rand((inp.nz - 1, inp.ny, inp.nx), dtype=torch.float32, device="cuda") + 1.0
        node = torch.empty(inp.shape, dtype=torch.float32, device="cuda")
        reps = 20
        def timed(fn):
            for _ in range(3):
                fn()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); a.record()
            for _ in range(reps):
                fn()
            b.record(); torch.cuda.synchronize()
            return a.elapsed_time(b) / reps
        t_c2n = timed(lambda: solver.cells_to_nodes(cell, node))
        t_n2c = timed(lambda: solver.nodes_to_cells(node, cell))
        bytes_f = (N + Nc) * 4                       # one field read once, one written once
        stag = {"cells_to_nodes_ms_per_field": t_c2n, "nodes_to_cells_ms": t_n2c,
                "algorithmic_bytes_per_launch": bytes_f,
                "cells_to_nodes_frac_of_hbm": bytes_f / (t_c2n * 1e-3) / 1e9 / peak,
                "nodes_to_cells_frac_of_hbm": bytes_f / (t_n2c * 1e-3) / 1e9 / peak,
                "note": "one field per launch; source + destination exceed the L2 at the 288^3 and 512x512x192 sizes"}
        del cell, node

    # ---- scattering source function: all bands of the same atmosphere, eps = 0.1, two
    #      iterations of the source update along the ray (fp64 kernel, one grid barrier per plane: DESIGN.md 7.5)
    scat = None
    if world == 1:
        kap, Bsrc = solver.coefficients(rho, T, P)
        eps = torch.full_like(kap, 0.1)
        solver.scatter_solve(kap, Bsrc, eps, 1)
        n_it = 2
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(); a.record()
        _, _, change = solver.scatter_solve(kap, Bsrc, eps, n_it)
        b.record(); torch.cuda.synchronize()
        t_it = a.elapsed_time(b) / n_it
        scat = {"ms_per_iteration": t_it, "node_band_ray_updates_per_s": inp.ncells * inp.nbands * inp.nrays / (t_it * 1e-3),
                "dtype": "f64", "bands": inp.nbands, "rays": inp.nrays, "eps": 0.1,
                "scheme": "source update along the ray (Gauss-Seidel)", "last_change_per_band": change[-1],
                "note": "one grid-wide barrier per plane of every ray; small grids are bound by it and by the dependent loads of a plane step, 288^3 by the strided accesses that are left on the x-march rays (S and J) and by three nodes per thread with four bands (DESIGN.md 7.5)"}
        del kap, Bsrc, eps

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        v, dt, cores, upd = oracle_sample(inp, 1)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt,
               "sample": f"band 0 of {inp.nbands} on the full {inp.nx}x{inp.ny}x{inp.nz} grid, 24 rays, "
                         f"{inp.npasses} passes = {upd:.3e} updates"}

    line = {
        "metric": METRIC, "value": agg["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": agg["ms"], "higher_is_better": True, "scaling": "strong" if strong else "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(args.config, inp), "grid": [inp.nx, inp.ny, inp.nz],
                   "bands": inp.nbands, "rays": inp.nrays, "passes": inp.npasses,
                   "updates_per_step": inp.updates, "parallelism": (f"band x octant shards x{world}, one sum all-reduce of Q and I_top" if strong else f"replicas x{world}"),
                   "cache": "working set (kaprho,S fields, 2 layouts) >> L2: inputs larger than L2, no flush needed",
                   "plan": plan},
        "solve_ms": agg["ms"], "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
        "staggering": stag, "scattering": scat, "thick_skip": thick,
        "gpu_launches": plan["launches"] * args.steps, "clocks": clocks,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
