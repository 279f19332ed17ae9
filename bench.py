#!/usr/bin/env python
"""bench.py -- particles pushed + mass-matrix-deposited per second (FP64) on B200, libecpush.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl reference]

A "step" is one pass of the whole hot path (gather, alpha, push, deposit of
rho/Jhat/M, per-cell pre-reduction and flush) over every particle of every species of the workload,
through the C ABI (ecsim_push_and_moments_all), starting from the cell-sorted state.  Default
workload: BASELINE.json configs[2] (128^3 cells, 2 species x 64 ppc = 268,435,456 particles), the
configuration the metric is quoted on.  Protocol: inputs
resident in HBM; each step timed with CUDA events on the library's stream; the particle state is
restored from a pristine device copy between steps, outside the timed region; the working set
(15 GB of particles, 4 GB of M) is far larger than the 126 MB L2, so no explicit flush is needed.

One JSON line on stdout (rank 0).  `--impl reference` times the CPU oracle (oracle/, as it
stands, all host cores) on a bounded sample of the same workload instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particles pushed+mass-matrix-deposited per sec (FP64); % of B200 roofline"
UNIT = "particles/s"
# algorithmic FP64 work per particle in the minimum (27-class) formulation and
# algorithmic HBM bytes per particle at 128 particles per node.
FLOP_PER_PARTICLE = 813.0
BYTES_PER_PARTICLE_CFG2 = 119.8
# FP64 vector peak derived from unit counts and clocks: 148 SM x 64 FMA/clk x 2 flop x 1.965 GHz
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
NORTH_STAR_ROOFLINE_PPS = min(8.0e12 / BYTES_PER_PARTICLE_CFG2, FP64_PEAK_TFLOPS * 1e12 / FLOP_PER_PARTICLE)


def profiled_traffic(kernel_substring: str, launch_list_glob: str = "profiles/r*_launches_cfg2.csv"):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a kernel, read from the newest COMMITTED ncu launch list
    of the headline workload (profiles/rNN?_launches_cfg2.csv, written by the command named in the README beside it).
    Returns (bytes, file) or (None, None): never a constant typed into this file."""
    import csv
    import glob
    for path in sorted(glob.glob(os.path.join(ROOT, launch_list_glob)), reverse=True):
        per_launch = {}
        try:
            for r in csv.reader(open(path)):
                if len(r) > 14 and kernel_substring in r[4] and r[12] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                    per_launch.setdefault(r[0], {})[r[12]] = float(r[14].replace(",", ""))
        except (OSError, ValueError):
            continue
        full = [v["dram__bytes_read.sum"] + v["dram__bytes_write.sum"] for v in per_launch.values() if len(v) == 2]
        if full:
            return sum(full) / len(full), os.path.relpath(path, ROOT)
    return None, None


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="libecpush", choices=["libecpush", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (default 2, the headline)")
    ap.add_argument("--scale", default=None, help="nx,ny,nz override of the grid (tests / quick runs)")
    ap.add_argument("--variant", default="fused", choices=["fused", "atomic"])
    ap.add_argument("--fused-warps", type=int, default=-1, help="8 / 12 / 16 warps per CTA of the fused kernel (library default 12)")
    ap.add_argument("--m-layout", type=int, default=27, choices=[27, 14],
                    help="mass-matrix storage: 27 slots per node (north-star, default) or the paper's 14 (L73)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-sample-planes", type=int, default=32, help="x-planes of cells the oracle sample covers")
    ap.add_argument("--no-rows", action="store_true", help="skip the timings of the separate SURVEY 8(f) calls (moments, push, apply_M, diagnostics)")
    ap.add_argument("--no-configs", action="store_true",
                    help="skip the block that times the other BASELINE.json configs (0, 1, 3, 4) and configs[2] with 14 M slots")
    ap.add_argument("--sustained-steps", type=int, default=-1,
                    help="consecutive steps WITHOUT restoring the particle state (default: 10; configs[1]: its 1 + 10 protocol; 0 = skip)")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------
def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def max_over_ranks(values, world, backend_device="cuda"):
    """Element-wise max of a list of floats over all ranks (torch.distributed); identity at world 1."""
    if world == 1:
        return list(values)
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def sum_over_ranks(value, world, backend_device="cuda"):
    if world == 1:
        return value
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.cpu()[0])


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    QUERY = ("timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits", "-lms", "25",
                 "-i", str(self.gpu)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self, t_begin=None, t_end=None):
        """Summary of the samples whose nvidia-smi timestamp lies in [t_begin, t_end] (time.time() values; the sampler is
        started long before, because nvidia-smi needs a few tenths of a second for its first line)."""
        import datetime
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            if t_begin is not None:
                try:
                    ts = datetime.datetime.strptime(f[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                except ValueError:
                    continue
                if ts < t_begin - 0.03 or ts > t_end + 0.03:
                    continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # under load = samples drawing more than half of the maximum power seen
        pmax = max(power)
        loaded = [c for c, p in zip(sm, power) if p >= 0.5 * pmax] or sm
        return {"sm_mhz": statistics.median(loaded), "sm_max_mhz": max(smax), "reasons": sorted(reasons),
                "power_w_max": pmax, "samples": len(sm)}


# ------------------------------------------------------------------------------------------------
def load_config(args):
    import workloads as wl
    scale = tuple(int(v) for v in args.scale.split(",")) if args.scale else None
    return wl.config(args.config, scale)


def workload_name(cfg):
    n = None
    return f"BASELINE.json configs[{cfg.idx}] {cfg.name}: {cfg.nx}x{cfg.ny}x{cfg.nz} cells, {len(cfg.species)} species"


def oracle_sample(cfg, planes, all_cores=True):
    """Time the CPU oracle (oracle/ecsim_oracle.c as it stands: plain C, gcc -O2 -ffp-contract=off) on the particles of
    the first `planes` x-planes of cells of the workload, on the full-size grid.  all_cores: through
    oracle.step_planes, which calls the same per-particle loop per x-plane of cells, even planes in parallel, then odd
    planes (no arithmetic of its own).  Returns (particles/s, n, seconds, threads used)."""
    import numpy as np
    import oracle
    import workloads as wl
    from workloads import grid_of, to_numpy
    planes = max(1, min(planes, cfg.nx))
    cells = list(range(planes * cfg.ny * cfg.nz))
    E, B = wl.gen_fields(cfg)
    En, Bn = E.numpy(), B.numpy()
    parts = [to_numpy(wl.gen_species(cfg, s, cells=cells)) for s in range(len(cfg.species))]
    n = sum(p["x"].shape[0] for p in parts)
    _, start = wl.cell_layout(cfg)
    plane_start = start.numpy()[::cfg.ny * cfg.nz].copy()
    plane_start[planes:] = plane_start[planes]           # planes beyond the sample hold no particles
    mom = oracle.Moments(cfg.nodes, with_abs=False)      # calloc-backed: only touched pages are committed
    oracle.lib()
    # planes of one colour run in parallel: at most ceil(planes / 2) threads have work
    threads = min(oracle.threads(), (planes + 1) // 2) if all_cores else 1
    t0 = time.perf_counter()
    for s, sp in enumerate(cfg.species):
        if all_cores:
            oracle.step_planes(grid_of(cfg), sp.qom, cfg.dt, parts[s], plane_start, En, Bn, mom)
        else:
            oracle.step(grid_of(cfg), sp.qom, cfg.dt, parts[s], En, Bn, mom)
    dt = time.perf_counter() - t0
    return n / dt, n, dt, threads


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    cfg = load_config(args)
    for _ in range(max(0, args.warmup)):
        oracle_sample(cfg, 1)
    rates, secs, n = [], [], 0
    for _ in range(max(1, args.steps)):
        r, n, dt, cores = oracle_sample(cfg, args.cpu_sample_planes)
        rates.append(r); secs.append(dt)
    cores = rates and cores or 1
    value = n * len(secs) / sum(secs)
    sample = (f"particles of the first {min(args.cpu_sample_planes, cfg.nx)} x-planes of cells "
              f"({n} particles, all species) on the full {cfg.nx}x{cfg.ny}x{cfg.nz} grid, one oracle step per bench step")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "note": "CPU oracle (oracle/ecsim_oracle.c, gcc -O2 -ffp-contract=off), "
                   "all host cores of this box (x-planes of cells in two colours); ms_per_step is per sample, not per full workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "host_cores": os.cpu_count(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def run_product(args):
    import torch
    import paper_2603_16624_b200 as pk
    import workloads as wl
    from workloads import PKEYS, grid_of

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libecpush has no CPU fallback")
    if local == 0:
        from paper_2603_16624_b200 import build as product_build
        product_build.build()                     # in-tree, only if missing or stale; other ranks wait at the barrier below
    torch.cuda.set_device(local % torch.cuda.device_count())
    sampler = ClockSampler(local % torch.cuda.device_count())
    sampler.start()
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
        dist.barrier()
    cfg = load_config(args)
    dev = torch.device("cuda")
    nsp = len(cfg.species)

    # ---- synthetic inputs, resident in HBM (every rank: an independent replica of the workload) ----
    E, B = wl.gen_fields(cfg, device=dev)
    pristine = []
    for s in range(nsp):
        p = wl.gen_species(cfg, s, device=dev)
        pristine.append({k: p[k].contiguous() for k in PKEYS})
        del p
    torch.cuda.empty_cache()
    n_s = [int(p["x"].numel()) for p in pristine]
    n_total = sum(n_s)
    work = [{k: torch.empty_like(p[k]) for k in PKEYS} for p in pristine]
    for s in range(nsp):
        work[s]["q"].copy_(pristine[s]["q"])

    ctx = pk.Ecsim(*grid_of(cfg), nsp)
    ctx.set_workspace(max(n_s))
    ctx.set_variant(pk.VARIANT_FUSED if args.variant == "fused" else pk.VARIANT_ATOMIC)
    if args.fused_warps > 0:
        ctx.set_fused_warps(args.fused_warps)
    ctx.enable_timing(True)
    rho = torch.empty(nsp, cfg.nodes, dtype=torch.float64, device=dev)
    J = torch.empty(nsp, 3, cfg.nodes, dtype=torch.float64, device=dev)
    ctx.set_m_layout(pk.M_14 if args.m_layout == 14 else pk.M_27)
    M = torch.empty(cfg.nodes, args.m_layout, 3, 3, dtype=torch.float64, device=dev)
    sorted_input = not cfg.shuffled

    def restore_arrays():
        for s in range(nsp):
            for k in ("x", "y", "z", "u", "v", "w") + (("q",) if cfg.shuffled else ()):
                work[s][k].copy_(pristine[s][k])
            ctx.load_particles(s, cfg.species[s].qom, work[s], sorted=sorted_input)

    def restore():
        restore_arrays()
        if sorted_input:
            for s in range(nsp):
                ctx.build_segments(s)        # set-up of the sorted state, not part of the step ("step_with_segments_ms" has it inside)

    def one_step():
        ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)

    fp64_probe, _ = ctx.probe_fp64(4096)

    # clock samples: nvidia-smi needs a few tenths of a second for its first line, so it was started with the process; the
    # samples kept are those stamped between the first warm-up step (same load as the timed ones) and the last timed step
    t_clock0 = time.time()
    for _ in range(max(3, args.warmup)):
        restore()
        one_step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kernel_ms = []
    launches0 = ctx.launch_count()
    launches_step = 0
    torch.cuda.synchronize()
    for i in range(args.steps):
        restore()
        torch.cuda.synchronize()
        l0 = ctx.launch_count()
        ev[i][0].record()
        one_step()
        ev[i][1].record()
        launches_step += ctx.launch_count() - l0
        torch.cuda.synchronize()
        kernel_ms.append(ctx.kernel_ms())
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop(t_clock0, time.time())
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = max_over_ranks([sum(step_ms)], world)[0]
    ms_per_step = total_ms / args.steps
    value = world * n_total * args.steps / (total_ms * 1e-3)
    k_ms = sum(kernel_ms) / len(kernel_ms)
    achieved_tflops = FLOP_PER_PARTICLE * n_total / (k_ms * 1e-3) / 1e12

    traffic, traffic_src = (None, None)
    if args.variant == "fused" and cfg.idx == 2 and not args.scale:
        traffic, traffic_src = profiled_traffic("k_fused_push_moments<12, 168, 0, 0")
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(3, args.warmup), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {
            "workload": workload_name(cfg), "particles": n_total, "variant": args.variant, "m_slots": args.m_layout,
            "multi_gpu": "replicas only (north_star: single GPU; each rank runs the whole workload)",
            "l2": "inputs (>= 15 GB at configs[2]) exceed the 126 MB L2; no explicit flush" if n_total * 56 > 2e9
                  else "working set may fit L2 (small config): not a headline number",
            "timing": "per-step CUDA events; particle state restored from a pristine device copy between steps, "
                      "outside the timed region; outputs written inside",
        },
        "roofline": {
            "bound": "alu", "kernel": "k_fused_push_moments" if args.variant == "fused" else "k_push_moments_atomic",
            "achieved": achieved_tflops, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved_tflops / FP64_PEAK_TFLOPS,
            "traffic": traffic, "traffic_source": traffic_src,
            "peak_source": "derived: 148 SM x 64 DFMA/clk x 2 x 1.965 GHz (DESIGN.md); fp64_probe_tflops is the DFMA "
                           "micro-benchmark measured in this run",
            "fp64_probe_tflops": fp64_probe, "kernel_ms": k_ms, "flop_per_particle": FLOP_PER_PARTICLE,
            "kernel_share_of_step": k_ms / ms_per_step,
        },
        "north_star_roofline": {"particles_per_s": NORTH_STAR_ROOFLINE_PPS, "frac": value / world / NORTH_STAR_ROOFLINE_PPS,
                                "definition": "slower of 119.8 B/particle at 8 TB/s and 813 flop/particle at 37.2 TFLOP/s"},
        "gpu_launches": launches_step,
        "clocks": clocks,
    }

    # ---- what a time loop sees: the step WITH the segment-table build, and consecutive steps ----
    line["step_with_segments_ms"] = measure_with_segments(args, cfg, ctx, restore_arrays, one_step, world)
    line["rows"] = None if args.no_rows else measure_rows(args, cfg, ctx, restore, E, B, rho, J, M, world)
    headline_run = cfg.idx == 2 and not args.scale and args.variant == "fused" and args.m_layout == 27
    configs_block = {}
    if headline_run and not args.no_configs and world == 1:
        # configs[2] with the paper's 14-slot storage (L73): same particles, same kernel, half the M bytes
        ctx.set_m_layout(pk.M_14)
        ms14 = timed_steps(restore, one_step, 3, 5)
        ctx.set_m_layout(pk.M_27)
        configs_block["configs[2] m_slots=14"] = config_entry(cfg, n_total, ms14, 14)
    n_sus = args.sustained_steps if args.sustained_steps >= 0 else (cfg.steps if cfg.steps > 1 else 10)
    if n_sus > 0:
        line["sustained"] = measure_sustained(args, cfg, ctx, restore_arrays, work, E, B, rho, J, M, n_sus, n_total, world)
    else:
        line["sustained"] = None

    # ---- end to end through the host-buffer entry point (rank-local, pinned host memory) ----
    ctx.close()
    del work, M, rho, J
    torch.cuda.empty_cache()
    if not args.no_e2e:
        line["e2e"] = run_e2e(args, cfg, None, pristine, E, B, world)
    else:
        line["e2e"] = None
    del pristine
    torch.cuda.empty_cache()

    if headline_run and not args.no_configs and world == 1:
        for idx in (0, 1, 3, 4):
            configs_block.update(measure_config(idx))
        line["configs"] = configs_block
    else:
        line["configs"] = None

    if rank == 0 and not args.no_cpu_baseline and world == 1:
        v, n, dt, cores = oracle_sample(cfg, args.cpu_sample_planes)
        v1, n1, dt1, _ = oracle_sample(cfg, max(1, args.cpu_sample_planes // 8), all_cores=False)
        line["cpu_baseline"] = {
            "value": v, "unit": UNIT, "cores": cores, "host_cores": os.cpu_count(), "kind": "oracle",
            "single_thread_value": v1,
            "sample": f"particles of the first {min(args.cpu_sample_planes, cfg.nx)} x-planes of cells ({n} particles, "
                      f"all species) on the full grid; {dt:.1f} s of CPU work"}
    else:
        line["cpu_baseline"] = None
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def _median(v):
    return statistics.median(v) if v else None


def timed_steps(prepare, step, warmup, steps):
    """Median over `steps` of one call of step(), CUDA events on torch's current stream (the context's stream);
    prepare() restores the particle state before every step, outside the timed region."""
    import torch
    ms = []
    for i in range(warmup + steps):
        prepare()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); step(); e1.record()
        torch.cuda.synchronize()
        if i >= warmup:
            ms.append(e0.elapsed_time(e1))
    return _median(ms)


def config_roofline_pps(cfg, n_total, m_slots, with_sort=False):
    """SURVEY 8(d) applied to a configuration: the slower of the FP64 bound (813 flop per particle) and the HBM bound
    (104 B per particle + (48 + 32 + 72 m_slots) B per node, at the contract's 8 TB/s); a step that has to sort first
    adds 144 B per particle of HBM-bound integer work (config 4: 144 B / 8 TB/s + 21.8 ps = 39.8 ps -> 25.1 G/s)."""
    bytes_pp = 104.0 + (48.0 + 32.0 + 72.0 * m_slots) * cfg.nodes / n_total
    t = max(bytes_pp / 8.0e12, FLOP_PER_PARTICLE / (FP64_PEAK_TFLOPS * 1e12))
    if with_sort:
        t += 144.0 / 8.0e12
    return 1.0 / t


def config_entry(cfg, n_total, ms, m_slots, with_sort=False, **extra):
    pps = n_total / (ms * 1e-3)
    roof = config_roofline_pps(cfg, n_total, m_slots, with_sort)
    out = {"workload": workload_name(cfg), "particles": n_total, "m_slots": m_slots, "ms_per_step": ms,
           "particles_per_s": pps, "roofline_particles_per_s": roof, "frac": pps / roof,
           "fits_l2": bool(n_total * 56 < 126e6)}
    out.update(extra)
    return out


def measure_config(idx):
    """One of the other BASELINE.json configurations on this GPU, timed like the headline (3 warm-ups, median of 5 steps,
    particle state restored from a pristine device copy outside the timed region, segment tables built outside):
      configs[0], [3]  one fused all-species step from the cell-sorted state
      configs[1]       the same, and its protocol of 1 + 10 consecutive steps with fixed fields, dense and resident
      configs[4]       particles in random order: the counting sort of both species and the step from the sorted state are
                       timed separately and summed; `one_call_ms` is ecsim_push_and_moments_all on the
                       unsorted species (it sorts first), one timed region
    Configs 0 and 1 fit (partly) in the 126 MB L2: reported, not headline numbers."""
    import torch
    import paper_2603_16624_b200 as pk
    import workloads as wl
    from workloads import PKEYS, grid_of
    cfg = wl.config(idx)
    dev = torch.device("cuda")
    nsp = len(cfg.species)
    E, B = wl.gen_fields(cfg, device=dev)
    pristine = [{k: v.contiguous() for k, v in wl.gen_species(cfg, s, device=dev).items() if k in PKEYS} for s in range(nsp)]
    n_s = [int(p["x"].numel()) for p in pristine]
    n_total = sum(n_s)
    work = [{k: p[k].clone() for k in PKEYS} for p in pristine]
    ctx = pk.Ecsim(*grid_of(cfg), nsp)
    ctx.set_workspace(max(n_s))
    rho = torch.empty(nsp, cfg.nodes, dtype=torch.float64, device=dev)
    J = torch.empty(nsp, 3, cfg.nodes, dtype=torch.float64, device=dev)
    M = torch.empty(cfg.nodes, 27, 3, 3, dtype=torch.float64, device=dev)

    def reload(sorted_flag):
        for s in range(nsp):
            for k in PKEYS:
                work[s][k].copy_(pristine[s][k])
            ctx.load_particles(s, cfg.species[s].qom, work[s], sorted=sorted_flag)

    def restore_sorted():
        reload(not cfg.shuffled)
        for s in range(nsp):
            if cfg.shuffled:
                ctx.sort_particles(s)
            else:
                ctx.build_segments(s)

    def step():
        ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)

    def sort_all():
        for s in range(nsp):
            ctx.sort_particles(s)

    name = f"configs[{idx}]"
    out = {}
    if cfg.shuffled:
        sort_ms = timed_steps(lambda: reload(False), sort_all, 3, 5)
        push_ms = timed_steps(restore_sorted, step, 3, 5)
        one_call_ms = timed_steps(lambda: reload(False), step, 2, 5)
        out[name] = config_entry(cfg, n_total, sort_ms + push_ms, 27, with_sort=True, sort_ms=sort_ms, push_ms=push_ms,
                                 one_call_ms=one_call_ms, sort_ms_per_species=sort_ms / nsp)
    else:
        ms = timed_steps(restore_sorted, step, 3, 5)
        out[name] = config_entry(cfg, n_total, ms, 27, strays_after_step=ctx.stray_count())
    if cfg.steps > 1:
        # configs[1]: one step, then cfg.steps - 1 more with the fields held fixed, state never restored
        for kind in ("dense", "resident"):
            restore_sorted()
            if kind == "resident":
                for s in range(nsp):
                    ctx.make_resident(s, 0.5)
            torch.cuda.synchronize()
            r0, l0 = ctx.resort_count(), ctx.relayout_count()
            ms, strays = [], []
            for _ in range(cfg.steps):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); step(); e1.record()
                torch.cuda.synchronize()
                ms.append(e0.elapsed_time(e1))
                strays.append(ctx.stray_count())
            tot = sum(ms)
            out[name][f"protocol_{kind}"] = {
                "steps": cfg.steps, "ms_per_step": tot / cfg.steps, "ms_each": [round(v, 3) for v in ms],
                "particles_per_s": n_total * cfg.steps / (tot * 1e-3),
                "frac": n_total * cfg.steps / (tot * 1e-3) / config_roofline_pps(cfg, n_total, 27),
                "strays_per_step": strays, "resorts": ctx.resort_count() - r0, "relayouts": ctx.relayout_count() - l0,
                **({"slack": 0.5} if kind == "resident" else {})}
    ctx.close()
    del work, pristine, M, rho, J, E, B
    torch.cuda.empty_cache()
    return out


def measure_with_segments(args, cfg, ctx, restore_arrays, one_step, world):
    """The headline step with the per-species segment tables (histogram + scan of cell-sorted arrays) built INSIDE the
    timed region: what the first step after a load costs."""
    import torch
    ms = []
    for _ in range(3):
        restore_arrays()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); one_step(); e1.record()
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    return max_over_ranks([_median(ms)], world)[0]


def measure_rows(args, cfg, ctx, restore, E, B, rho, J, M, world):
    """The other entry points of SURVEY 8(f) on the same workload, from the sorted state, CUDA events, median of 3:
    the two halves of a real time step (ecsim_moments_all, ecsim_push_all), the operator sum M E (ecsim_apply_M; HBM-bound:
    its GB/s count M read once + E + out) and the diagnostic moments of species 0 (ecsim_diagnostics)."""
    import torch
    import paper_2603_16624_b200 as pk
    dev = E.device
    nodes = cfg.nodes

    def timed(fn, prepare=None):
        ms = []
        for _ in range(3):
            if prepare:
                prepare()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        return max_over_ranks([_median(ms)], world)[0]

    def restore_sorted():
        restore()
        if cfg.shuffled:                       # configs[4]: the sort is part of its step, not of these rows
            for s in range(len(cfg.species)):
                ctx.sort_particles(s)

    out = {}
    restore_sorted()
    out["moments_all_ms"] = timed(lambda: ctx.moments_all(B, cfg.dt, rho, J, M, accumulate=pk.ACC_NONE))
    out["push_all_ms"] = timed(lambda: ctx.push_all(E, B, cfg.dt, cfg.theta), prepare=restore_sorted)
    restore_sorted()
    ctx.moments_all(B, cfg.dt, rho, J, M, accumulate=pk.ACC_NONE)
    ME = torch.empty(3, nodes, dtype=torch.float64, device=dev)
    t = timed(lambda: ctx.apply_M(M, E, ME))
    out["apply_M_ms"] = t
    out["apply_M_GBps"] = (M.numel() + 6 * nodes) * 8 / (t * 1e-3) / 1e9
    d_rho = torch.empty(nodes, dtype=torch.float64, device=dev)
    d_J = torch.empty(3, nodes, dtype=torch.float64, device=dev)
    d_P = torch.empty(6, nodes, dtype=torch.float64, device=dev)
    d_Q = torch.empty(3, nodes, dtype=torch.float64, device=dev)
    out["diagnostics_species0_ms"] = timed(lambda: ctx.diagnostics(0, d_rho, d_J, d_P, d_Q))
    return out


def measure_sustained(args, cfg, ctx, restore_arrays, work, E, B, rho, J, M, n_steps, n_total, world):
    """n_steps CONSECUTIVE steps, fields fixed, particle state never restored (configs[1]'s protocol; 10 steps of the
    headline workload by default): every stray, re-sort and fresh layout is inside the timed steps.
      dense:    the caller's arrays pushed in place (ecsim_push_and_moments_all): leavers become strays, re-sorts by rent-or-buy
      resident: library-managed gapped double buffers (ecsim_make_resident): the sort-preserving push, no strays.
      resident_split: the same species stepped as a real ECsim time step does: ecsim_moments_all, [the field
                solve would run here], ecsim_push_all -- two passes over the particles instead of one."""
    import torch
    import paper_2603_16624_b200 as pk
    nsp = len(cfg.species)
    out = {}
    for kind in ("dense", "resident", "resident_split"):
        restore_arrays()
        if kind != "dense":
            torch.cuda.synchronize()
            torch.cuda.empty_cache()              # the gapped buffers of the previous kind go back to the driver
            free, _ = torch.cuda.mem_get_info()
            need = sum(ctx.resident_bytes(int(work[s]["x"].numel()), 0.5) for s in range(nsp))
            if need > free - (2 << 30):
                out[kind] = {"skipped": f"needs {need / 1e9:.1f} GB of device memory, {free / 1e9:.1f} GB free"}
                continue
            for s in range(nsp):
                ctx.make_resident(s, 0.5)
        torch.cuda.synchronize()
        lent = [ctx.resident_bytes(int(work[s]["x"].numel()), 0.5) for s in range(nsp)] if kind != "dense" else None
        r0, l0 = ctx.resort_count(), ctx.relayout_count()
        ms, strays, leavers = [], [], []
        for _ in range(n_steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            if kind == "resident_split":
                ctx.moments_all(B, cfg.dt, rho, J, M, accumulate=pk.ACC_NONE)
                ctx.push_all(E, B, cfg.dt, cfg.theta)
            else:
                ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M, accumulate=pk.ACC_NONE)
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
            strays.append(ctx.stray_count())
            leavers.append(ctx.leaver_count())
        tot = max_over_ranks([sum(ms)], world)[0]
        out[kind] = {"steps": n_steps, "ms_per_step": tot / n_steps, "ms_first": ms[0], "ms_each": [round(v, 3) for v in ms],
                     "ms_median_after_first": _median(ms[1:]) if len(ms) > 1 else None,
                     "particles_per_s": world * n_total * n_steps / (tot * 1e-3),
                     "north_star_frac": n_total * n_steps / (tot * 1e-3) / NORTH_STAR_ROOFLINE_PPS,
                     "strays_per_step": strays, "leavers_per_step": leavers,
                     "resorts": ctx.resort_count() - r0, "relayouts": ctx.relayout_count() - l0}
        if lent is not None:
            out[kind]["slack"] = 0.5
            out[kind]["lent_bytes_per_species"] = lent      # the gapped double buffers + tables the caller lends (ecsim_resident_bytes)
    return out


def run_e2e(args, cfg, ctx_unused, pristine, E, B, world):
    """Same metric through ecsim_push_and_moments_host_all: pinned host buffers in, host buffers out, the
    host<->device copies inside the timed region."""
    import torch
    import paper_2603_16624_b200 as pk
    from workloads import PKEYS, grid_of
    nsp = len(cfg.species)
    n_s = [int(p["x"].numel()) for p in pristine]
    host = [{k: torch.empty(n_s[s], dtype=torch.float64).pin_memory() for k in PKEYS} for s in range(nsp)]
    Eh, Bh = E.cpu().pin_memory(), B.cpu().pin_memory()
    rho = torch.empty(nsp, cfg.nodes, dtype=torch.float64).pin_memory()
    J = torch.empty(nsp, 3, cfg.nodes, dtype=torch.float64).pin_memory()
    M = torch.empty(cfg.nodes, args.m_layout, 3, 3, dtype=torch.float64).pin_memory()
    ctx = pk.Ecsim(*grid_of(cfg), nsp)
    ctx.set_workspace_host_all(max(n_s), sum(n_s))
    ctx.set_m_layout(pk.M_14 if args.m_layout == 14 else pk.M_27)
    if args.variant == "atomic":
        ctx.set_variant(pk.VARIANT_ATOMIC)
    qoms = [sp.qom for sp in cfg.species]

    def refill():
        for s in range(nsp):
            for k in PKEYS:
                host[s][k].copy_(pristine[s][k])
        torch.cuda.synchronize()

    def step():
        ctx.push_and_moments_host_all(qoms, not cfg.shuffled, host, Eh, Bh, cfg.dt, cfg.theta, rho, J, M,
                                      accumulate=pk.ACC_NONE)

    refill(); step()                                   # warm-up
    times = []
    for _ in range(max(1, args.e2e_steps)):
        refill()
        t0 = time.perf_counter()
        step()                                         # the host call ends with a stream synchronise
        times.append(time.perf_counter() - t0)
    ctx.close()
    t = max_over_ranks([sum(times)], world)[0]
    n_total = sum(n_s)
    nodes = cfg.nodes
    h2d = sum(7 * 8 * n for n in n_s) + 6 * 8 * nodes
    d2h = sum(6 * 8 * n for n in n_s) + (9 * args.m_layout + 4 * nsp) * 8 * nodes
    return {"value": world * n_total * len(times) / t, "unit": UNIT, "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": d2h, "steps": len(times),
            "api": "ecsim_push_and_moments_host_all (all species in one call), pinned host memory, copies inside the timed region"}


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_product(args)


if __name__ == "__main__":
    main()
