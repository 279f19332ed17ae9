"""Consecutive steps on the state the previous step left (no restore): what a time loop with fixed fields sees,
including strays and re-sorts.  Usage example of the binding and the source of profiles/r01d.

    python -m paper_2603_16624_b200.multistep [config index, default 2] [steps, default 14]
"""
from __future__ import annotations

import os
import sys

import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_2603_16624_b200 as pk  # noqa: E402
import workloads as wl  # noqa: E402

PKEYS = ("x", "y", "z", "u", "v", "w", "q")


def main():
    idx = int(sys.argv[1]) if len(sys.argv) > 1 else 2
    steps = int(sys.argv[2]) if len(sys.argv) > 2 else 14
    cfg = wl.config(idx)
    dev = torch.device("cuda")
    nsp = len(cfg.species)
    E, B = wl.gen_fields(cfg, device=dev)
    parts = []
    for s in range(nsp):
        p = wl.gen_species(cfg, s, device=dev)
        parts.append({k: p[k].contiguous() for k in PKEYS})
        del p
    ctx = pk.Ecsim(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, nsp)
    ctx.set_workspace(max(int(p["x"].numel()) for p in parts))
    for s, sp in enumerate(cfg.species):
        ctx.load_particles(s, sp.qom, parts[s], sorted=not cfg.shuffled)
    rho = torch.empty(nsp, cfg.nodes, dtype=torch.float64, device=dev)
    J = torch.empty(nsp, 3, cfg.nodes, dtype=torch.float64, device=dev)
    M = torch.empty(cfg.nodes, 27, 3, 3, dtype=torch.float64, device=dev)
    n = sum(int(p["x"].numel()) for p in parts)
    for step in range(steps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.push_and_moments_all(E, B, cfg.dt, cfg.theta, rho, J, M)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        print(f"step {step:2d}: {ms:8.3f} ms  {n / ms / 1e6:6.2f} G particles/s  strays {ctx.stray_count():9d}  "
              f"re-sorts so far {ctx.resort_count()}")
    ctx.close()


if __name__ == "__main__":
    main()
