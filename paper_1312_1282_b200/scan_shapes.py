"""Shape scan: time qmc_sweep for every compiled kernel shape that fits a workload, next to the planner's own choice.

    python -m paper_1312_1282_b200.scan_shapes --config 3 [--mode fp64|fp32c] [--sweeps 2] [--tiles 1,2,4] [--clusters 1]
    python -m paper_1312_1282_b200.scan_shapes --atoms 40960 --walkers 1 --mode fp32c --clusters 4,8

The constants of the launch heuristic (csrc/qmc_sweep_plan.cu) were fitted to the output of this tool on a B200
(profiles/r02_shapes.md); run it again on other hardware.  Shapes are forced through qmc_set_tuning, timed with CUDA
events after a few warm-up sweeps, best of three.
"""
from __future__ import annotations

import argparse
import itertools

from . import binding, workloads as wl


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=0, help="BASELINE.json config 1..5 (or use --atoms/--walkers)")
    ap.add_argument("--atoms", type=int, default=0)
    ap.add_argument("--walkers", type=int, default=1)
    ap.add_argument("--mode", choices=["fp32c", "fp64", "default"], default="default")
    ap.add_argument("--sweeps", type=int, default=2)
    ap.add_argument("--tiles", default="1,2,4")
    ap.add_argument("--clusters", default="1")
    args = ap.parse_args()
    import torch

    if args.config:
        w = wl.config(args.config)
        if args.mode != "default":
            w = wl.with_mode(w, wl.MODE_FP64 if args.mode == "fp64" else wl.MODE_FP32C)
    else:
        mode = wl.MODE_FP64 if args.mode == "fp64" else wl.MODE_FP32C
        w = wl.Workload(f"N{args.atoms}", args.atoms, (wl.Group(wl.RHO_EQ, 2.89, args.walkers, 1.0),), 1, mode)
    binding.load_library()
    N = w.n_atoms
    tiles = [int(t) for t in args.tiles.split(",")] if w.mode == wl.MODE_FP32C else [1]
    clusters = [int(c) for c in args.clusters.split(",")]
    label = f"{w.name} {'fp64' if w.mode == wl.MODE_FP64 else 'fp32c'} W={w.n_walkers}"

    def make():
        return binding.QMC(N, w.walkers_per_group, w.box_L, w.jastrow_b, w.hbar2_over_2m, w.aziz, w.mode, jitter=wl.JITTER)

    def timed(q):
        q.init_walkers(w.seed)
        q.sweep(3, w.steps)
        torch.cuda.synchronize()
        best = 1e9
        for _ in range(3):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            q.sweep(args.sweeps, w.steps)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1) / args.sweeps)
        return best

    results = []
    for C, T, J, K in itertools.product(clusters, (32, 64, 128, 256, 512, 1024), (1, 2, 4, 6, 8, 10, 12, 16, 20, 32), tiles):
        per_block = (N + C - 1) // C
        if T * J < per_block or T * J > 1.4 * per_block + 128 or (C > 1 and K > 1):
            continue
        binding.set_tuning()
        for key, val in (("sweep_cluster", C), ("sweep_threads", T), ("sweep_per_thread", J), ("sweep_tile", K)):
            binding.set_tuning(key, val)
        try:
            q = make()
        except binding.QmcError:
            continue
        inf = q.info()
        if (inf["sweep_cluster"], inf["sweep_threads"], inf["sweep_pairs_per_thread"], inf["sweep_tile"]) != (C, T, J, K):
            q.close()
            continue
        ms = timed(q)
        print(f"{label} cluster={C} T={T} J={J} V={inf['sweep_vector']} P={inf['sweep_pending']} K={K} "
              f"ctas/sm={inf['sweep_ctas_per_sm']} smem={inf['sweep_smem_bytes']}  {ms:.4f} ms/sweep  acc={float(q.acceptance().mean()):.3f}", flush=True)
        results.append((ms, C, T, J, K))
        q.close()
    binding.set_tuning()
    q = make()
    inf = q.info()
    ms = timed(q)
    print(f"{label} PLANNER: cluster={inf['sweep_cluster']} T={inf['sweep_threads']} J={inf['sweep_pairs_per_thread']} V={inf['sweep_vector']} "
          f"K={inf['sweep_tile']} ctas/sm={inf['sweep_ctas_per_sm']}  {ms:.4f} ms/sweep; best forced: "
          + ", ".join(f"{m:.4f} (C={c} T={t} J={j} K={k})" for m, c, t, j, k in sorted(results)[:3]))


if __name__ == "__main__":
    main()
