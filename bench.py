#!/usr/bin/env python
"""bench.py -- throughput of the He-4 VMC hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--mode fp32c|fp64]
                    [--sweeps-per-step m] [--impl ours|reference] [--no-cpu-baseline]

One STEP = the whole hot path over all walkers of the workload: m Metropolis sweeps (default 1)
+ one local-energy evaluation + the acceptance read-out.
Default workload: BASELINE.json configs[2] = N = 1952 atoms, 2048 walkers, fp32 coordinates with
fp64 sums, the configuration the metric is quoted on.  Prints ONE JSON line (see DESIGN.md
"Measurement" for every key).  --impl reference times the CPU oracle on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1312_1282_b200 import workloads as wl  # noqa: E402

# Algorithmic FP instructions per u-evaluation of the sweep: thread-level
# instructions on the pipe that bounds the mode, for ONE trial-position pair evaluation.  The counts are
# checked against ncu's sm__sass_thread_inst_executed_op_* per executed pair evaluation in profiles/r02_instr.md.
ALG_INSTR = {wl.MODE_FP32C: 24.0, wl.MODE_FP64: 31.0}
LANES_PER_SM = {wl.MODE_FP32C: 128, wl.MODE_FP64: 64}
# SURVEY.md section 8(d)'s own estimate of the same count for the FP32C pair term (a second reading of "algorithmic")
SURVEY_INSTR_FP32C = 28.0
# DRAM bytes per launch of the dominant kernel (dram__bytes_read.sum + dram__bytes_write.sum).  These are NOT measured
# by this run: they are typed in from the ncu --set full capture of this command that profiles/r02b_kernels.md
# summarises (round-2 sweep kernels, unchanged since; 2048 walkers of 1952 atoms).  None where no capture exists.
# `traffic_compulsory` in the JSON line is computed from W, N and the mode instead.
NCU_TRAFFIC_BYTES = {("c3-N1952", wl.MODE_FP32C): 80.0e6 + 22.4e6, ("c3-N1952-fp64", wl.MODE_FP64): 129.7e6 + 70.4e6}
NCU_TRAFFIC_SOURCE = "profiles/r02b_kernels.md (ncu --set full of this command, round-2 kernels; a constant, not measured by this run)"
# Issue slots per EXECUTED pair evaluation of the FP32C sweep on each pipe, in thread terms (warp instructions x 32 /
# executed pair evaluations), and ncu's pipe utilisation of the same launch: profiles/r02b_instr.md and
# profiles/r02b_kernels.md (sweep_kernel<float, 128, 16, 4, 1, 0>, 2048 x 1952, acceptance 0.523).  Constants from
# those files, quoted so that the pipe bound below can be recomputed by a reader.
NCU_SWEEP32_SLOTS = {"issue": 19.36, "fma": 6.23, "alu": 7.89, "xu": 2.26, "fp64": 0.55, "lsu": 2.03}
NCU_SWEEP32_UTIL_PCT = {"pipe_fma": 37.7, "pipe_xu": 57.8, "pipe_alu": 51.4, "issue_active": 61.9}
# thread-level instructions per SM and clock each pipe can take (guide: 4 schedulers x 1 warp instruction per clock;
# FMA 128 lanes, of which a packed FFMA2 holds its lane for two clocks -- profiles/r01_pipes.md; ALU 64; XU 16; FP64 64)
PIPE_LANES = {"issue": 128.0, "fma": 128.0, "alu": 64.0, "xu": 16.0, "fp64": 64.0, "lsu": 32.0}
EQUIL_SWEEPS = {1: 200, 2: 200, 3: 150, 4: 20, 5: 60}      # untimed, before the warm-up (time the liquid, not the melting lattice)


def pair_counts(w: wl.Workload, m: int):
    """(sweep pair evaluations, energy pairs) per step over all walkers: N(N-1) per walker-sweep
    (one trial evaluation per (moved, other) pair) and N(N-1)/2 per energy evaluation."""
    N, W = w.n_atoms, w.n_walkers
    return W * m * N * (N - 1), W * N * (N - 1) // 2


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (nvidia-smi, 5 Hz)."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()

    def run(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        while not self._stop_evt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                self.samples.append(float(f[0]))
                self.max_mhz = float(f[1])
                for n, v in zip(names, f[2:6]):
                    if v.lower().startswith("active"):
                        self.reasons.add(n)
            except Exception:
                pass
            self._stop_evt.wait(0.2)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=10)
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def cpu_baseline(w: wl.Workload, m: int, budget_s: float = 12.0):
    """The oracle as it stands on the host cores: one OS thread per walker, `cores` walkers of the
    same workload (same seed, so a subset of the GPU run's chains), whole steps until ~budget_s."""
    import oracle
    cores = oracle.num_threads()
    N, g = w.n_atoms, w.groups[0]
    s = oracle.System(N, w.box_L[0], g.b, w.hbar2_over_2m, w.aziz)
    x = oracle.init_walkers(s, w.seed, 0, cores, wl.JITTER)
    oracle.sweep(s, x[:1].copy(), w.seed, 0, 0, 0, g.step)          # load/compile outside the timing
    steps, t0, t = 0, time.perf_counter(), 0
    while True:
        oracle.sweep(s, x, w.seed, 0, t, m, g.step)
        oracle.local_energy(s, x)
        t += m
        steps += 1
        el = time.perf_counter() - t0
        if el >= budget_s or steps >= 50:
            break
    pairs = steps * cores * (m * N * (N - 1) + N * (N - 1) // 2)
    # ONE core, as the paper's CPU column is ("a single-core CPU execution"): a single walker, which
    # the oracle runs on one thread (it parallelises over walkers only)
    x1 = x[:1].copy()
    n1, t1 = 0, time.perf_counter()
    while True:
        oracle.sweep(s, x1, w.seed, 0, t, m, g.step)
        oracle.local_energy(s, x1)
        t += m
        n1 += 1
        el1 = time.perf_counter() - t1
        if el1 >= min(3.0, budget_s / 4) or n1 >= 20:
            break
    pairs_step_walker = m * N * (N - 1) + N * (N - 1) // 2
    single = n1 * pairs_step_walker / el1
    full_pairs = w.n_walkers * w.sweeps * (N * (N - 1) + N * (N - 1) // 2)       # BASELINE.json: energy every sweep
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as fh:
            for ln in fh:
                if ln.startswith("model name"):
                    model = ln.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return {"value": pairs / el, "unit": "pair-evals/s", "cores": cores, "kind": "oracle",
            "sample": f"{cores} walkers x {steps} steps (m={m} sweeps + 1 energy) of {w.name}, fp64, {el:.1f} s wall",
            "walker_sweeps_per_s": steps * cores * m / el, "ms_per_step_sample": 1e3 * el / steps,
            "cpu_model": model,
            "single_core_pair_evals_per_s": single,
            "single_core_sample": f"1 walker x {n1} steps on one thread, {el1:.1f} s wall",
            "full_config_seconds_extrapolated": {"all_cores": full_pairs / (pairs / el), "single_core": full_pairs / single,
                                                 "of": f"{w.n_walkers} walkers x {w.sweeps} sweeps, energy every sweep"}}


def run_reference(args, w, m):
    """--impl reference: the reference arm for this tier is the CPU oracle (no reference code exists)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cores = oracle.num_threads()
    N, g = w.n_atoms, w.groups[0]
    s = oracle.System(N, w.box_L[0], g.b, w.hbar2_over_2m, w.aziz)
    x = oracle.init_walkers(s, w.seed, 0, cores, wl.JITTER)
    t = 0
    for _ in range(args.warmup):
        oracle.sweep(s, x, w.seed, 0, t, m, g.step)
        oracle.local_energy(s, x)
        t += m
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.sweep(s, x, w.seed, 0, t, m, g.step)
        oracle.local_energy(s, x)
        t += m
    el = time.perf_counter() - t0
    pairs = args.steps * cores * (m * N * (N - 1) + N * (N - 1) // 2)
    val = pairs / el
    sample = f"each step = {cores} walkers (one per core) of {w.name}: m={m} sweeps + 1 energy, fp64 oracle"
    print(json.dumps({
        "impl": "reference", "metric": "pair evaluations/s (sweep N(N-1) + energy N(N-1)/2 per walker-step)",
        "value": val, "unit": "pair-evals/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "walkers_per_step": cores, "sweeps_per_step": m, "mode": "oracle-fp64"},
        "cpu_baseline": {"value": val, "unit": "pair-evals/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "pair-evals/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "walker_sweeps_per_s": args.steps * cores * m / el,
    }))


def spawn_ranks(n: int):
    """`python bench.py --gpus N` without a launcher: start N ranks (one per GPU) under torch.distributed.run and
    replace this process by it (VERDICT r1 missing #4).  NCCL_DEBUG stays whatever the caller set."""
    import socket
    sock = socket.socket()
    sock.bind(("127.0.0.1", 0))
    port = sock.getsockname()[1]
    sock.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def plumbing_only(args):
    """--plumbing-only: the rank plumbing without any GPU work (CPU test of the launch path): every rank joins a gloo
    group, the ranks count themselves, rank 0 prints the line's n_gpus."""
    import torch
    import torch.distributed as dist
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
        t = torch.ones(1)
        dist.all_reduce(t)
        assert int(t.item()) == world
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps({"plumbing_only": True, "n_gpus": world, "requested_gpus": args.gpus}))


class Timed:
    """One workload on this rank's GPU: context, equilibration, warm-up, K timed steps (sweep | energy + acceptance)."""

    def __init__(self, w, m, dev, rank, proposal=0, sigma=0.8):
        import torch
        from paper_1312_1282_b200 import binding
        self.torch, self.w, self.m, self.dev = torch, w, m, dev
        W = w.n_walkers
        self.q = binding.QMC(w.n_atoms, w.walkers_per_group, w.box_L, w.jastrow_b, w.hbar2_over_2m, w.aziz, w.mode,
                             walker_id_base=rank * W, jitter=wl.JITTER, device=str(dev))
        self.q.init_walkers(w.seed)
        self.steps = w.steps
        if proposal == 1:
            self.q.set_proposal(1)
            self.steps = [sigma] * len(w.groups)
        self.e_out = torch.empty((W, 4), dtype=torch.float64, device=dev)
        self.a_out = torch.empty((W,), dtype=torch.float64, device=dev)

    def one_step(self):
        self.q.sweep(self.m, self.steps)
        self.q.local_energy(self.e_out)
        self.q.acceptance(self.a_out)

    def run(self, equil, warmup, K, flush, barrier=None, sampler=None):
        torch, q = self.torch, self.q
        if equil > 0:
            q.sweep(equil, self.steps)                     # untimed: melt the lattice
        for _ in range(warmup):
            self.one_step()
        torch.cuda.synchronize()
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
        if barrier:
            barrier()
        torch.cuda.synchronize()
        if sampler:
            sampler.start()
        launches0 = q.info()["kernel_launches"]
        for k in range(K):
            flush.zero_()                                   # L2 flush between timed iterations (untimed)
            ev[k][0].record()
            q.sweep(self.m, self.steps)
            ev[k][1].record()
            q.local_energy(self.e_out)
            q.acceptance(self.a_out)
            ev[k][2].record()
        torch.cuda.synchronize()
        self.launches = q.info()["kernel_launches"] - launches0
        if barrier:
            barrier()
        self.sweep_ms = [ev[k][0].elapsed_time(ev[k][1]) for k in range(K)]
        self.step_ms = [ev[k][0].elapsed_time(ev[k][2]) for k in range(K)]
        self.t_sweep = sum(self.sweep_ms) * 1e-3
        self.t_total = sum(self.step_ms) * 1e-3
        self.acc = float(self.a_out.mean())
        self.e_mean = (self.e_out.mean(0) / self.w.n_atoms).tolist()
        return self


def summarize(t: "Timed", K, sm_count, sm_max_mhz, world=1):
    """Throughput and roofline keys of one timed workload (shared by the headline and the `configs` block)."""
    w, m = t.w, t.m
    sweep_pairs, energy_pairs = pair_counts(w, m)
    peak = sm_count * LANES_PER_SM[w.mode] * sm_max_mhz * 1e6
    t_launch = t.t_sweep / K
    achieved = sweep_pairs * ALG_INSTR[w.mode] / t_launch
    info = t.q.info()
    return {
        "workload": w.name, "N": w.n_atoms, "walkers": w.n_walkers, "groups": len(w.groups),
        "mode": "fp32c" if w.mode == wl.MODE_FP32C else "fp64", "steps": K,
        "ms_per_step": 1e3 * t.t_total / K, "sweep_ms": 1e3 * t.t_sweep / K, "energy_ms": 1e3 * (t.t_total - t.t_sweep) / K,
        "ms_per_step_median": statistics.median(t.step_ms), "sweep_ms_median": statistics.median(t.sweep_ms),
        "pair_evals_per_s": world * K * (sweep_pairs + energy_pairs) / t.t_total,
        "sweep_pair_evals_per_s": world * K * sweep_pairs / t.t_sweep,
        "energy_pairs_per_s": world * K * energy_pairs / (t.t_total - t.t_sweep),
        "walker_sweeps_per_s": world * K * w.n_walkers * m / t.t_total,
        "sweep_roofline_frac": achieved / peak, "sweep_roofline_executed_frac": achieved * (1.0 + t.acc) / peak,
        "acceptance": t.acc, "energy_per_atom_K": dict(zip(["E_PB", "V", "T_PB", "T_JF"], t.e_mean)),
        "sweep_shape": {k: info[k] for k in ("sweep_threads", "sweep_pairs_per_thread", "sweep_vector", "sweep_pending",
                                              "sweep_tile", "sweep_ctas_per_sm")},
        "energy_shape": {k: info[k] for k in ("energy_threads", "energy_variant", "energy_ctas_per_sm")},
    }


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--mode", choices=["fp32c", "fp64", "default"], default="default")
    ap.add_argument("--sweeps-per-step", type=int, default=1)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="skip the `configs` block (the other BASELINE.json configs)")
    ap.add_argument("--equil", type=int, default=None, help="untimed equilibration sweeps before the warm-up (default per config)")
    ap.add_argument("--walkers", type=int, default=None, help="truncate walkers per group (debugging)")
    ap.add_argument("--proposal", type=int, choices=[0, 1], default=0,
                    help="0: particles in order, uniform cube (BASELINE.json); 1: the paper's random particle + "
                         "Gaussian displacement (NEXT-1), standard deviation --sigma per component")
    ap.add_argument("--sigma", type=float, default=0.8, help="proposal 1: standard deviation per component, Angstrom")
    ap.add_argument("--time-to-error", type=int, default=None, metavar="S",
                    help="after the timed steps: S more steps with the energy recorded, reblocked -> the paper's "
                         "t*sigma^2 and seconds to 1 mK per atom (PAPER.md l.504-511); 0 = skip; default 40 for the "
                         "headline config on one GPU (under a second), else 0")
    ap.add_argument("--large-n", action="store_true", help="add the NEXT-3 cluster-kernel figures (N = 40960, one walker on 8 SMs)")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="qmc_set_tuning override for the headline workload, e.g. --tune sweep_tile=4 (tuning experiments; "
                         "the defaults are the product)")
    ap.add_argument("--plumbing-only", action="store_true", help="rank plumbing only, no GPU work (CPU test of --gpus N)")
    args = ap.parse_args()

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        spawn_ranks(args.gpus)                               # does not return
    if args.plumbing_only:
        return plumbing_only(args)

    w = wl.config(args.config)
    if args.mode != "default":
        w = wl.with_mode(w, wl.MODE_FP64 if args.mode == "fp64" else wl.MODE_FP32C)
    if args.walkers:
        w = w.truncated(args.walkers)
    m = args.sweeps_per_step
    if args.impl == "reference":
        if args.steps is None:
            args.steps = 5
        return run_reference(args, w, m)
    if args.steps is None:
        args.steps = 20

    import torch
    import torch.distributed as dist
    from paper_1312_1282_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")

    # weak scaling: every rank runs the workload's W walkers; global walker ids continue across ranks
    W, N = w.n_walkers, w.n_atoms
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)   # 256 MiB > 126 MB L2
    K = args.steps
    sampler = ClockSampler(local) if rank == 0 else None
    equil = EQUIL_SWEEPS[args.config] if args.equil is None else args.equil
    for kv in args.tune:
        key, val = kv.split("=")
        binding.set_tuning(key, int(val))
    head = Timed(w, m, dev, rank, args.proposal, args.sigma)
    binding.set_tuning()
    head.run(equil, args.warmup, K, flush, barrier=dist.barrier if world > 1 else None, sampler=sampler)
    clocks = sampler.stop() if sampler else None
    q, steps = head.q, head.steps
    t_sweep, t_total = head.t_sweep, head.t_total
    if world > 1:
        tt = torch.tensor([t_total, t_sweep], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_total, t_sweep = float(tt[0]), float(tt[1])
        head.t_total, head.t_sweep = t_total, t_sweep
    acc, e_mean, launches = head.acc, head.e_mean, head.launches

    # ---- end to end through the host-buffer call (rank-local, same walkers): coordinates and pair sums travel
    # host -> device -> host every step; the copies overlap the compute chunk by chunk inside qmc_step_host ----
    h_x = q.get_positions().cpu().pin_memory()
    h_S = torch.empty((W, N), dtype=torch.float64).pin_memory()
    h_e = torch.empty((W, 4), dtype=torch.float64).pin_memory()
    h_a = torch.empty((W,), dtype=torch.float64).pin_memory()
    Ke = max(3, min(K, 10))
    q.step_host(m, steps, h_x, h_e, h_a, h_x, h_S_out=h_S)                      # warm-up; the first S_i come back
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        q.step_host(m, steps, h_x, h_e, h_a, h_x, h_S_in=h_S, h_S_out=h_S)      # state in, energies + state out
    t_e2e = time.perf_counter() - t0
    t0 = time.perf_counter()
    for _ in range(3):
        q.step_host(m, steps, h_x, h_e, h_a, h_x)                                 # coordinates only: S_i rebuilt on the device
    t_e2e_xyz = (time.perf_counter() - t0) / 3
    if world > 1:
        tt = torch.tensor([t_e2e], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_e2e = float(tt[0])

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    sweep_pairs, energy_pairs = pair_counts(w, m)
    pairs_step = sweep_pairs + energy_pairs
    value = world * K * pairs_step / t_total
    info = q.info()
    mode_name = "fp32c" if w.mode == wl.MODE_FP32C else "fp64"

    # ---- roofline of the dominant kernel (the sweep): plain-ALU bound ---------------------------
    peak_meas = binding.pipe_peak(0 if w.mode == wl.MODE_FP64 else 1)
    # live instruction rates of the other pipes the pair loop leans on (thread-level instr/s)
    rates = {"ffma2": binding.pipe_peak(2), "mufu_rsq": binding.pipe_peak(3), "i2f": binding.pipe_peak(4),
             "f2f": binding.pipe_peak(5)}
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    peak_derived = info["sm_count"] * LANES_PER_SM[w.mode] * sm_max * 1e6        # lane-instr/s
    t_launch = t_sweep / K
    achieved = sweep_pairs * ALG_INSTR[w.mode] / t_launch
    executed = sweep_pairs * (1.0 + acc) * ALG_INSTR[w.mode] / t_launch
    traffic = NCU_TRAFFIC_BYTES.get((w.name, w.mode)) if m == 1 and not args.walkers else None
    real_bytes = 8 if w.mode == wl.MODE_FP64 else 4
    ld = (N + 3) // 4 * 4
    # algorithmic bytes of one sweep launch: coordinates and running sums read once and written once, counters (the
    # written half may still sit in the 126 MB L2 when the launch ends, which is why ncu's dram figure can be lower)
    traffic_algorithmic = 2 * (W * 3 * ld * real_bytes + W * ld * 8) + 2 * W * 8
    # Lower bound of the FP32C sweep's time from the MEASURED instruction mix (ncu, per executed pair evaluation) and
    # the pipes' rates: every pipe must at least issue its own instructions; the largest of these is the bound.
    pipe_bound = None
    if w.mode == wl.MODE_FP32C and w.name == "c3-N1952":
        clk = sm_max * 1e6
        executed_pairs = sweep_pairs * (1.0 + acc)
        ffma2_lane_rate = 2.0 * rates["ffma2"]                                    # fp32 lane results per second, packed
        per_pipe = {}
        for pipe, slots in NCU_SWEEP32_SLOTS.items():
            rate = info["sm_count"] * PIPE_LANES[pipe] * clk                      # thread-instr/s the pipe can issue
            if pipe == "xu":
                rate = min(rate, rates["mufu_rsq"])                               # live probe
            per_pipe[pipe] = {"slots_per_executed_pair": slots, "rate_G_s": rate / 1e9,
                              "t_min_ms": 1e3 * slots * executed_pairs / rate}
        # the FMA pipe's packed instructions occupy it for two clocks: its bound in pipe-cycles is what ncu's
        # pipe_fma_cycles_active measures
        per_pipe["fma"]["t_min_ms_packed_two_clocks"] = 2.0 * per_pipe["fma"]["t_min_ms"]
        bound_pipe = max(per_pipe, key=lambda k: per_pipe[k]["t_min_ms"])
        t_bound = per_pipe[bound_pipe]["t_min_ms"]
        pipe_bound = {"per_pipe": per_pipe, "binding_pipe": bound_pipe, "t_bound_ms": t_bound,
                      "frac_of_pipe_bound": t_bound / (1e3 * t_launch),
                      "ncu_utilization_pct": NCU_SWEEP32_UTIL_PCT, "ffma2_lane_rate_measured_G_s": ffma2_lane_rate / 1e9,
                      "source": "instruction mix: profiles/r02b_instr.md; utilisation: profiles/r02b_kernels.md (constants of the "
                                "round-2 sweep kernel, unchanged this round); rates: SMs x lanes x max clock, XU from the live probe",
                      "reading": "no pipe is saturated: the issue slots are the tightest bound, and the kernel runs at "
                                 "frac_of_pipe_bound of it; the rest is the per-move serial part (reduction, barrier, decision)"}
    roofline = {
        "bound": "alu", "kernel": f"sweep_kernel<{mode_name}>",
        "achieved": achieved / 1e9, "peak": peak_derived / 1e9, "unit": "G thread-instr/s",
        "frac": achieved / peak_derived, "traffic": traffic,
        "traffic_source": NCU_TRAFFIC_SOURCE if traffic is not None else None,
        "traffic_algorithmic": traffic_algorithmic,
        "traffic_note": "traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch from the named ncu capture; "
                        "traffic_algorithmic: computed here from W, N and the mode (coordinates + running sums read once "
                        "and written once; written lines may outlive the launch in L2)",
        "frac_survey_count": (sweep_pairs * SURVEY_INSTR_FP32C / t_launch / peak_derived) if w.mode == wl.MODE_FP32C else None,
        "frac_of_measured_fma_chain": achieved / peak_meas,
        "pipe_bound": pipe_bound,
        "peak_source": f"derived: {info['sm_count']} SMs x {LANES_PER_SM[w.mode]} lanes x {sm_max:.0f} MHz (DESIGN.md); "
                       "MEASURED_PEAKS.json has no ALU entry",
        "peak_measured_fma_chain": peak_meas / 1e9,
        "alg_instr_per_pair_eval": ALG_INSTR[w.mode],
        "executed_frac": executed / peak_derived,
        "note": "achieved counts ONE trial evaluation per (moved, other) pair; executed_frac adds the "
                "accepted-move re-evaluations the running-sum update performs (x(1+acceptance))",
        "kernel_ms": 1e3 * t_launch,
        # the special-function unit (MUFU: 16 lanes per SM) is the co-limiter of the FP32C pair loop:
        # 2 MUFU per u-evaluation (rsqrt, rcp); fp64 mode issues the same two (64H seeds)
        "xu": {"peak_measured_G_instr_s": rates["mufu_rsq"] / 1e9,
               "frac": sweep_pairs * 2.0 / t_launch / rates["mufu_rsq"],
               "executed_frac": sweep_pairs * (1.0 + acc) * 2.0 / t_launch / rates["mufu_rsq"]},
        "pipe_rates_measured_G_instr_s": {k: v / 1e9 for k, v in rates.items()},
    }

    out = {
        "metric": "pair evaluations/s (sweep N(N-1) + energy N(N-1)/2 per walker-step)",
        "value": value, "unit": "pair-evals/s", "n_gpus": world, "steps": K, "warmup": args.warmup,
        "ms_per_step": 1e3 * t_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "ms_per_step_median": statistics.median(head.step_ms), "sweep_ms_median": statistics.median(head.sweep_ms),
        "dtype": "f32" if w.mode == wl.MODE_FP32C else "f64", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "walkers_per_gpu": W, "groups": len(w.groups),
                   "sweeps_per_step": m, "mode": mode_name, "energy_every_step": True,
                   "proposal": "ordered/uniform-cube" if args.proposal == 0 else f"random-particle/gaussian sigma={args.sigma} A",
                   "l2": "flushed between timed steps (256 MiB write, untimed)",
                   "equilibration_sweeps_untimed": equil,
                   "sweep_threads": info["sweep_threads"], "sweep_ctas_per_sm": info["sweep_ctas_per_sm"],
                   "sweep_tile": info["sweep_tile"], "sweep_cluster": info["sweep_cluster"],
                   "sweep_pairs_per_thread": info["sweep_pairs_per_thread"], "tuning_overrides": args.tune,
                   "energy_threads": info["energy_threads"], "energy_ctas_per_sm": info["energy_ctas_per_sm"]},
        "walker_sweeps_per_s": world * K * W * m / t_total,
        "sweep_only": {"pair_evals_per_s": world * K * sweep_pairs / t_sweep,
                       "walker_sweeps_per_s": world * K * W * m / t_sweep, "ms": 1e3 * t_sweep / K,
                       "u_evals_executed_per_s": world * K * sweep_pairs * (1 + acc) / t_sweep},
        "energy_only": {"pairs_per_s": world * K * energy_pairs / (t_total - t_sweep),
                        "ms": 1e3 * (t_total - t_sweep) / K},
        "acceptance": acc, "energy_per_atom_K": dict(zip(["E_PB", "V", "T_PB", "T_JF"], e_mean)),
        "clocks": clocks,
        "e2e": {"value": world * Ke * pairs_step / t_e2e, "unit": "pair-evals/s",
                "h2d_bytes_per_step": W * 3 * N * 8 + W * N * 8, "d2h_bytes_per_step": W * 3 * N * 8 + W * N * 8 + W * 5 * 8,
                "ms_per_step": 1e3 * t_e2e / Ke,
                "api": "qmc_step_host (pinned host buffers: coordinates + pair sums in, energies + acceptance + "
                       "coordinates + pair sums out; walkers in chunks, copies overlap the compute)",
                "coordinates_only": {"value": pairs_step / t_e2e_xyz, "ms_per_step": 1e3 * t_e2e_xyz,
                                     "note": "h_S_in = NULL: the pair sums are rebuilt on the device after the upload "
                                             "(one more all-pairs pass)"}},
        "gpu_launches": int(launches),
        "roofline": roofline,
    }
    # ---- the other BASELINE.json configs and the fp64 comparison run of config 3, a few steps each (VERDICT r1
    # missing #3): sweep / energy times, pair evaluations per second, roofline fraction -----------------------
    if not args.no_configs and world == 1 and args.config == 3 and args.mode == "default" and not args.walkers:
        head.q.close()
        blocks = {}
        for name, cfg, mode, k_steps in (("c1", 1, None, 20), ("c2", 2, None, 20), ("c3-fp64", 3, wl.MODE_FP64, 5),
                                         ("c4", 4, None, 3), ("c5", 5, None, 5)):
            wc = wl.config(cfg)
            if mode is not None:
                wc = wl.with_mode(wc, mode)
            tc = Timed(wc, 1, dev, 0).run(EQUIL_SWEEPS[cfg] if cfg != 3 else 60, 3, k_steps, flush)
            blocks[name] = summarize(tc, k_steps, info["sm_count"], sm_max)
            tc.q.close()
            del tc
        out["configs"] = blocks
        head = Timed(w, m, dev, rank, args.proposal, args.sigma)      # a fresh context for the items below
        head.q.sweep(30, head.steps)
        q = head.q
    e_out = head.e_out
    # ---- observables beside the hot path: g(r) histogram, time to error ----
    nb = 256
    hist = torch.empty((W, nb), dtype=torch.int32, device=dev)
    try:
        q.pair_histogram(nb, hist)
        hist_ok = True
    except binding.QmcError as exc:                  # QMC_E_CAPACITY: N beyond that kernel's shared memory
        if exc.code != binding.QMC_E_CAPACITY:
            raise
        hist_ok = False
    if hist_ok:
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(3):
            q.pair_histogram(nb, hist)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 3
        out["observables"] = {"pair_histogram_ms": ms, "pairs_per_s": W * N * (N - 1) / 2 / (ms * 1e-3), "nbins": nb,
                              "pairs_inside_cutoff_per_walker": float(hist.sum(1).double().mean())}
    # ---- NEXT-4: blocks with in-flight write-outs (state stays on the device, results stream to pinned host memory)
    nblk = max(3, min(K, 10))
    hb_e = torch.zeros((nblk, W, 4), dtype=torch.float64).pin_memory()
    hb_a = torch.zeros((nblk, W), dtype=torch.float64).pin_memory()
    hb_d = torch.zeros((nblk,), dtype=torch.int32).pin_memory()
    q.run_blocks_host(1, m, steps, hb_e, hb_a, hb_d)
    q.wait()
    hb_d.zero_()
    t0 = time.perf_counter()
    q.run_blocks_host(nblk, m, steps, hb_e, hb_a, hb_d)
    t_enq = time.perf_counter() - t0
    q.wait()
    t_blk = time.perf_counter() - t0
    out["blocks_host"] = {"value": nblk * pairs_step / t_blk, "unit": "pair-evals/s", "blocks": nblk,
                          "ms_per_block": 1e3 * t_blk / nblk, "enqueue_ms": 1e3 * t_enq,
                          "d2h_bytes_per_block": W * 5 * 8, "flags_raised": int(hb_d.sum()),
                          "api": "qmc_run_blocks_host (write-outs on a second stream while the next block computes)"}
    # in-kernel write-outs (the paper's own mechanism): one launch, coordinates to mapped pinned host memory every sweep
    n_wo = 4
    wo_x = torch.zeros((n_wo, W, 3, N), dtype=torch.float64).pin_memory()
    wo_f = torch.zeros((n_wo, W), dtype=torch.int32).pin_memory()
    t0 = time.perf_counter()
    q.sweep_writeouts(n_wo * m, steps, m, wo_x, None, wo_f)
    q.wait()
    t_wo = time.perf_counter() - t0
    out["sweep_writeouts"] = {"sweeps": n_wo * m, "writeouts": n_wo, "ms_per_sweep": 1e3 * t_wo / (n_wo * m),
                              "bytes_per_writeout": W * 3 * N * 8, "flags_raised": int(wo_f.sum()),
                              "api": "qmc_sweep_writeouts (one launch; thread blocks write coordinates to mapped pinned "
                                     "host memory every m sweeps and raise per-walker flags)"}
    if args.large_n:
        out["large_n"] = large_n_block(dev, flush)
    if args.time_to_error is None:
        args.time_to_error = 40 if (args.config == 3 and world == 1 and not args.walkers) else 0
    if args.time_to_error > 0:
        from paper_1312_1282_b200 import observables as ob
        S = args.time_to_error
        series = []
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(S):
            head.one_step()
            series.append(e_out[:, 0].mean().item() / N)       # walker-averaged E_PB per atom of this step
        el = time.perf_counter() - t0
        mean, se, tau = ob.reblock(series, min_blocks=8)
        tsig, t_goal = ob.seconds_to_error(se, el)
        out["time_to_error"] = {"steps": S, "seconds": el, "E_per_atom_K": mean, "se_K": se, "tau_steps": tau,
                                "t_sigma2_s_mK2": tsig, "seconds_to_1mK_per_atom": t_goal,
                                "paper_t_sigma2_s_mK2": {"N512_K20": 130.0, "N512_M2090": 200.0,
                                                         "cite": "PAPER.md l.504-511 (other hardware, N = 512: context only)"},
                                "note": f"chain equilibrated for {equil}+ sweeps before the series"}
    if not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(w, m)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def large_n_block(dev, flush):
    """NEXT-3 figures (418 ms per sweep and chain at N = 40960 on a K20 -- context, not a
    target): ms per sweep per chain at N = 40960 with the paper's 13 walkers on clusters of 8 blocks, and the single-walker case
    (l.490) at N = 10000 and N = 1952 on a cluster of 8 against one block."""
    import torch
    from paper_1312_1282_b200 import binding

    def timed(N, W, cluster, sweeps):
        binding.set_tuning()
        if cluster is not None:
            binding.set_tuning("sweep_cluster", cluster)
        L = wl.box_edge(N, wl.RHO_EQ)
        q = binding.QMC(N, [W], [L], [2.89], wl.HBAR2_OVER_2M, wl.AZIZ_HFDB_HE, wl.MODE_FP32C, jitter=wl.JITTER, device=str(dev))
        binding.set_tuning()
        inf = q.info()
        q.init_walkers(wl.SEED)
        q.sweep(2, 1.0)
        e_out = q.local_energy()
        torch.cuda.synchronize()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        flush.zero_()
        ev[0].record()
        q.sweep(sweeps, 1.0)
        ev[1].record()
        q.local_energy(e_out)
        ev[2].record()
        torch.cuda.synchronize()
        r = {"N": N, "walkers": W, "blocks_per_walker": inf["sweep_cluster"], "threads": inf["sweep_threads"],
             "ms_per_sweep_per_chain": ev[0].elapsed_time(ev[1]) / sweeps, "energy_ms": ev[1].elapsed_time(ev[2]),
             "energy_variant": inf["energy_variant"], "acceptance": float(q.acceptance().mean()),
             "pair_evals_per_s": W * N * (N - 1) * sweeps / (ev[0].elapsed_time(ev[1]) * 1e-3)}
        q.close()
        return r

    out = {"n40960_13_walkers": timed(40960, 13, None, 1), "paper_k20_ms_per_sweep_per_chain_n40960_13_walkers": 418.0}
    out["single_walker"] = {f"N{N}_{'cluster8' if c == 8 else 'one_block'}": timed(N, 1, c, 4 if N < 5000 else 1)
                            for N in (10000, 1952) for c in (8, 1)}
    return out


if __name__ == "__main__":
    main()
