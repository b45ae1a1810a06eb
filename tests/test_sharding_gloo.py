"""N>1 path on CPU: world_size-2 gloo processes each own a contiguous walker shard (no data-path
collective), compute it (here with the oracle standing in for the device), and the final reduction /
gather reproduces the single-process result exactly."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1312_1282_b200 import parallel, workloads as wl


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _run_shard(w, wpg, base):
    """per-walker [E_PB, V, T_PB, T_JF] after 3 sweeps for the walkers of one shard (oracle compute)."""
    import oracle
    rows, wid = [], base
    lo = 0
    for g, grp in enumerate(w.groups):
        n = wpg[g]
        if n:
            s = oracle.System(w.n_atoms, w.box_L[g], grp.b, w.hbar2_over_2m, w.aziz)
            x = oracle.init_walkers(s, w.seed, wid, n, wl.JITTER)
            oracle.sweep(s, x, w.seed, wid, 0, 3, grp.step)
            rows.append(oracle.local_energy(s, x)[:, :4])
            wid += n
    return np.concatenate(rows) if rows else np.zeros((0, 4))


def _worker(rank, world, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.Workload("t", 32, (wl.Group(wl.RHO_EQ, 2.89, 5, 1.0), wl.Group(0.0240, 2.8, 4, 0.9)), 3, wl.MODE_FP64)
    wpg, base = parallel.shard_for_rank(w, rank, world)
    local = torch.from_numpy(_run_shard(w, wpg, base))
    counts = [sum(parallel.shard_for_rank(w, r, world)[0]) for r in range(world)]
    allrows = parallel.gather_walkers(local, counts)
    stats = parallel.walker_statistics(local)
    if rank == 0:
        ret["rows"] = allrows.numpy()
        ret["mean"] = stats["mean"].numpy()
        ret["se"] = stats["se"].numpy()
        ret["n"] = float(stats["n"])
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_walker_sharding_matches_single_process():
    world, port = 2, _free_port()
    mgr = mp.Manager()
    ret = mgr.dict()
    mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
    w = wl.Workload("t", 32, (wl.Group(wl.RHO_EQ, 2.89, 5, 1.0), wl.Group(0.0240, 2.8, 4, 0.9)), 3, wl.MODE_FP64)
    ref = _run_shard(w, w.walkers_per_group, 0)
    assert ret["n"] == 9
    assert np.array_equal(ret["rows"], ref)                      # same walkers, bit for bit, in global order
    assert np.allclose(ret["mean"], ref.mean(0), rtol=1e-13)
    assert np.allclose(ret["se"], ref.std(0, ddof=1) / 3.0, rtol=1e-9)


def test_shard_groups_split_across_group_boundaries():
    w = wl.config(5)
    assert wl.shard_groups(w, 0, w.n_walkers) == (w.walkers_per_group, 0)
    wpg, base = wl.shard_groups(w, 1000, 2100)
    assert base == 1000 and wpg[:3] == [24, 1024, 52] and sum(wpg) == 1100
    for world in (2, 3, 8):
        tot = [0] * 16
        for r in range(world):
            wpg, base = parallel.shard_for_rank(w, r, world)
            assert base == wl.walker_shard(w.n_walkers, r, world)[0]
            tot = [a + b for a, b in zip(tot, wpg)]
        assert tot == w.walkers_per_group


def test_bench_gpus_flag_starts_that_many_ranks():
    """`python bench.py --gpus 2` with no launcher around it starts two ranks itself (torch.distributed.run on
    127.0.0.1) and rank 0 reports n_gpus = 2; --plumbing-only keeps the GPU out of it (gloo), so this runs on CPU."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    env["OMP_NUM_THREADS"] = "1"
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--plumbing-only"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, r.stdout
    out = json.loads(lines[0])
    assert out["n_gpus"] == 2 and out["requested_gpus"] == 2
    # and a single process stays a single rank
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--plumbing-only"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0 and json.loads(r.stdout.strip().splitlines()[-1])["n_gpus"] == 1
