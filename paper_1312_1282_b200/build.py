"""Build libqmc_b200.so (hand-written CUDA for sm_100a) in-tree with nvcc.

    python -m paper_1312_1282_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The translation units compile in parallel.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libqmc_b200.so")
PROBE_LIB = os.path.join(HERE, "libqmc_probe_b200.so")      # measurement tool (include/qmc_probe.h), not the product
PROBE_SRC = os.path.join(HERE, "probe", "qmc_probe.cu")
SOURCES = ["qmc_api.cu", "qmc_sweep_plan.cu", "qmc_sweep_f32.cu", "qmc_sweep_f64.cu", "qmc_sweep_tile_f32.cu", "qmc_sweep_cluster_f32.cu", "qmc_sweep_cluster_f64.cu", "qmc_energy.cu",
           "qmc_energy_f32.cu", "qmc_energy_f32s.cu", "qmc_energy_f64.cu", "qmc_observables.cu"]
HEADERS = ["qmc_device.cuh", "qmc_internal.h", "qmc_sweep_impl.cuh", "qmc_sweep_tile.cuh", "qmc_sweep_cluster.cuh", "qmc_f32c.cuh", "qmc_energy_f32_pair.cuh", os.path.join("..", "..", "include", "qmc.h")]
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Xcompiler", "-O2"]


def _stale() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(PROBE_LIB):
        return True
    t = min(os.path.getmtime(LIB), os.path.getmtime(PROBE_LIB))
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.abspath(__file__), PROBE_SRC]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)

    def compile_one(src: str) -> str:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        cmd = [NVCC, *FLAGS, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src}")
        return obj

    with ThreadPoolExecutor(max_workers=len(SOURCES)) as ex:
        objs = list(ex.map(compile_one, SOURCES))
    subprocess.check_call([NVCC, "-shared", "-o", LIB, *objs, "-gencode", "arch=compute_100a,code=sm_100a", "-ldl"])
    subprocess.check_call([NVCC, *FLAGS, "-shared", "-o", PROBE_LIB, PROBE_SRC])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
