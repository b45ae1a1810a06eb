"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/qmc.h declares; host-only logic (parameter validation, state sizing, sharding) behaves;
and the product fails loudly -- no CPU fallback -- when there is no GPU.  No compute calls."""
import ctypes as C
import os
import re
import subprocess

import pytest

from conftest import ROOT
from paper_1312_1282_b200 import binding, workloads as wl


@pytest.fixture(scope="module")
def lib():
    from paper_1312_1282_b200 import build
    build.build()
    return binding.load_library()


def header_symbols(name="qmc.h"):
    text = open(os.path.join(ROOT, "include", name)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(qmc_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    declared = header_symbols()
    assert sorted(binding.EXPORTS) == declared
    nm = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    exported = set(re.findall(r" T (qmc_[a-z_0-9]+)", nm))
    assert set(declared) <= exported
    for name in declared:
        assert getattr(lib, name) is not None
    # the measurement tool is a library of its own (include/qmc_probe.h), outside the product ABI
    nm = subprocess.run(["nm", "-D", "--defined-only", binding.PROBE_LIB_PATH], capture_output=True, text=True).stdout
    assert set(header_symbols("qmc_probe.h")) == set(re.findall(r" T (qmc_[a-z_0-9]+)", nm)) == {"qmc_probe_rate"}
    assert not set(header_symbols("qmc_probe.h")) & exported


def test_tuning_keys(lib):
    for key in ("sweep_threads", "sweep_per_thread", "sweep_vector", "sweep_pending", "sweep_tile", "sweep_cluster",
                "energy_threads", "energy_ordered"):
        assert lib.qmc_set_tuning(key.encode(), 1) == 0
    assert lib.qmc_set_tuning(b"no_such_key", 1) == binding.QMC_E_ARG
    assert lib.qmc_set_tuning(None, 0) == 0              # reset


def test_library_is_sm100a_and_not_linked_to_the_oracle():
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    ldd = subprocess.run(["ldd", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "oracle" not in ldd
    # the product sources never mention the oracle package
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1312_1282_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "vmc_oracle" not in src, f


def _params(N=64, mode=binding.QMC_FP64, W=4, L=None, b=2.89):
    L = wl.box_edge(N, wl.RHO_EQ) if L is None else L
    return binding._make_params(N, [W], [L], [b], wl.HBAR2_OVER_2M, wl.AZIZ_HFDB_HE, mode, 0, wl.JITTER)


def test_state_bytes_accounts_for_coordinates_pair_sums_and_counters(lib):
    p, keep = _params(N=1952, mode=binding.QMC_FP32C, W=2048)
    n = lib.qmc_state_bytes(C.byref(p))
    want = 2048 * (3 * 1952 * 4 + 1952 * 8 + 8)
    assert want <= n <= want + 3 * 256
    p, keep = _params(N=1952, mode=binding.QMC_FP64, W=2048)
    n64 = lib.qmc_state_bytes(C.byref(p))
    assert n64 - n == 2048 * 3 * 1952 * 4
    p, keep = _params(N=1, W=4)
    assert lib.qmc_state_bytes(C.byref(p)) == 0          # invalid -> 0


def test_invalid_parameters_are_rejected_before_touching_the_gpu(lib):
    ctx = C.c_void_p()
    for kw in ({"N": 1}, {"mode": 7}, {"W": 0}, {"L": -3.0}):
        p, keep = _params(**kw)
        rc = lib.qmc_create(C.byref(p), None, None, 0, C.byref(ctx))
        assert rc == binding.QMC_E_ARG and not ctx.value
        assert len(lib.qmc_last_error(None)) > 0


def test_no_gpu_means_a_loud_failure_not_a_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    w = wl.config(1)
    with pytest.raises(RuntimeError):
        binding.QMC.from_workload(w)
    # and the C entry point itself reports a CUDA error
    p, keep = _params()
    ctx = C.c_void_p()
    assert lib.qmc_create(C.byref(p), None, None, 0, C.byref(ctx)) == binding.QMC_E_CUDA
    with pytest.raises(binding.QmcError):
        binding.pipe_peak(0)


def test_workloads_match_baseline_configs():
    sizes = {1: (64, 64, 200), 2: (256, 1024, 500), 3: (1952, 2048, 1000), 4: (10000, 296, 100), 5: (512, 16384, 300)}
    for i, (N, W, S) in sizes.items():
        w = wl.config(i)
        assert (w.n_atoms, w.n_walkers, w.sweeps) == (N, W, S)
        for g, L in zip(w.groups, w.box_L):
            assert abs(N / L ** 3 - g.rho) < 1e-12 and 0 < g.step < L / 2
    assert len(wl.config(5).groups) == 16
    assert abs(wl.config(3).box_L[0] - 44.6968) < 1e-3


def test_walker_shards_partition_the_walkers():
    for W in (1, 7, 64, 2048):
        for world in (1, 2, 3, 8):
            spans = [wl.walker_shard(W, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == W
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            assert max(e - b for b, e in spans) - min(e - b for b, e in spans) <= 1


def test_liquid_configuration_is_seeded_and_respects_the_core():
    import numpy as np
    L = wl.box_edge(200, wl.RHO_EQ)
    a = wl.liquid_configuration(200, L, 3)
    b = wl.liquid_configuration(200, L, 3)
    assert a.shape == (3, 200) and np.array_equal(a, b)
    d = a.T[:, None, :] - a.T[None, :, :]
    d -= L * np.rint(d / L)
    r = np.sqrt((d ** 2).sum(-1)) + np.eye(200) * 1e9
    assert r.min() >= 2.3 and (a >= 0).all() and (a < L).all()
    c = wl.liquid_configuration(50, L, 4, fp32_grid=True)
    k = c / L * 2 ** 23
    assert np.abs(k - np.rint(k)).max() < 1e-6 and np.array_equal(np.rint(k) / 2 ** 23 * L, c)
