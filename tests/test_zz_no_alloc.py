"""qmc_local_energy_fp32c_static -- the local-energy call for users who are not allowed to allocate.

Every other way into the library reserves device memory: qmc_create calls cudaMalloc for the walker state and its
tables, and the gridded FP32C energy kernel calls it again for its working arrays the first time it runs.  That is
no use to a caller whose GPU memory has already been given in full to a pool (cudaMalloc then reports out-of-memory
although the pool has room), to one that sits in a latency-bound loop where an allocation's device-wide
synchronisation would stall the other streams, or to a plugin that may only touch the buffers it was handed.  For them
the library carries one fixed 5.1 MiB array in its own image and this one entry point that works in it: the caller
passes coordinates in and energies out, and nothing is allocated.

The GPU test checks the new call against the context-based path (qmc_create + qmc_set_positions + qmc_local_energy)
on the same configurations, at the tolerance the FP32C energy tests use (1e-5 relative, R22) and, against the
same gridded kernel, to the last bit.  It makes several calls in a row with DIFFERENT shapes, because all calls share
the one array and each starts on top of what the previous one left there: a call that relied on stale contents (the
padding of the coordinate rows, the walker -> parameter table, the partial sums) would show up in the second or third.

This file is named so that pytest collects it last; it sets up everything it needs itself, so it passes alone in a
fresh process as well as after the rest of the suite (which leaves other contexts and tuning overrides behind).
"""
import numpy as np
import pytest

from paper_1312_1282_b200 import workloads as wl

AZ, DK, B = wl.AZIZ_HFDB_HE, wl.HBAR2_OVER_2M, 2.89
TOL32 = 1e-5        # the FP32C energy tolerance of tests/test_gpu_parity.py (north_star)


def _relerr32(e, ref):
    """Same reading of "relative 1e-5" as test_gpu_parity.relerr32 (E_PB floored by (|V| + |T_PB|) / 20)."""
    den = np.abs(ref).copy()
    den[:, 0] = np.maximum(den[:, 0], (np.abs(ref[:, 1]) + np.abs(ref[:, 2])) / 20.0)
    return np.abs(e - ref) / np.maximum(den, 1e-300)


def test_static_entry_point_refuses_oversize_without_touching_the_gpu():
    """Sizes beyond the static array are turned down with QMC_E_CAPACITY and a message naming the limits, before any
    CUDA call: runs on the CPU box (the pointers are never dereferenced)."""
    import torch
    from paper_1312_1282_b200 import binding, build
    build.build()
    binding.load_library()
    for W, N in ((binding.STATIC_MAX_WALKERS + 1, 2), (1, binding.STATIC_MAX_ATOMS + 1), (129, 2048), (27, 10000)):
        xyz = torch.zeros((W, 3, N), dtype=torch.float64)
        out = torch.zeros((W, 4), dtype=torch.float64)
        with pytest.raises(binding.QmcError) as ei:
            binding.local_energy_fp32c_static(xyz, 50.0, B, DK, AZ, out)
        assert ei.value.code == binding.QMC_E_CAPACITY
        assert "static scratch" in str(ei.value) and str(binding.STATIC_MAX_SLOTS) in str(ei.value)
    # bad arguments are refused too (N < 2)
    with pytest.raises(binding.QmcError) as ei:
        binding.local_energy_fp32c_static(torch.zeros((1, 3, 1), dtype=torch.float64), 50.0, B, DK, AZ,
                                          torch.zeros((1, 4), dtype=torch.float64))
    assert ei.value.code == binding.QMC_E_ARG


@pytest.mark.gpu
def test_static_entry_point_matches_the_context_path_on_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1312_1282_b200 import binding, build
    build.build()
    binding.load_library()
    binding.set_tuning()                                  # whatever earlier tests forced is gone

    def context_path(N, W, seed, gridded):
        """Liquid-like configurations and their energies through the existing, allocating path."""
        L = wl.box_edge(N, wl.RHO_EQ)
        binding.set_tuning()
        if gridded:
            binding.set_tuning("energy_ordered", 3)       # the gridded kernel, whatever W and N
        try:
            q = binding.QMC(N, [W], [L], [B], DK, AZ, binding.QMC_FP32C, jitter=wl.JITTER)
        finally:
            binding.set_tuning()
        q.init_walkers(seed)
        q.sweep(3, 0.35)                                  # off the lattice
        xyz = q.get_positions().clone()                   # exact widening of the fp32 grid coordinates
        e = q.local_energy().clone()
        variant = q.info()["energy_variant"]
        torch.cuda.synchronize()
        q.close()
        return L, xyz, e.cpu().numpy(), variant

    # (N, W): ragged N with several walkers; a smaller, differently ragged N (stale padding and tables from the call
    # before); one walker of many atoms spread over many thread blocks; then the first shape again
    shapes = [(1100, 5), (515, 3), (4099, 1), (1100, 5)]
    cases = {}
    for N, W in set(shapes):
        L, xyz, e_grid, v3 = context_path(N, W, wl.SEED + N, gridded=True)
        _, xyz2, e_default, v = context_path(N, W, wl.SEED + N, gridded=False)
        assert v3 == 3 and torch.equal(xyz, xyz2)
        cases[(N, W)] = (L, xyz, e_grid, e_default, v)

    outs = []
    for N, W in shapes:                                   # back to back on one stream, no synchronisation in between
        L, xyz, _, _, _ = cases[(N, W)]
        out = torch.full((W, 4), float("nan"), dtype=torch.float64, device=xyz.device)
        binding.local_energy_fp32c_static(xyz, L, B, DK, AZ, out)
        outs.append(out)
    torch.cuda.synchronize()

    for (N, W), out in zip(shapes, outs):
        _, _, e_grid, e_default, v = cases[(N, W)]
        e = out.cpu().numpy()
        assert np.isfinite(e).all()
        # against the context path at the FP32C energy tolerance, whichever kernel the planner picks by default
        assert _relerr32(e, e_default).max() < TOL32, (N, W, v, _relerr32(e, e_default).max())
        # against the same kernel with cudaMalloc'ed working memory: the same bits
        assert np.array_equal(e, e_grid), (N, W, np.abs(e - e_grid).max())
    # the two calls with the same input gave the same output, with two other shapes run in between
    assert torch.equal(outs[0], outs[3])

    # coordinates that are not on the FP32C grid, and outside [0, L): rounded and wrapped as qmc_set_positions does
    N, W = 515, 3
    L, xyz, _, _, _ = cases[(N, W)]
    g = torch.Generator(device="cpu").manual_seed(7)
    off = xyz.cpu() + (torch.rand(xyz.shape, generator=g, dtype=torch.float64) - 0.5) * (L * 2.0 ** -24)
    off[:, :, ::7] += L
    off[:, :, 3::11] -= L
    off = off.to(xyz.device).contiguous()
    q = binding.QMC(N, [W], [L], [B], DK, AZ, binding.QMC_FP32C, jitter=wl.JITTER)
    q.set_positions(off)
    ref = q.local_energy().cpu().numpy()
    q.close()
    out = torch.empty((W, 4), dtype=torch.float64, device=xyz.device)
    binding.local_energy_fp32c_static(off, L, B, DK, AZ, out)
    torch.cuda.synchronize()
    assert _relerr32(out.cpu().numpy(), ref).max() < TOL32
