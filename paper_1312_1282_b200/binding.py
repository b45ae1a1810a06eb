"""Thin Python binding of the C ABI in include/qmc.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libqmc_b200.so.  PyTorch supplies
device buffers (tensor.data_ptr()) and the CUDA stream handle, nothing else.  There is no
CPU fallback: a missing library or a missing GPU raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libqmc_b200.so")

QMC_FP64, QMC_FP32C = 0, 1
QMC_OK, QMC_E_ARG, QMC_E_CAPACITY, QMC_E_CUDA, QMC_E_STATE = 0, -1, -2, -3, -4

# every symbol include/qmc.h declares
EXPORTS = (
    "qmc_state_bytes", "qmc_create", "qmc_destroy", "qmc_init_walkers", "qmc_sweep", "qmc_local_energy",
    "qmc_acceptance", "qmc_step_host", "qmc_last_error", "qmc_get_positions", "qmc_set_positions",
    "qmc_set_seed", "qmc_get_pair_sums", "qmc_refresh_pair_sums", "qmc_trace_decisions", "qmc_info",
    "qmc_pair_histogram", "qmc_set_proposal", "qmc_run_blocks_host", "qmc_wait", "qmc_sweep_writeouts",
    "qmc_set_tuning", "qmc_local_energy_fp32c_static", "qmc_create_tuned",
)
# limits of qmc_local_energy_fp32c_static (include/qmc.h)
STATIC_MAX_WALKERS, STATIC_MAX_ATOMS, STATIC_MAX_SLOTS, STATIC_SCRATCH_BYTES = 4096, 65536, 262144, 5382656
PROBE_LIB_PATH = os.path.join(HERE, "libqmc_probe_b200.so")


class QmcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"qmc error {code}: {msg}")
        self.code = code


class _Params(C.Structure):
    _fields_ = [
        ("N", C.c_int32), ("n_groups", C.c_int32),
        ("walkers_per_group", C.POINTER(C.c_int32)), ("box_L", C.POINTER(C.c_double)),
        ("jastrow_b", C.POINTER(C.c_double)),
        ("hbar2_over_2m", C.c_double), ("aziz", C.c_double * 9),
        ("mode", C.c_int32), ("walker_id_base", C.c_uint32), ("jitter", C.c_double),
    ]


class Info(C.Structure):
    _fields_ = [
        ("W", C.c_int32), ("N", C.c_int32), ("n_groups", C.c_int32), ("mode", C.c_int32),
        ("sweep_threads", C.c_int32), ("sweep_ctas_per_sm", C.c_int32), ("sweep_smem_bytes", C.c_int32),
        ("sweep_pairs_per_thread", C.c_int32),
        ("energy_threads", C.c_int32), ("energy_ctas_per_sm", C.c_int32), ("energy_smem_bytes", C.c_int32),
        ("sm_count", C.c_int32), ("t", C.c_uint32), ("kernel_launches", C.c_uint64),
        ("sweep_vector", C.c_int32), ("sweep_pending", C.c_int32), ("sweep_tile", C.c_int32),
        ("energy_variant", C.c_int32), ("sweep_cluster", C.c_int32),
    ]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


_lib = None


def load_library() -> C.CDLL:
    """dlopen libqmc_b200.so and declare the prototypes.  Raises if it has not been built
    (python -m paper_1312_1282_b200.build): the product has no other path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} is missing: build the CUDA library first (python -m paper_1312_1282_b200.build). "
            "There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    lib.qmc_state_bytes.argtypes = [C.POINTER(_Params)]
    lib.qmc_state_bytes.restype = C.c_size_t
    lib.qmc_create.argtypes = [C.POINTER(_Params), vp, vp, C.c_size_t, C.POINTER(vp)]
    lib.qmc_create_tuned.argtypes = [C.POINTER(_Params), vp, vp, C.c_size_t, C.POINTER(C.c_char_p), C.POINTER(C.c_int32),
                                     C.c_int32, C.POINTER(vp)]
    lib.qmc_destroy.argtypes = [vp]
    lib.qmc_init_walkers.argtypes = [vp, C.c_uint64]
    lib.qmc_sweep.argtypes = [vp, C.c_int32, dp]
    lib.qmc_local_energy.argtypes = [vp, vp]
    lib.qmc_acceptance.argtypes = [vp, vp]
    lib.qmc_pair_histogram.argtypes = [vp, C.c_int32, vp]
    lib.qmc_set_proposal.argtypes = [vp, C.c_int32]
    lib.qmc_run_blocks_host.argtypes = [vp, C.c_int32, C.c_int32, dp, vp, vp, C.c_int32, vp, vp]
    lib.qmc_sweep_writeouts.argtypes = [vp, C.c_int32, dp, C.c_int32, vp, vp, vp]
    lib.qmc_set_tuning.argtypes = [C.c_char_p, C.c_int32]
    lib.qmc_wait.argtypes = [vp]
    lib.qmc_step_host.argtypes = [vp, vp, vp, C.c_int32, dp, vp, vp, vp, vp]
    lib.qmc_last_error.argtypes = [vp]
    lib.qmc_last_error.restype = C.c_char_p
    lib.qmc_get_positions.argtypes = [vp, vp]
    lib.qmc_set_positions.argtypes = [vp, vp]
    lib.qmc_set_seed.argtypes = [vp, C.c_uint64, C.c_uint32]
    lib.qmc_get_pair_sums.argtypes = [vp, vp]
    lib.qmc_refresh_pair_sums.argtypes = [vp]
    lib.qmc_trace_decisions.argtypes = [vp, C.c_int32, C.c_int32, vp, vp, C.c_int64]
    lib.qmc_info.argtypes = [vp, C.POINTER(Info)]
    lib.qmc_local_energy_fp32c_static.argtypes = [vp, C.c_int32, C.c_int32, C.c_double, C.c_double, dp, C.c_double, vp, vp,
                                                  C.c_char_p, C.c_size_t]
    for name in EXPORTS:
        if name not in ("qmc_state_bytes", "qmc_last_error"):
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _make_params(N, walkers_per_group, box_L, jastrow_b, hbar2_over_2m, aziz, mode, walker_id_base, jitter):
    g = len(walkers_per_group)
    assert len(box_L) == g and len(jastrow_b) == g
    keep = ((C.c_int32 * g)(*walkers_per_group), (C.c_double * g)(*box_L), (C.c_double * g)(*jastrow_b))
    p = _Params(int(N), g, keep[0], keep[1], keep[2], float(hbar2_over_2m), (C.c_double * 9)(*aziz),
                int(mode), int(walker_id_base), float(jitter))
    return p, keep


_probe = None


def pipe_peak(which: int, stream=None) -> float:
    """Thread-level instructions per second of one instruction kind, measured live by the separate probe library
    (include/qmc_probe.h: 0 DFMA, 1 FFMA, 2 FFMA2, 3 MUFU.RSQ, 4 I2FP, 5 F2F)."""
    import torch
    global _probe
    if _probe is None:
        if not os.path.exists(PROBE_LIB_PATH):
            raise FileNotFoundError(f"{PROBE_LIB_PATH} is missing: python -m paper_1312_1282_b200.build")
        _probe = C.CDLL(PROBE_LIB_PATH)
        _probe.qmc_probe_rate.argtypes = [C.c_int32, C.c_void_p, C.POINTER(C.c_double)]
        _probe.qmc_probe_rate.restype = C.c_int
    if not torch.cuda.is_available():
        raise QmcError(QMC_E_CUDA, "no CUDA device")
    st = torch.cuda.current_stream() if stream is None else stream
    out = C.c_double()
    rc = _probe.qmc_probe_rate(which, C.c_void_p(st.cuda_stream), C.byref(out))
    if rc != 0:
        raise QmcError(rc, "qmc_probe_rate failed")
    return out.value


def set_tuning(key: Optional[str] = None, value: int = -1):
    """qmc_set_tuning: process-wide launch-heuristic override for contexts created afterwards; set_tuning() resets."""
    lib = load_library()
    rc = lib.qmc_set_tuning(key.encode() if key is not None else None, int(value))
    if rc != 0:
        raise QmcError(rc, lib.qmc_last_error(None).decode())


def local_energy_fp32c_static(xyz, box_L: float, jastrow_b: float, hbar2_over_2m: float, aziz: Sequence[float], out,
                              stream=None):
    """qmc_local_energy_fp32c_static: FP32C local energies [W][4] (E_PB, V, T_PB, T_JF in K) of the configurations
    xyz [W][3][N] (float64 CUDA tensor, Angstrom) written into `out` ([W][4] float64 CUDA tensor), with no context and no
    allocation on the library's side: its working memory is a fixed 5.1 MiB array inside the library image.  This is the
    call for code that cannot reserve device memory itself -- the GPU's memory is already committed to a pool, or an
    allocation (which may synchronise the whole device) is not acceptable where the call is made, or the caller may
    only touch buffers it was handed.  Both tensors are the caller's; this wrapper creates none.  Limits:
    W <= STATIC_MAX_WALKERS, N <= STATIC_MAX_ATOMS, W * roundup32(N) <= STATIC_MAX_SLOTS, else QmcError(QMC_E_CAPACITY).
    The first call on a device looks up the array's address: make it before any stream capture.  Every call on a GPU
    shares the one array, so calls that could overlap on the device (different streams) must be ordered by the caller.
    Asynchronous on `stream` (default: torch's current stream)."""
    import torch
    lib = load_library()
    assert xyz.dim() == 3 and xyz.shape[1] == 3 and xyz.dtype == torch.float64 and xyz.is_contiguous(), (xyz.shape, xyz.dtype)
    W, _, N = (int(v) for v in xyz.shape)
    assert out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= 4 * W, (out.shape, out.dtype)
    if 1 <= W <= STATIC_MAX_WALKERS and 2 <= N <= STATIC_MAX_ATOMS and W * ((N + 31) // 32 * 32) <= STATIC_MAX_SLOTS:
        # sizes the library will accept reach the kernels: both tensors have to be on the same GPU, which is made current
        assert xyz.is_cuda and out.is_cuda and xyz.device == out.device, (xyz.device, out.device)
        torch.cuda.set_device(xyz.device)
        st = torch.cuda.current_stream(xyz.device) if stream is None else stream
        handle = C.c_void_p(st.cuda_stream)
    else:
        handle = None                       # the library refuses these sizes before any CUDA call
    err = C.create_string_buffer(512)
    rc = lib.qmc_local_energy_fp32c_static(C.c_void_p(xyz.data_ptr()), W, N, float(box_L), float(jastrow_b),
                                           (C.c_double * 9)(*aziz), float(hbar2_over_2m), C.c_void_p(out.data_ptr()),
                                           handle, err, len(err))
    if rc != 0:
        raise QmcError(rc, err.value.decode())
    return out


class QMC:
    """One context: W independent walkers of N atoms.  Methods mirror the C calls one to one."""

    def __init__(self, N: int, walkers_per_group: Sequence[int], box_L: Sequence[float],
                 jastrow_b: Sequence[float], hbar2_over_2m: float, aziz: Sequence[float], mode: int,
                 walker_id_base: int = 0, jitter: float = 0.05, device: str = "cuda:0", stream=None,
                 library_owns_state: bool = False, tuning: Optional[dict] = None):
        """tuning: this context's own launch overrides ({"sweep_threads": 128, ...}, the keys of qmc_set_tuning) through
        qmc_create_tuned; None: qmc_create, which takes the process-wide defaults of set_tuning()."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1312_1282_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self._torch = torch
        self._lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.stream = torch.cuda.current_stream(self.device) if stream is None else stream
        self.N = int(N)
        self.W = int(sum(walkers_per_group))
        self.n_groups = len(walkers_per_group)
        self.mode = int(mode)
        self._params, self._keep = _make_params(N, walkers_per_group, box_L, jastrow_b, hbar2_over_2m, aziz,
                                                mode, walker_id_base, jitter)
        nbytes = self._lib.qmc_state_bytes(C.byref(self._params))
        if nbytes == 0:
            raise QmcError(QMC_E_ARG, "invalid parameters")
        self._ctx = C.c_void_p()
        if library_owns_state:
            self._state, base, given = None, None, 0
        else:
            self._state = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base, given = C.c_void_p((self._state.data_ptr() + 255) & ~255), nbytes
        if tuning is None:
            rc = self._lib.qmc_create(C.byref(self._params), C.c_void_p(self.stream.cuda_stream), base, given,
                                      C.byref(self._ctx))
        else:
            n = len(tuning)
            keys = (C.c_char_p * max(n, 1))(*[k.encode() for k in tuning])
            vals = (C.c_int32 * max(n, 1))(*[int(v) for v in tuning.values()])
            rc = self._lib.qmc_create_tuned(C.byref(self._params), C.c_void_p(self.stream.cuda_stream), base, given,
                                            keys, vals, n, C.byref(self._ctx))
        if rc != 0:
            self._ctx = C.c_void_p()
            raise QmcError(rc, self._lib.qmc_last_error(None).decode())

    @classmethod
    def from_workload(cls, w, walker_range=None, **kw) -> "QMC":
        """Context for a workloads.Workload; walker_range=(begin,end) selects a shard of global walker ids."""
        from . import workloads
        wpg, base = list(w.walkers_per_group), 0
        if walker_range is not None:
            wpg, base = workloads.shard_groups(w, *walker_range)
        return cls(w.n_atoms, wpg, w.box_L, w.jastrow_b, w.hbar2_over_2m, w.aziz, w.mode,
                   walker_id_base=base, **kw)

    # -- helpers ---------------------------------------------------------------------------
    def _check(self, rc: int):
        if rc != 0:
            raise QmcError(rc, self._lib.qmc_last_error(self._ctx).decode())

    def _ptr(self, t, dtype, numel, device_type="cuda"):
        torch = self._torch
        assert t.dtype == dtype and t.is_contiguous() and t.numel() >= numel and t.device.type == device_type, \
            (t.dtype, t.shape, t.device)
        return C.c_void_p(t.data_ptr())

    def _steps(self, steps):
        if isinstance(steps, (int, float)):
            steps = [float(steps)] * self.n_groups
        assert len(steps) == self.n_groups
        return (C.c_double * self.n_groups)(*steps)

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self._lib.qmc_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the five calls --------------------------------------------------------------------
    def init_walkers(self, seed: int):
        self._check(self._lib.qmc_init_walkers(self._ctx, C.c_uint64(seed)))

    def sweep(self, n_sweeps: int, steps):
        self._check(self._lib.qmc_sweep(self._ctx, int(n_sweeps), self._steps(steps)))

    def local_energy(self, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty((self.W, 4), dtype=torch.float64, device=self.device)
        self._check(self._lib.qmc_local_energy(self._ctx, self._ptr(out, torch.float64, self.W * 4)))
        return out

    def acceptance(self, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty((self.W,), dtype=torch.float64, device=self.device)
        self._check(self._lib.qmc_acceptance(self._ctx, self._ptr(out, torch.float64, self.W)))
        return out

    def run_blocks_host(self, n_blocks: int, sweeps_per_block: int, steps, h_energy, h_acc=None, h_done=None,
                        xyz_every: int = 0, h_xyz=None):
        """qmc_run_blocks_host: asynchronous; h_energy [n_blocks][W][4], h_acc [n_blocks][W] float64, h_done [n_blocks]
        int32 and h_xyz [n_blocks // xyz_every][W][3][N] float64 are pinned host tensors that must stay alive until wait()."""
        torch = self._torch
        n_xyz = (n_blocks // xyz_every) if (h_xyz is not None and xyz_every > 0) else 0
        self._check(self._lib.qmc_run_blocks_host(
            self._ctx, int(n_blocks), int(sweeps_per_block), self._steps(steps),
            self._ptr(h_energy, torch.float64, n_blocks * self.W * 4, "cpu"),
            self._ptr(h_acc, torch.float64, n_blocks * self.W, "cpu") if h_acc is not None else None,
            int(xyz_every),
            self._ptr(h_xyz, torch.float64, n_xyz * self.W * 3 * self.N, "cpu") if h_xyz is not None else None,
            self._ptr(h_done, torch.int32, n_blocks, "cpu") if h_done is not None else None))

    def sweep_writeouts(self, n_sweeps: int, steps, every: int, xyz_out, n_acc_out, flags):
        """qmc_sweep_writeouts: ONE launch of n_sweeps sweeps whose thread blocks write coordinates / accepted-move
        counts out every `every` sweeps and raise flags[k][w].  The tensors are device tensors, or pinned host tensors
        (mapped into the device address space by CUDA's unified addressing), float64 / int64 / int32."""
        torch = self._torch
        n_out = n_sweeps // every
        for t_, dt, n in ((xyz_out, torch.float64, n_out * self.W * 3 * self.N), (n_acc_out, torch.int64, n_out * self.W),
                          (flags, torch.int32, n_out * self.W)):
            if t_ is not None:
                assert t_.dtype == dt and t_.is_contiguous() and t_.numel() >= n and (t_.is_cuda or t_.is_pinned())
        self._check(self._lib.qmc_sweep_writeouts(
            self._ctx, int(n_sweeps), self._steps(steps), int(every), C.c_void_p(xyz_out.data_ptr()),
            C.c_void_p(n_acc_out.data_ptr()) if n_acc_out is not None else None, C.c_void_p(flags.data_ptr())))

    def wait(self):
        self._check(self._lib.qmc_wait(self._ctx))

    def set_proposal(self, kind: int):
        """0: particles in order, uniform cube; 1: random particle, Gaussian displacement (qmc.h)."""
        self._check(self._lib.qmc_set_proposal(self._ctx, int(kind)))

    def pair_histogram(self, nbins: int, out=None):
        """[W][nbins] int32 tensor of pair-distance counts (uint32 on the C side; counts stay below 2^31)."""
        torch = self._torch
        if out is None:
            out = torch.empty((self.W, nbins), dtype=torch.int32, device=self.device)
        self._check(self._lib.qmc_pair_histogram(self._ctx, int(nbins), self._ptr(out, torch.int32, self.W * nbins)))
        return out

    def step_host(self, n_sweeps: int, steps, h_xyz_in=None, h_energy=None, h_acc=None, h_xyz_out=None,
                  h_S_in=None, h_S_out=None):
        """qmc_step_host with host tensors (pinned for asynchronous copies); h_S_in / h_S_out [W][N] carry the
        running pair sums along with the coordinates (opaque state, see qmc.h)."""
        torch = self._torch
        n = self.W * 3 * self.N

        def hp(t, numel):
            return self._ptr(t, torch.float64, numel, "cpu") if t is not None else None
        self._check(self._lib.qmc_step_host(
            self._ctx, hp(h_xyz_in, n), hp(h_S_in, self.W * self.N), int(n_sweeps), self._steps(steps),
            hp(h_energy, self.W * 4), hp(h_acc, self.W), hp(h_xyz_out, n), hp(h_S_out, self.W * self.N)))

    # -- state access and parity hooks -----------------------------------------------------
    def get_positions(self, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty((self.W, 3, self.N), dtype=torch.float64, device=self.device)
        self._check(self._lib.qmc_get_positions(self._ctx, self._ptr(out, torch.float64, self.W * 3 * self.N)))
        return out

    def set_positions(self, xyz):
        torch = self._torch
        xyz = torch.as_tensor(xyz, dtype=torch.float64).to(self.device).contiguous()
        assert tuple(xyz.shape) == (self.W, 3, self.N)
        self._check(self._lib.qmc_set_positions(self._ctx, self._ptr(xyz, torch.float64, self.W * 3 * self.N)))
        self.stream.synchronize()       # xyz may be a temporary

    def set_seed(self, seed: int, t: int = 0):
        self._check(self._lib.qmc_set_seed(self._ctx, C.c_uint64(seed), C.c_uint32(t)))

    def pair_sums(self):
        torch = self._torch
        out = torch.empty((self.W, self.N), dtype=torch.float64, device=self.device)
        self._check(self._lib.qmc_get_pair_sums(self._ctx, self._ptr(out, torch.float64, self.W * self.N)))
        return out

    def refresh_pair_sums(self):
        self._check(self._lib.qmc_refresh_pair_sums(self._ctx))

    def trace_decisions(self, w_begin: int, w_end: int, moves_capacity: int, margins: bool = True):
        """Start recording; returns (dec uint8 [w_end-w_begin][capacity], margin float64 or None)."""
        torch = self._torch
        nw = w_end - w_begin
        dec = torch.zeros((nw, moves_capacity), dtype=torch.uint8, device=self.device)
        mar = torch.zeros((nw, moves_capacity), dtype=torch.float64, device=self.device) if margins else None
        self._check(self._lib.qmc_trace_decisions(
            self._ctx, w_begin, w_end, C.c_void_p(dec.data_ptr()),
            C.c_void_p(mar.data_ptr()) if mar is not None else None, moves_capacity))
        self._trace_keep = (dec, mar)
        return dec, mar

    def stop_trace(self):
        self._check(self._lib.qmc_trace_decisions(self._ctx, 0, 0, None, None, 0))
        self._trace_keep = None

    def info(self) -> dict:
        inf = Info()
        self._check(self._lib.qmc_info(self._ctx, C.byref(inf)))
        return inf.as_dict()
