"""ctypes loader for the CPU oracle (oracle/vmc_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, bench.py's cpu_baseline /
--impl reference legs and __graft_entry__.smoke() may import this package.  It
imports nothing from paper_1312_1282_b200 and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vmc_oracle.c")
_LIB = os.path.join(_HERE, "libvmc_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no FMA contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


class _Sys(C.Structure):
    _fields_ = [("N", C.c_int32), ("L", C.c_double), ("b", C.c_double), ("Dk", C.c_double),
                ("aziz", C.c_double * 9), ("proposal", C.c_int32)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        u8p = C.POINTER(C.c_uint8)
        sp = C.POINTER(_Sys)
        _lib.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        _lib.orc_move_variates.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_double, dp, dp]
        for name in ("orc_u", "orc_du", "orc_d2u"):
            fn = getattr(_lib, name)
            fn.argtypes = [C.c_double] * 3
            fn.restype = C.c_double
        _lib.orc_aziz.argtypes = [C.c_double, dp]
        _lib.orc_aziz.restype = C.c_double
        _lib.orc_log_psi.argtypes = [sp, dp]
        _lib.orc_log_psi.restype = C.c_double
        _lib.orc_pair_sums.argtypes = [sp, dp, dp]
        _lib.orc_delta_log_psi.argtypes = [sp, dp, C.c_int, dp]
        _lib.orc_delta_log_psi.restype = C.c_double
        _lib.orc_local_energy.argtypes = [sp, dp, dp]
        _lib.orc_grad_lap.argtypes = [sp, dp, dp, dp]
        _lib.orc_init_walkers.argtypes = [sp, C.c_uint64, C.c_uint32, C.c_int32, C.c_double, dp]
        _lib.orc_sweep_walkers.argtypes = [sp, dp, C.c_uint64, C.c_uint32, C.c_int32, C.c_uint32, C.c_int32,
                                           C.c_double, u8p, dp, u8p, C.POINTER(C.c_int64)]
        _lib.orc_local_energy_walkers.argtypes = [sp, dp, C.c_int32, dp]
        _lib.orc_num_threads.restype = C.c_int32
        _lib.orc_normal_pair.argtypes = [C.c_uint32, C.c_uint32, dp]
        _lib.orc_move_variates_gauss.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_int32, C.c_double,
                                                 C.POINTER(C.c_int32), dp, dp]
        _lib.orc_pair_histogram.argtypes = [sp, dp, C.c_int, C.POINTER(C.c_uint32)]
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


class System:
    """N atoms in a cubic periodic box of edge L, Jastrow b, hbar^2/2m = Dk, potential constants."""

    def __init__(self, N: int, L: float, b: float, Dk: float, aziz: Sequence[float], proposal: int = 0):
        """proposal 0: particles in order, uniform cube (R7); 1: the paper's random particle +
        Gaussian displacement of standard deviation `step` per component (l.144, l.325)."""
        self.N, self.L, self.b, self.Dk, self.aziz = int(N), float(L), float(b), float(Dk), tuple(aziz)
        self.proposal = int(proposal)
        self._s = _Sys(self.N, self.L, self.b, self.Dk, (C.c_double * 9)(*self.aziz), self.proposal)

    @property
    def ref(self):
        return C.byref(self._s)


def num_threads() -> int:
    return int(_load().orc_num_threads())


def philox4x32_10(ctr: Sequence[int], key: Sequence[int]) -> np.ndarray:
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    _load().orc_philox4x32_10(c, k, o)
    return np.array(list(o), dtype=np.uint32)


def move_variates(seed: int, w: int, t: int, s: int, step: float):
    d = np.zeros(3)
    xi = C.c_double()
    _load().orc_move_variates(seed, w, t, s, step, _dp(d), C.byref(xi))
    return d, xi.value


def u(r: float, L: float, b: float) -> float:
    return _load().orc_u(r, L, b)


def du(r: float, L: float, b: float) -> float:
    return _load().orc_du(r, L, b)


def d2u(r: float, L: float, b: float) -> float:
    return _load().orc_d2u(r, L, b)


def aziz(r: float, consts: Sequence[float]) -> float:
    a = (C.c_double * 9)(*consts)
    return _load().orc_aziz(r, a)


def log_psi(sys: System, xyz) -> float:
    x = _f64(xyz)
    assert x.shape == (3, sys.N)
    return _load().orc_log_psi(sys.ref, _dp(x))


def pair_sums(sys: System, xyz) -> np.ndarray:
    x = _f64(xyz)
    assert x.shape == (3, sys.N)
    S = np.zeros(sys.N)
    _load().orc_pair_sums(sys.ref, _dp(x), _dp(S))
    return S


def delta_log_psi(sys: System, xyz, s: int, trial) -> float:
    x = _f64(xyz)
    t = _f64(trial)
    return _load().orc_delta_log_psi(sys.ref, _dp(x), int(s), _dp(t))


def grad_lap(sys: System, xyz):
    x = _f64(xyz)
    G = np.zeros((3, sys.N))
    lam = np.zeros(sys.N)
    _load().orc_grad_lap(sys.ref, _dp(x), _dp(G), _dp(lam))
    return G, lam


def init_walkers(sys: System, seed: int, w0: int, W: int, jitter: float) -> np.ndarray:
    """[W][3][N] float64: jittered FCC start (reading R13)."""
    xyz = np.zeros((W, 3, sys.N))
    _load().orc_init_walkers(sys.ref, seed, w0, W, jitter, _dp(xyz))
    return xyz


def sweep(sys: System, xyz: np.ndarray, seed: int, w0: int, t0: int, n_sweeps: int, step: float,
          want_trace: bool = False, force: Optional[np.ndarray] = None):
    """Advance W walkers IN PLACE by n_sweeps sweeps.  xyz: [W][3][N] float64 C-contiguous.
    Returns (n_accepted[W], decisions[W][n_sweeps*N] or None, margins or None)."""
    assert xyz.dtype == np.float64 and xyz.flags.c_contiguous and xyz.shape[1:] == (3, sys.N)
    W = xyz.shape[0]
    moves = n_sweeps * sys.N
    dec = np.zeros((W, moves), np.uint8) if want_trace else None
    mar = np.zeros((W, moves)) if want_trace else None
    nacc = np.zeros(W, np.int64)
    u8p = C.POINTER(C.c_uint8)
    if force is not None:
        force = np.ascontiguousarray(force, np.uint8)
        assert force.shape == (W, moves)
    _load().orc_sweep_walkers(
        sys.ref, _dp(xyz), seed, w0, W, t0, n_sweeps, step,
        dec.ctypes.data_as(u8p) if dec is not None else None,
        _dp(mar) if mar is not None else None,
        force.ctypes.data_as(u8p) if force is not None else None,
        nacc.ctypes.data_as(C.POINTER(C.c_int64)))
    return nacc, dec, mar


def local_energy(sys: System, xyz) -> np.ndarray:
    """[W][6] = E_PB, V, T_PB, T_JF, T_CW (totals, K) and the cutoff guard min|r^2/h^2-1|."""
    x = _f64(xyz)
    if x.ndim == 2:
        x = x[None]
    assert x.shape[1:] == (3, sys.N)
    out = np.zeros((x.shape[0], 6))
    _load().orc_local_energy_walkers(sys.ref, _dp(x), x.shape[0], _dp(out))
    return out


def pair_histogram(sys: System, xyz, nbins: int) -> np.ndarray:
    """[W][nbins] uint32: counts of pair distances r < L/2 in bins of width (L/2)/nbins, per configuration
    (pair distribution function)."""
    x = _f64(xyz)
    if x.ndim == 2:
        x = x[None]
    assert x.shape[1:] == (3, sys.N)
    out = np.zeros((x.shape[0], nbins), np.uint32)
    for w in range(x.shape[0]):
        xw = np.ascontiguousarray(x[w])
        _load().orc_pair_histogram(sys.ref, _dp(xw), nbins, out[w].ctypes.data_as(C.POINTER(C.c_uint32)))
    return out


def normal_pair(w1: int, w2: int):
    """Two standard normals from two 32-bit words (proposal 1's Box-Muller, bit-specified)."""
    z = np.zeros(2)
    _load().orc_normal_pair(w1, w2, _dp(z))
    return float(z[0]), float(z[1])


def move_variates_gauss(seed: int, w: int, t: int, m: int, N: int, step: float):
    """(particle s, delta[3], xi) of move m of sweep t of walker w under proposal 1."""
    d = np.zeros(3)
    xi = C.c_double()
    s = C.c_int32()
    _load().orc_move_variates_gauss(seed, w, t, m, N, step, C.byref(s), _dp(d), C.byref(xi))
    return int(s.value), d, float(xi.value)
