"""Host-side reduction of what the kernels return into the paper's reported quantities: the pair
distribution function g(r) from pair-distance histograms and the error of a
mean of correlated samples by reblocking (l.193, l.321, Ref. [30] Flyvbjerg & Petersen), with the
paper's cost figure t * sigma^2 (l.504-511).  No method arithmetic of the hot path lives here."""
from __future__ import annotations

import math
from typing import Sequence

import numpy as np


def g_of_r(hist, n_atoms: int, box_L: float):
    """hist: [..., nbins] counts of pairs i<j with r < L/2 in bins of width (L/2)/nbins, per configuration
    (leading axes are averaged).  Returns (r_mid[nbins], g[nbins]): g = counts / (pairs an ideal gas of the
    same density would put into the shell) = counts / (N/2 * rho * shell volume)."""
    h = np.asarray(hist, dtype=np.float64)
    nbins = h.shape[-1]
    mean = h.reshape(-1, nbins).mean(0)
    dr = 0.5 * box_L / nbins
    edges = dr * np.arange(nbins + 1)
    shell = 4.0 / 3.0 * math.pi * (edges[1:] ** 3 - edges[:-1] ** 3)
    rho = n_atoms / box_L ** 3
    ideal = 0.5 * n_atoms * rho * shell
    return 0.5 * (edges[1:] + edges[:-1]), mean / ideal


def reblock(series: Sequence[float], min_blocks: int = 16):
    """Standard error of the mean of a correlated series by blocking transformations: halve the series by
    averaging neighbours until fewer than 2*min_blocks values remain; the error estimate is the largest
    sqrt(var / (n - 1)) seen (the plateau, approached from below for positively correlated data).
    Returns (mean, standard_error, tau) with tau = (se / naive_se)^2 / 2 the integrated autocorrelation
    time in samples (1/2 for uncorrelated data; Eq.(13)-(15) l.230-266 use the same quantity)."""
    x = np.asarray(series, dtype=np.float64).ravel()
    n = x.size
    if n < 2:
        raise ValueError("reblock needs at least two samples")
    mean = float(x.mean())
    naive = math.sqrt(float(x.var(ddof=1)) / n)
    best = naive
    y = x
    while y.size >= 2 * min_blocks:
        m = y.size // 2
        y = 0.5 * (y[0:2 * m:2] + y[1:2 * m:2])
        best = max(best, math.sqrt(float(y.var(ddof=1)) / y.size))
    tau = 0.5 * (best / naive) ** 2 if naive > 0 else 0.5
    return mean, best, tau


def seconds_to_error(se_per_atom_K: float, seconds: float, target_K: float = 1e-3):
    """The paper's cost figures (l.504-511): t * sigma^2 in s*mK^2 and the time to reach `target_K` per atom,
    from a run of `seconds` that reached the standard error `se_per_atom_K` (error ~ 1/sqrt(t))."""
    t_sigma2 = seconds * (se_per_atom_K * 1e3) ** 2
    return t_sigma2, seconds * (se_per_atom_K / target_K) ** 2
