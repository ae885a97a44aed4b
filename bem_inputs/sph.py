"""Orthonormal spherical harmonics with Condon-Shortley phase,
used ONLY to synthesise input densities and the config-3 deformation.  The FMM
in the CUDA path has its own solid-harmonic recurrences; nothing here is shared
with it or with the oracle's arithmetic."""
from __future__ import annotations

import math
import numpy as np


def _assoc_legendre(n: int, m: int, x):
    """P_n^m(x) with Condon-Shortley phase, m >= 0, by upward recurrence in n."""
    x = np.asarray(x, dtype=np.float64)
    pmm = np.ones_like(x)
    if m > 0:
        somx2 = np.sqrt(np.maximum(0.0, (1.0 - x) * (1.0 + x)))
        fact = 1.0
        for _ in range(m):
            pmm = -pmm * fact * somx2
            fact += 2.0
    if n == m:
        return pmm
    pmmp1 = x * (2 * m + 1) * pmm
    if n == m + 1:
        return pmmp1
    pll = pmmp1
    for ll in range(m + 2, n + 1):
        pll = (x * (2 * ll - 1) * pmmp1 - (ll + m - 1) * pmm) / (ll - m)
        pmm, pmmp1 = pmmp1, pll
    return pll


def _norm(n: int, m: int) -> float:
    return math.sqrt((2 * n + 1) / (4 * math.pi) * math.factorial(n - m) / math.factorial(n + m))


def real_sph_harm(n: int, m: int, theta, phi):
    """Re Y_n^m(theta, phi), m >= 0; theta = polar angle, phi = azimuth."""
    return _norm(n, m) * _assoc_legendre(n, m, np.cos(theta)) * np.cos(m * np.asarray(phi))


def real_sph_harm_im(n: int, m: int, theta, phi):
    """Im Y_n^m(theta, phi), m >= 0."""
    return _norm(n, m) * _assoc_legendre(n, m, np.cos(theta)) * np.sin(m * np.asarray(phi))
