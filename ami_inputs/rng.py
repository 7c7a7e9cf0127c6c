"""Stateless counter-based uniform generator (reading P22).

The paper draws its sample points with ``at::rand``.  For a
streamed driver that generates samples on the device, and for tests that must
feed the very same samples to a CPU oracle, a stateless generator is needed:
the value of component ``c`` of sample ``i`` depends only on ``(seed, i, c)``.

Specification (implemented here with numpy and, independently, in the CUDA
driver; the two are compared bit for bit in the tests):

    ctr = i * n_comp + c                                   (uint64)
    z   = seed + 0x9E3779B97F4A7C15 * (ctr + 1)            (mod 2**64)
    z   = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9             (mod 2**64)
    z   = (z ^ (z >> 27)) * 0x94D049BB133111EB             (mod 2**64)
    z   =  z ^ (z >> 31)
    u   = (z >> 11) * 2**-53                               in [0, 1)
    k   = (u - 0.5) * TWO_PI                               in [-pi, pi)

(the 64-bit finaliser is the public-domain splitmix64 mixer).  ``u - 0.5`` is
exact in binary64 and the product is a single correctly rounded multiply, so
the host and device values agree bitwise.
"""
from __future__ import annotations

import math

import numpy as np

SEED_BASE = 20231117  # config i uses SEED_BASE + i
TWO_PI = 2.0 * math.pi

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def uniform01(seed: int, ctr: np.ndarray) -> np.ndarray:
    """u in [0,1) for every 64-bit counter in ``ctr`` (any shape)."""
    ctr = np.asarray(ctr, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + _GOLDEN * (ctr + np.uint64(1))
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def momenta(seed: int, n: int, m: int, start: int = 0, d: int = 2) -> np.ndarray:
    """Internal momenta ``k_int`` of Eq. 8: float64 [n][m*d]
    viewed as [n][m][d], sample ``start + row`` in row ``row``, uniform in
    [-pi, pi)."""
    n_comp = m * d
    i = np.arange(start, start + n, dtype=np.uint64)[:, None]
    c = np.arange(n_comp, dtype=np.uint64)[None, :]
    u = uniform01(seed, i * np.uint64(n_comp) + c)
    return ((u - 0.5) * TWO_PI).reshape(n, m, d)


def energies(seed: int, n: int, n_eps: int, a: float, start: int = 0) -> np.ndarray:
    """Energies drawn directly, uniform in [-a, a): the paper's first example fills ``energy_t`` with
    ``2 a rand - a`` instead of a dispersion.  float64 [n][n_eps], sample
    ``start + row`` in row ``row``; counter = sample * n_eps + symbol."""
    i = np.arange(start, start + n, dtype=np.uint64)[:, None]
    c = np.arange(n_eps, dtype=np.uint64)[None, :]
    u = uniform01(seed, i * np.uint64(n_eps) + c)
    return (2.0 * u - 1.0) * a
