"""Initial phase-space density psi0 (reading A12 of SURVEY.md section 8(c)).

psi0 = exp(-(q^2/sigma_q^2 + p^2/sigma_p^2)/2) / (2 pi sigma_q sigma_p) + noise * u,
u ~ U[0,1) i.i.d. per cell from a counter-based generator (splitmix64 keyed by
(seed, flat cell index z = N*x + y), top 24 bits), then divided by dq*dp*sum(psi0) in double and
rounded to fp32 ONCE.  Layout [x][y], p (index y) contiguous (z = N_y*x + y).
"""
from __future__ import annotations

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = x + _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def uniform_noise(n_cells: int, seed: int) -> np.ndarray:
    """U[0,1) doubles with 24 random bits, one per flat cell index, reproducible from `seed`."""
    idx = np.arange(n_cells, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.full(1, seed, dtype=np.uint64))[0]
        bits = _splitmix64(idx ^ key)
    return (bits >> np.uint64(40)).astype(np.float64) * (1.0 / (1 << 24))


def grid_axis(N: int, lo: float, hi: float) -> np.ndarray:
    """Nodes lo + i*(hi-lo)/(N-1): both ends are nodes (reading A2)."""
    return lo + np.arange(N, dtype=np.float64) * ((hi - lo) / (N - 1))


def gaussian_psi0(N, q_min, q_max, p_min, p_max, sigma_q=1.0, sigma_p=1.0,
                  q0=0.0, p0=0.0) -> np.ndarray:
    """Un-normalised double Gaussian on the grid, shape [x][y]."""
    q = grid_axis(N, q_min, q_max)[:, None]
    p = grid_axis(N, p_min, p_max)[None, :]
    g = np.exp(-0.5 * (((q - q0) / sigma_q) ** 2 + ((p - p0) / sigma_p) ** 2))
    return g / (2.0 * np.pi * sigma_q * sigma_p)


def make_psi0(N, q_min, q_max, p_min, p_max, sigma_q=1.0, sigma_p=1.0,
              noise=0.0, seed=0, q0=0.0, p0=0.0) -> np.ndarray:
    psi = gaussian_psi0(N, q_min, q_max, p_min, p_max, sigma_q, sigma_p, q0, p0)
    if noise:
        psi = psi + noise * uniform_noise(N * N, seed).reshape(N, N)
    dq = (q_max - q_min) / (N - 1)
    dp = (p_max - p_min) / (N - 1)
    psi = psi / (dq * dp * psi.sum())
    return psi.astype(np.float32)
