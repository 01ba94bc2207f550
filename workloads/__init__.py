"""Seeded synthetic inputs for the Vlasov-Fokker-Planck step (shared by oracle and CUDA path).

This module holds NONE of the method's per-step arithmetic (no rotation, interpolation, wake,
kick, Fokker-Planck or moments).  It only builds what the C-ABI boundary takes as *inputs*:

* the parameter sets of BASELINE.json's five configs (C0..C4);
* the initial density psi0 (Gaussian + seeded uniform noise, reading A12), rounded to fp32 once;
* the impedance array Z_k (free-space CSR, Eq. 6; parallel-plates shielded CSR,
  PAPER.md L69-79 Eq. 7-8) in the normalisation of reading A5, rounded to complex fp32 once.

Both consumers (``oracle/`` and the CUDA library) receive the *same fp32 arrays*.
"""
from .configs import CONFIGS, Workload, get_workload
from .psi0 import gaussian_psi0, uniform_noise, make_psi0
from .impedance import (
    zhat_free_space,
    zhat_parallel_plates,
    kappa_grid,
    make_impedance,
)

__all__ = [
    "CONFIGS",
    "Workload",
    "get_workload",
    "gaussian_psi0",
    "uniform_noise",
    "make_psi0",
    "zhat_free_space",
    "zhat_parallel_plates",
    "kappa_grid",
    "make_impedance",
]
