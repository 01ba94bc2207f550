"""CSR impedance arrays Z_k handed to the library (reading A5 of SURVEY.md section 8(c)).

The library never sees Pi or S_csr, only Z.  Dimensionless wavenumber kappa = k * sigma_z0.

* free space (Eq. 6):
      Zhat_fs(kappa) = Gamma(2/3) * 3^(-1/3) * (sqrt(3)/2 + i/2) * kappa^(1/3)
* parallel plates (Eq. 7-8, "j" read as i, p = 0,1,2,...):
      Zhat_pp(kappa; Pi) = 2 pi^2 2^(1/3) Pi^(2/3) kappa^(-1/3)
                           * sum_p [ Ai'(u_p) Ci'(u_p) + u_p Ai(u_p) Ci(u_p) ],  Ci = Ai - i Bi,
      u_p = pi^2 (2p+1)^2 2^(-8/3) (Pi/kappa)^(4/3)
* discretisation: Z_k = 4 pi S_csr Zhat(kappa_k), kappa_k = 2 pi k / (N_f dq), Z_0 = 0 (PAPER.md
  L65: Z -> 0 for f -> 0), Z_{N_f/2} <- its real part (Hermitian spectrum of a real wake).

Numerics: Ai'Bi' + u Ai Bi cancels to relative u^-3, and Ai, Bi over/underflow
for large u.  The exponentially scaled Airy functions make the products Ai*Bi and Ai'*Bi' exact
(the scale factors cancel) and Ai^2-type terms a plain exp(-4/3 u^1.5) underflow; beyond u = 300
the imaginary summand is replaced by its leading asymptote -3/(16 pi u^(5/2)) ... derived from
Ai Bi ~ 1/(2 pi sqrt(u)) (1 + 5/(32 u^3)), Ai'Bi' ~ -sqrt(u)/(2 pi) (1 - 7/(32 u^3)).
This is set-up cost (host, double, once per run), never per step.
"""
from __future__ import annotations

import numpy as np
from scipy.special import airye, gamma

_U_EXACT_MAX = 300.0


def zhat_free_space(kappa) -> np.ndarray:
    kappa = np.asarray(kappa, dtype=np.float64)
    pref = gamma(2.0 / 3.0) * 3.0 ** (-1.0 / 3.0)
    return pref * (np.sqrt(3.0) / 2.0 + 0.5j) * np.cbrt(kappa)


def _summand(u: np.ndarray) -> np.ndarray:
    """Ai'(u) Ci'(u) + u Ai(u) Ci(u) for u > 0, complex."""
    u = np.asarray(u, dtype=np.float64)
    out = np.zeros(u.shape, dtype=np.complex128)
    small = u <= _U_EXACT_MAX
    if np.any(small):
        us = u[small]
        eai, eaip, ebi, ebip = airye(us)           # eai = Ai e^{+zeta}, ebi = Bi e^{-zeta}
        zeta = (2.0 / 3.0) * us ** 1.5
        damp = np.exp(-2.0 * zeta)
        re = (eaip * eaip + us * eai * eai) * damp  # Ai'^2 + u Ai^2
        im = -(eaip * ebip + us * eai * ebi)        # -(Ai'Bi' + u Ai Bi); scale factors cancel
        out[small] = re + 1j * im
    big = ~small
    if np.any(big):
        out[big] = -1j * 3.0 / (16.0 * np.pi * u[big] ** 2.5)
    return out


def zhat_parallel_plates(kappa, Pi: float, rtol: float = 1e-13, p_max: int = 2_000_000) -> np.ndarray:
    """Zhat_pp(kappa; Pi) for kappa > 0 (array), summing p until the tail is below rtol."""
    kappa = np.atleast_1d(np.asarray(kappa, dtype=np.float64))
    out = np.empty(kappa.shape, dtype=np.complex128)
    c_u = np.pi ** 2 * 2.0 ** (-8.0 / 3.0)
    for i, k in enumerate(kappa):
        scale = c_u * (Pi / k) ** (4.0 / 3.0)
        total = 0.0 + 0.0j
        p0 = 0
        block = 4096
        while p0 < p_max:
            p = np.arange(p0, p0 + block, dtype=np.float64)
            terms = _summand(scale * (2.0 * p + 1.0) ** 2)
            total += terms.sum()
            p0 += block
            # remaining tail of the ~ (2p+1)^-5 series, bounded by the integral of the asymptote
            u_last = scale * (2.0 * p0 + 1.0) ** 2
            tail = 3.0 / (16.0 * np.pi) * u_last ** -2.5 * (2.0 * p0 + 1.0) / 8.0
            if u_last > _U_EXACT_MAX and tail <= rtol * abs(total):
                break
        pref = 2.0 * np.pi ** 2 * 2.0 ** (1.0 / 3.0) * Pi ** (2.0 / 3.0) * k ** (-1.0 / 3.0)
        out[i] = pref * total
    return out


def kappa_grid(N: int, pad: int, dq: float) -> np.ndarray:
    """kappa_k = 2 pi k / (N_f dq), k = 0 .. N_f/2."""
    Nf = pad * N
    return 2.0 * np.pi * np.arange(Nf // 2 + 1, dtype=np.float64) / (Nf * dq)


def make_impedance(N: int, pad: int, dq: float, S_csr: float, Pi=None,
                   dtype=np.complex64) -> np.ndarray:
    """Z_k = 4 pi S_csr Zhat(kappa_k), k = 0..N_f/2; Pi=None -> free space, else parallel plates."""
    kap = kappa_grid(N, pad, dq)
    Z = np.zeros(kap.shape, dtype=np.complex128)
    if Pi is None:
        Z[1:] = zhat_free_space(kap[1:])
    else:
        Z[1:] = zhat_parallel_plates(kap[1:], Pi)
    Z *= 4.0 * np.pi * S_csr
    Z[0] = 0.0
    Z[-1] = Z[-1].real
    return Z.astype(dtype)
