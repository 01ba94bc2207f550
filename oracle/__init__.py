"""ctypes loader for the CPU oracle (``vfps_oracle.c``) -- TEST INFRASTRUCTURE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It holds argument marshalling only; every
formula lives in ``vfps_oracle.c`` where it cites the passage of the paper it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vfps_oracle.c")
_LIB = os.path.join(_HERE, "libvfps_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp the oracle into oracle/libvfps_oracle.so (rebuilt if the source is newer)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Params(C.Structure):
    _fields_ = [("N", C.c_int), ("q_min", C.c_double), ("q_max", C.c_double),
                ("p_min", C.c_double), ("p_max", C.c_double), ("steps_per_period", C.c_int),
                ("beta", C.c_double), ("interp_order", C.c_int), ("pad", C.c_int),
                ("renormalise", C.c_int), ("manhattan", C.c_int), ("clamp", C.c_int)]


_dp = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.vfpo_num_threads.restype = C.c_int
        L.vfpo_set_num_threads.argtypes = [C.c_int]
        L.vfpo_lagrange_weights.argtypes = [C.c_int, C.c_double, _dp]
        L.vfpo_rotate.argtypes = [C.c_int] + [C.c_double] * 5 + [C.c_int, _dp, _dp, C.c_int]
        L.vfpo_drift.argtypes = [C.c_int] + [C.c_double] * 5 + [C.c_int, _dp, _dp, C.c_int]
        L.vfpo_rf_kick.argtypes = [C.c_int] + [C.c_double] * 5 + [C.c_int, _dp, _dp, C.c_int]
        L.vfpo_project.argtypes = [C.c_int, C.c_double, _dp, _dp]
        L.vfpo_wake_function.argtypes = [C.c_int, C.c_int, _dp, _dp]
        L.vfpo_wake.argtypes = [C.c_int, _dp, _dp, _dp]
        L.vfpo_kick.argtypes = [C.c_int, C.c_double, C.c_double, C.c_int, _dp, _dp, _dp, C.c_int]
        L.vfpo_fokker_planck.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.vfpo_moments.argtypes = [C.c_int] + [C.c_double] * 4 + [_dp, _dp]
        L.vfpo_csr_power.argtypes = [C.c_int, C.c_int, C.c_double, _dp, _dp]
        L.vfpo_csr_power.restype = C.c_double
        L.vfpo_step.argtypes = [C.POINTER(Params)] + [C.c_void_p] * 6
        L.vfpo_run.argtypes = [C.POINTER(Params), C.c_void_p, _dp, C.c_int, C.c_void_p, C.c_int]
        _lib = L
    return _lib


def num_threads() -> int:
    return lib().vfpo_num_threads()


def set_num_threads(n: int) -> None:
    lib().vfpo_set_num_threads(int(n))


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _z_pairs(Z) -> np.ndarray:
    """complex array [N_f/2+1] -> contiguous (re, im) doubles."""
    Zc = np.ascontiguousarray(np.asarray(Z, dtype=np.complex128))
    return Zc.view(np.float64)


def lagrange_weights(order: int, t: float) -> np.ndarray:
    out = np.zeros(order)
    lib().vfpo_lagrange_weights(order, float(t), out)
    return out


def rotate(psi, q_min, q_max, p_min, p_max, dphi, order, clamp: bool = False) -> np.ndarray:
    psi = _f64(psi)
    out = np.empty_like(psi)
    lib().vfpo_rotate(psi.shape[0], q_min, q_max, p_min, p_max, dphi, order, psi, out, int(clamp))
    return out


def drift(psi, q_min, q_max, p_min, p_max, dphi, order, clamp: bool = False) -> np.ndarray:
    """First half of the Manhattan rotation (L136): psi_A(q, p) = psi(q - dphi p, p)."""
    psi = _f64(psi)
    out = np.empty_like(psi)
    lib().vfpo_drift(psi.shape[0], q_min, q_max, p_min, p_max, dphi, order, psi, out, int(clamp))
    return out


def rf_kick(psi, q_min, q_max, p_min, p_max, dphi, order, clamp: bool = False) -> np.ndarray:
    """Second half of the Manhattan rotation (L136): psi_B(q, p) = psi_A(q, p + dphi q)."""
    psi = _f64(psi)
    out = np.empty_like(psi)
    lib().vfpo_rf_kick(psi.shape[0], q_min, q_max, p_min, p_max, dphi, order, psi, out, int(clamp))
    return out


def project(psi, dp) -> np.ndarray:
    psi = _f64(psi)
    rho = np.empty(psi.shape[0])
    lib().vfpo_project(psi.shape[0], dp, psi, rho)
    return rho


def wake_function(N: int, Nf: int, Z) -> np.ndarray:
    """w[d] for d = -(N-1)..(N-1), stored at index d + N - 1."""
    w = np.empty(2 * N - 1)
    lib().vfpo_wake_function(N, Nf, _z_pairs(Z), w)
    return w


def wake(w, rho) -> np.ndarray:
    rho = _f64(rho)
    V = np.empty_like(rho)
    lib().vfpo_wake(rho.shape[0], _f64(w), rho, V)
    return V


def kick(psi, dp, dphi, order, V, clamp: bool = False) -> np.ndarray:
    psi = _f64(psi)
    out = np.empty_like(psi)
    lib().vfpo_kick(psi.shape[0], dp, dphi, order, _f64(V), psi, out, int(clamp))
    return out


def fokker_planck(psi, p_min, p_max, b) -> np.ndarray:
    psi = _f64(psi)
    out = np.empty_like(psi)
    lib().vfpo_fokker_planck(psi.shape[0], p_min, p_max, b, psi, out)
    return out


def moments(psi, q_min, q_max, p_min, p_max) -> np.ndarray:
    """{M0, <q>, <p>, sigma_q, sigma_p}"""
    psi = _f64(psi)
    out = np.empty(5)
    lib().vfpo_moments(psi.shape[0], q_min, q_max, p_min, p_max, psi, out)
    return out


def csr_power(rho, Nf, dq, Z) -> float:
    rho = _f64(rho)
    return lib().vfpo_csr_power(rho.shape[0], Nf, dq, _z_pairs(Z), rho)


class Oracle:
    """One simulation (one batch member) advanced by the C oracle; state in double."""

    def __init__(self, N, q_min, q_max, p_min, p_max, steps_per_period, beta, interp_order,
                 pad=2, Z: Optional[np.ndarray] = None, renormalise: bool = True, manhattan: bool = False,
                 clamp: bool = False):
        self.P = Params(N, q_min, q_max, p_min, p_max, steps_per_period, beta, interp_order, pad,
                        1 if renormalise else 0, 1 if manhattan else 0, 1 if clamp else 0)
        self.N = N
        self.Z = None if Z is None else _z_pairs(np.asarray(Z).reshape(-1)).copy()
        if self.Z is not None and self.Z.size != 2 * (pad * N // 2 + 1):
            raise ValueError("Z must have pad*N/2+1 entries")
        self.psi = np.zeros((N, N))
        self.steps = 0

    @classmethod
    def from_workload(cls, wl, member: int = 0, renormalise: bool = True, manhattan: bool = False,
                      clamp: bool = False) -> "Oracle":
        Z = wl.impedance([member])
        o = cls(wl.N, wl.q_min, wl.q_max, wl.p_min, wl.p_max, wl.steps_per_period, wl.beta,
                wl.interp_order, wl.pad, None if Z is None else Z[0], renormalise, manhattan, clamp)
        o.set_psi(wl.psi0([member])[0])
        return o

    def set_psi(self, psi) -> None:
        self.psi = _f64(psi).reshape(self.N, self.N).copy()
        self.steps = 0

    def step(self, n: int = 1, diag: bool = True, diag_every: int = 1) -> Optional[np.ndarray]:
        """Advance n steps; returns diag [n][6] = {C, <q>, <p>, sigma_q, sigma_p, P_csr}."""
        d = np.full((n, 6), np.nan) if diag else None
        zp = None if self.Z is None else self.Z.ctypes.data
        lib().vfpo_run(C.byref(self.P), zp, self.psi, n,
                       None if d is None else d.ctypes.data, diag_every)
        self.steps += n
        return d

    def profile(self) -> np.ndarray:
        dp = (self.P.p_max - self.P.p_min) / (self.N - 1)
        return project(self.psi, dp)

    def wake(self) -> np.ndarray:
        if self.Z is None:
            return np.zeros(self.N)
        w = np.empty(2 * self.N - 1)
        lib().vfpo_wake_function(self.N, self.P.pad * self.N, self.Z, w)
        return wake(w, self.profile())

    def moments6(self) -> np.ndarray:
        """{C (current charge), <q>, <p>, sigma_q, sigma_p, P_csr} of the current psi."""
        P = self.P
        m = moments(self.psi, P.q_min, P.q_max, P.p_min, P.p_max)
        out = np.zeros(6)
        out[:5] = m
        if self.Z is not None:
            dq = (P.q_max - P.q_min) / (self.N - 1)
            out[5] = lib().vfpo_csr_power(self.N, P.pad * self.N, dq, self.Z, self.profile())
        return out
