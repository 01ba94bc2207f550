"""ctypes binding of libvfps.so with the same names as include/vfps.h.

``Simulation`` wraps one ``vfps_handle``.  Device arrays are ``torch`` CUDA tensors (used for
their memory and stream only); the ``*_host`` methods take / return numpy arrays and go through
the library's host-pointer entry points.  No arithmetic of the method happens here.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional

import numpy as np

from .build import build, lib_path

ENGINE_AUTO, ENGINE_STREAM, ENGINE_GRAPH, ENGINE_CLUSTER, ENGINE_GRID = 0, 1, 2, 3, 4
WAKE_AUTO, WAKE_FFT, WAKE_DIRECT = 0, 1, 2
OPT_ENGINE, OPT_WAKE, OPT_TIMING, OPT_CLUSTER_SIZE, OPT_CLUSTER_KERNEL, OPT_GRID_KERNEL = 1, 2, 3, 4, 5, 6
NUM_KERNELS = 7
FLAG_RENORMALISE, FLAG_CLAMP, FLAG_ROT_MANHATTAN = 1, 2, 4

# every symbol include/vfps.h declares (tests check the library exports each of them)
EXPORTS = [
    "vfps_create", "vfps_create_host", "vfps_destroy", "vfps_set_option", "vfps_get_option",
    "vfps_set_impedance", "vfps_set_impedance_host",
    "vfps_set_psi", "vfps_set_psi_host", "vfps_step", "vfps_step_host",
    "vfps_get_psi", "vfps_get_psi_host", "vfps_get_profile", "vfps_get_profile_host",
    "vfps_get_wake", "vfps_get_wake_host", "vfps_get_moments", "vfps_get_moments_host",
    "vfps_step_count", "vfps_launch_count", "vfps_engine_name", "vfps_wake_name",
    "vfps_kernel_time", "vfps_reset_kernel_times", "vfps_kernel_name",
    "vfps_last_error", "vfps_version",
    "vfps_wake_noalloc", "vfps_noalloc_last_error",
]
NOALLOC_MAX_N = 4096      # VFPS_NOALLOC_MAX_N of include/vfps.h


class VfpsError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"vfps error {code}: {text}")
        self.code = code


class VfpsParams(C.Structure):
    _fields_ = [("N", C.c_int), ("q_min", C.c_double), ("q_max", C.c_double),
                ("p_min", C.c_double), ("p_max", C.c_double), ("steps_per_period", C.c_int),
                ("beta", C.c_double), ("interp_order", C.c_int), ("pad", C.c_int),
                ("members", C.c_int), ("flags", C.c_int)]


_lib = None


def load():
    """Build (if stale) and load libvfps.so; raises if that is impossible -- no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = C.CDLL(lib_path())
    vp, ip = C.c_void_p, C.c_int
    L.vfps_create.argtypes = [C.POINTER(VfpsParams), vp, vp, C.POINTER(vp)]
    L.vfps_create_host.argtypes = [C.POINTER(VfpsParams), vp, vp, C.POINTER(vp)]
    L.vfps_destroy.argtypes = [vp]
    L.vfps_set_option.argtypes = [vp, ip, ip]
    L.vfps_get_option.argtypes = [vp, ip, C.POINTER(ip)]
    for name in ("vfps_set_impedance", "vfps_set_impedance_host",
                 "vfps_set_psi", "vfps_set_psi_host", "vfps_get_psi", "vfps_get_psi_host",
                 "vfps_get_profile", "vfps_get_profile_host", "vfps_get_wake", "vfps_get_wake_host",
                 "vfps_get_moments", "vfps_get_moments_host"):
        getattr(L, name).argtypes = [vp, vp]
    L.vfps_step.argtypes = [vp, ip, vp]
    L.vfps_step_host.argtypes = [vp, ip, vp]
    L.vfps_step_count.argtypes = [vp, C.POINTER(C.c_longlong)]
    L.vfps_launch_count.argtypes = [vp, C.POINTER(C.c_longlong)]
    L.vfps_kernel_time.argtypes = [vp, ip, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
    L.vfps_reset_kernel_times.argtypes = [vp]
    L.vfps_kernel_name.argtypes = [ip]
    L.vfps_wake_noalloc.argtypes = [ip, ip, vp, vp, vp, vp]
    L.vfps_noalloc_last_error.argtypes = []
    strings = ("vfps_engine_name", "vfps_wake_name", "vfps_last_error", "vfps_version", "vfps_kernel_name",
               "vfps_noalloc_last_error")
    for name in EXPORTS:
        getattr(L, name).restype = C.c_char_p if name in strings else C.c_int
    for name in strings[:3]:
        getattr(L, name).argtypes = [vp]
    _lib = L
    return L


def version() -> str:
    return load().vfps_version().decode()


def _dev_ptr(t, dtype_name: str, numel: int, what: str) -> int:
    import torch
    want = getattr(torch, dtype_name)
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == want and t.is_contiguous()):
        raise TypeError(f"{what}: need a contiguous CUDA tensor of dtype {dtype_name}")
    if t.numel() != numel:
        raise ValueError(f"{what}: expected {numel} elements, got {t.numel()}")
    return t.data_ptr()


def wake_noalloc(N: int, pad: int, Z, rho, V_out, stream=None) -> None:
    """vfps_wake_noalloc (include/vfps.h): V_out[x] = sum_x' w[x - x'] rho[x'], w = Re IDFT(Z), with no device
    allocation -- the wake function lives in a 32 KB array built into the library (N <= NOALLOC_MAX_N).
    Z: complex64 CUDA tensor of N*pad/2 + 1 values; rho, V_out: float32 CUDA tensors of N values (V_out is written).
    stream: a torch.cuda.Stream, default the current one.  Calls that overlap on the GPU race on the built-in array."""
    import torch
    L = load()
    nz = (N * pad) // 2 + 1 if N > 0 and pad > 0 else 0
    zp = None if Z is None else _dev_ptr(Z, "complex64", nz, "Z")
    rp = None if rho is None else _dev_ptr(rho, "float32", N, "rho")
    vo = None if V_out is None else _dev_ptr(V_out, "float32", N, "V_out")
    st = (stream if stream is not None else torch.cuda.current_stream()).cuda_stream
    rc = L.vfps_wake_noalloc(int(N), int(pad), zp, rp, vo, st)
    if rc != 0:
        raise VfpsError(rc, L.vfps_noalloc_last_error().decode())


def _host_arr(a, dtype, numel: int, what: str) -> np.ndarray:
    arr = np.ascontiguousarray(a, dtype=dtype)
    if arr.size != numel:
        raise ValueError(f"{what}: expected {numel} elements, got {arr.size}")
    return arr


class Simulation:
    """One vfps_handle.  Z: None, a CUDA complex64 tensor or a host complex64 array
    [members][pad*N/2+1]."""

    def __init__(self, N, q_min, q_max, p_min, p_max, steps_per_period, beta, interp_order=4,
                 pad=2, members=1, flags=FLAG_RENORMALISE, Z=None, stream=None, device=None):
        import torch
        self._L = load()
        self._h = C.c_void_p()
        if not torch.cuda.is_available():
            raise VfpsError(-3, "no CUDA device: vfps has no CPU fallback")
        self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
        torch.cuda.set_device(self.device)
        self.P = VfpsParams(N, q_min, q_max, p_min, p_max, steps_per_period, beta, interp_order, pad,
                            members, flags)
        self.N, self.members, self.Nf = N, members, N * pad
        self.stream = stream
        sp = C.c_void_p(stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream)
        self._stream_ptr = sp
        nz = members * (self.Nf // 2 + 1)
        if Z is None:
            rc = self._L.vfps_create(C.byref(self.P), None, sp, C.byref(self._h))
        elif isinstance(Z, torch.Tensor):
            zp = _dev_ptr(Z, "complex64", nz, "Z")
            rc = self._L.vfps_create(C.byref(self.P), C.c_void_p(zp), sp, C.byref(self._h))
        else:
            zh = _host_arr(Z, np.complex64, nz, "Z")
            rc = self._L.vfps_create_host(C.byref(self.P), zh.ctypes.data_as(C.c_void_p), sp, C.byref(self._h))
        if rc != 0:
            raise VfpsError(rc, self._L.vfps_last_error(None).decode())

    @classmethod
    def from_workload(cls, wl, members=None, **kw) -> "Simulation":
        idx = list(range(wl.members) if members is None else members)
        sim = cls(wl.N, wl.q_min, wl.q_max, wl.p_min, wl.p_max, wl.steps_per_period, wl.beta,
                  wl.interp_order, wl.pad, len(idx), Z=wl.impedance(idx), **kw)
        sim.set_psi_host(wl.psi0(idx))
        return sim

    # ---------------------------------------------------------------- plumbing
    def _check(self, rc: int) -> None:
        if rc != 0:
            raise VfpsError(rc, self._L.vfps_last_error(self._h).decode())

    def close(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            self._L.vfps_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _new(self, *shape):
        import torch
        return torch.empty(*shape, dtype=torch.float32, device=self.device)

    # ---------------------------------------------------------------- options / info
    def set_option(self, option: int, value: int) -> None:
        self._check(self._L.vfps_set_option(self._h, option, value))

    def set_engine(self, engine: int) -> None:
        self.set_option(OPT_ENGINE, engine)

    def set_wake_mode(self, mode: int) -> None:
        self.set_option(OPT_WAKE, mode)

    def get_option(self, option: int) -> int:
        v = C.c_int()
        self._check(self._L.vfps_get_option(self._h, option, C.byref(v)))
        return v.value

    def set_cluster_size(self, size: int) -> None:
        self.set_option(OPT_CLUSTER_SIZE, size)

    @property
    def cluster_size(self) -> int:
        return self.get_option(OPT_CLUSTER_SIZE)

    def set_cluster_kernel(self, version: int) -> None:
        self.set_option(OPT_CLUSTER_KERNEL, version)

    @property
    def cluster_kernel(self) -> int:
        return self.get_option(OPT_CLUSTER_KERNEL)

    def set_grid_kernel(self, version: int) -> None:
        self.set_option(OPT_GRID_KERNEL, version)

    @property
    def grid_kernel(self) -> int:
        return self.get_option(OPT_GRID_KERNEL)

    @property
    def engine_name(self) -> str:
        return self._L.vfps_engine_name(self._h).decode()

    @property
    def wake_name(self) -> str:
        return self._L.vfps_wake_name(self._h).decode()

    def step_count(self) -> int:
        v = C.c_longlong()
        self._check(self._L.vfps_step_count(self._h, C.byref(v)))
        return v.value

    def kernel_times(self) -> dict:
        """{kernel name: (total ms, launches bracketed)} accumulated while OPT_TIMING is on."""
        out = {}
        for k in range(NUM_KERNELS):
            ms, cnt = C.c_double(), C.c_longlong()
            self._check(self._L.vfps_kernel_time(self._h, k, C.byref(ms), C.byref(cnt)))
            out[self._L.vfps_kernel_name(k).decode()] = (ms.value, cnt.value)
        return out

    def reset_kernel_times(self) -> None:
        self._check(self._L.vfps_reset_kernel_times(self._h))

    def launch_count(self) -> int:
        v = C.c_longlong()
        self._check(self._L.vfps_launch_count(self._h, C.byref(v)))
        return v.value

    # ---------------------------------------------------------------- device-pointer calls
    def set_psi(self, psi) -> None:
        self._check(self._L.vfps_set_psi(self._h, _dev_ptr(psi, "float32", self.members * self.N * self.N, "psi")))

    def step(self, n: int = 1, diag=None) -> None:
        dp = None if diag is None else _dev_ptr(diag, "float32", n * self.members * 6, "diag")
        self._check(self._L.vfps_step(self._h, int(n), dp))

    def get_psi(self, out=None):
        out = self._new(self.members, self.N, self.N) if out is None else out
        self._check(self._L.vfps_get_psi(self._h, _dev_ptr(out, "float32", self.members * self.N * self.N, "psi_out")))
        return out

    def get_profile(self, out=None):
        out = self._new(self.members, self.N) if out is None else out
        self._check(self._L.vfps_get_profile(self._h, _dev_ptr(out, "float32", self.members * self.N, "rho_out")))
        return out

    def get_wake(self, out=None):
        out = self._new(self.members, self.N) if out is None else out
        self._check(self._L.vfps_get_wake(self._h, _dev_ptr(out, "float32", self.members * self.N, "V_out")))
        return out

    def get_moments(self, out=None):
        out = self._new(self.members, 6) if out is None else out
        self._check(self._L.vfps_get_moments(self._h, _dev_ptr(out, "float32", self.members * 6, "out")))
        return out

    # ---------------------------------------------------------------- host-pointer calls
    def set_impedance_host(self, Z) -> None:
        """New impedance [members][Nf/2+1] for the running simulation (adiabatic current scan)."""
        zh = _host_arr(Z, np.complex64, self.members * (self.Nf // 2 + 1), "Z")
        self._check(self._L.vfps_set_impedance_host(self._h, zh.ctypes.data_as(C.c_void_p)))

    def set_psi_host(self, psi) -> None:
        a = _host_arr(psi, np.float32, self.members * self.N * self.N, "psi")
        self._check(self._L.vfps_set_psi_host(self._h, a.ctypes.data_as(C.c_void_p)))

    def step_host(self, n: int = 1, diag: bool = True) -> Optional[np.ndarray]:
        d = np.empty((n, self.members, 6), dtype=np.float32) if diag else None
        self._check(self._L.vfps_step_host(self._h, int(n), None if d is None else d.ctypes.data_as(C.c_void_p)))
        return d

    def _get_host(self, fn, *shape) -> np.ndarray:
        out = np.empty(shape, dtype=np.float32)
        self._check(fn(self._h, out.ctypes.data_as(C.c_void_p)))
        return out

    def get_psi_host(self) -> np.ndarray:
        return self._get_host(self._L.vfps_get_psi_host, self.members, self.N, self.N)

    def get_profile_host(self) -> np.ndarray:
        return self._get_host(self._L.vfps_get_profile_host, self.members, self.N)

    def get_wake_host(self) -> np.ndarray:
        return self._get_host(self._L.vfps_get_wake_host, self.members, self.N)

    def get_moments_host(self) -> np.ndarray:
        return self._get_host(self._L.vfps_get_moments_host, self.members, 6)
