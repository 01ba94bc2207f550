"""paper_1611_05293_b200 -- thin Python binding of the vfps C-ABI library (include/vfps.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of
``csrc/``.  PyTorch supplies device memory and streams.  There is no CPU fallback: if the
shared library cannot be built or loaded, importing symbols from it raises.
"""
from .build import build, build_peaks, lib_path
from .binding import (
    ENGINE_AUTO, ENGINE_STREAM, ENGINE_GRAPH, ENGINE_CLUSTER, ENGINE_GRID,
    WAKE_AUTO, WAKE_FFT, WAKE_DIRECT, OPT_ENGINE, OPT_WAKE, OPT_TIMING, OPT_CLUSTER_SIZE,
    OPT_CLUSTER_KERNEL, OPT_GRID_KERNEL,
    FLAG_RENORMALISE, FLAG_CLAMP, FLAG_ROT_MANHATTAN,
    VfpsError, VfpsParams, Simulation, load, version, EXPORTS, wake_noalloc, NOALLOC_MAX_N,
)

__all__ = [
    "build", "build_peaks", "lib_path", "load", "version", "EXPORTS",
    "ENGINE_AUTO", "ENGINE_STREAM", "ENGINE_GRAPH", "ENGINE_CLUSTER", "ENGINE_GRID",
    "WAKE_AUTO", "WAKE_FFT", "WAKE_DIRECT", "OPT_ENGINE", "OPT_WAKE", "OPT_TIMING", "OPT_CLUSTER_SIZE",
    "OPT_CLUSTER_KERNEL", "OPT_GRID_KERNEL",
    "FLAG_RENORMALISE", "FLAG_CLAMP", "FLAG_ROT_MANHATTAN",
    "VfpsError", "VfpsParams", "Simulation", "wake_noalloc", "NOALLOC_MAX_N",
]
