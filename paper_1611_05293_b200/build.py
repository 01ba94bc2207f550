"""In-tree build of libvfps.so for sm_100a with nvcc (cross-compiles without a GPU)."""
from __future__ import annotations

import glob
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_LIB = os.path.join(_HERE, "libvfps.so")
_PEAKS_SRC = os.path.join(_CSRC, "peaks", "vfps_peaks.cu")
_PEAKS_LIB = os.path.join(_HERE, "libvfps_peaks.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared",
    "-Xptxas=-v",            # registers / spills / shared memory per kernel go to build.log
    "-cudart", "static",
]


def lib_path() -> str:
    return _LIB


def _sources():
    return sorted(glob.glob(os.path.join(_CSRC, "*.cu")))


def _stale() -> bool:
    if not os.path.exists(_LIB):
        return True
    t = os.path.getmtime(_LIB)
    deps = _sources() + glob.glob(os.path.join(_CSRC, "*.cuh")) + \
        glob.glob(os.path.join(_HERE, "..", "include", "*.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu into paper_1611_05293_b200/libvfps.so (rebuilt when a source is newer)."""
    if not force and not _stale():
        return _LIB
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        if os.path.exists(_LIB):
            return _LIB          # GPU box without a toolkit: use the library that travelled
        raise RuntimeError("nvcc not found and libvfps.so is missing: cannot build the CUDA library")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", _LIB] + _sources()
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stderr[-4000:])
    with open(os.path.join(_HERE, "build.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    return _LIB


def build_peaks(force: bool = False) -> str:
    """Compile the measurement harness csrc/peaks/vfps_peaks.cu into libvfps_peaks.so (its own
    library: nothing of it is linked into libvfps.so)."""
    if not force and os.path.exists(_PEAKS_LIB) and os.path.getmtime(_PEAKS_LIB) >= os.path.getmtime(_PEAKS_SRC):
        return _PEAKS_LIB
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        if os.path.exists(_PEAKS_LIB):
            return _PEAKS_LIB
        raise RuntimeError("nvcc not found and libvfps_peaks.so is missing")
    cmd = [nvcc] + NVCC_FLAGS + ["-o", _PEAKS_LIB, _PEAKS_SRC]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stderr[-4000:])
    return _PEAKS_LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
    print(build_peaks(force=True))
