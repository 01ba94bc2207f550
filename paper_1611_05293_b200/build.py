"""In-tree build of libvfps.so for sm_100a with nvcc (cross-compiles without a GPU)."""
from __future__ import annotations

import glob
import os
import re
import shutil
import subprocess
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_LIB = os.path.join(_HERE, "libvfps.so")
_PEAKS_SRC = os.path.join(_CSRC, "peaks", "vfps_peaks.cu")
_PEAKS_LIB = os.path.join(_HERE, "libvfps_peaks.so")

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC",
    "-Xptxas=-v",            # registers / spills / shared memory per kernel go to build.log
]
# -DVFPS_PHASE_CLOCKS (environment VFPS_PHASE_CLOCKS=1 at build time) compiles the per-phase
# clock stamps of the persistent kernels and the VFPS_PHASE_DUMP host code in; release builds
# leave them out.
_OBJ = os.path.join(_HERE, "build")


def lib_path() -> str:
    """libvfps.so, or the instrumented libvfps_pc.so when VFPS_PHASE_CLOCKS=1 is in the environment."""
    return os.path.join(_HERE, "libvfps_pc.so") if _extra_flags() else _LIB


def _sources():
    return sorted(glob.glob(os.path.join(_CSRC, "*.cu")))


_INC = re.compile(r'^\s*#\s*include\s+"([^"]+)"', re.M)


def _deps(path, seen=None):
    """The file and every header it includes with quotes, recursively."""
    seen = set() if seen is None else seen
    path = os.path.normpath(path)
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    with open(path) as f:
        for inc in _INC.findall(f.read()):
            _deps(os.path.join(os.path.dirname(path), inc), seen)
    return seen


def _extra_flags():
    return ["-DVFPS_PHASE_CLOCKS"] if os.environ.get("VFPS_PHASE_CLOCKS") == "1" else []


def _obj_path(src):
    tag = "_pc" if _extra_flags() else ""
    return os.path.join(_OBJ, os.path.splitext(os.path.basename(src))[0] + tag + ".o")


def _obj_stale(src) -> bool:
    obj = _obj_path(src)
    if not os.path.exists(obj):
        return True
    t = os.path.getmtime(obj)
    return any(os.path.getmtime(d) > t for d in _deps(src))


def _stale() -> bool:
    if not os.path.exists(lib_path()):
        return True
    t = os.path.getmtime(lib_path())
    return any(_obj_stale(s) or os.path.getmtime(_obj_path(s)) > t for s in _sources())


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/*.cu into objects (in parallel, only those whose sources or headers changed)
    and link paper_1611_05293_b200/libvfps.so."""
    if not force and not _stale():
        return lib_path()
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        if os.path.exists(lib_path()):
            return lib_path()          # GPU box without a toolkit: use the library that travelled
        raise RuntimeError("nvcc not found and libvfps.so is missing: cannot build the CUDA library")
    os.makedirs(_OBJ, exist_ok=True)
    todo = [s for s in _sources() if force or _obj_stale(s)]
    logs = {}

    def compile_one(src):
        cmd = [nvcc] + NVCC_FLAGS + _extra_flags() + ["-c", "-o", _obj_path(src), src]
        res = subprocess.run(cmd, capture_output=True, text=True)
        return src, cmd, res

    with ThreadPoolExecutor(max_workers=max(1, min(len(todo), os.cpu_count() or 1))) as pool:
        for src, cmd, res in pool.map(compile_one, todo):
            logs[src] = " ".join(cmd) + "\n" + res.stdout + res.stderr
            if verbose or res.returncode != 0:
                print(logs[src])
            if res.returncode != 0:
                raise RuntimeError("nvcc failed on " + os.path.basename(src) + ":\n" + res.stderr[-4000:])
    for src, text in logs.items():
        with open(_obj_path(src)[:-2] + ".log", "w") as f:
            f.write(text)
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "static",
           "-o", lib_path()] + [_obj_path(s) for s in _sources()]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        print(res.stdout)
        print(res.stderr)
    if res.returncode != 0:
        raise RuntimeError("link failed:\n" + res.stderr[-4000:])
    with open(os.path.join(_HERE, "build_pc.log" if _extra_flags() else "build.log"), "w") as f:      # ptxas -v of every object, current state
        for s in _sources():
            lp = _obj_path(s)[:-2] + ".log"
            if os.path.exists(lp):
                with open(lp) as g:
                    f.write(g.read())
    return lib_path()


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
    cmd = [nvcc] + NVCC_FLAGS + ["-shared", "-cudart", "static", "-o", _PEAKS_LIB, _PEAKS_SRC]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + res.stderr[-4000:])
    return _PEAKS_LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
    print(build_peaks(force=True))
