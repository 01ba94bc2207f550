"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, and exports every
symbol include/vfps.h declares; the binding's struct matches the header; and without a GPU the
product path fails loudly instead of falling back."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    text = open(os.path.join(ROOT, "include", "vfps.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vfps_[a-z_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol(vfps):
    lib = ctypes.CDLL(vfps.lib_path())
    syms = header_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(lib, s), f"libvfps.so does not export {s}"
    assert sorted(vfps.EXPORTS) == syms          # the binding covers the whole header


def test_params_struct_matches_header(vfps):
    text = open(os.path.join(ROOT, "include", "vfps.h")).read()
    body = re.search(r"typedef struct vfps_params \{(.*?)\} vfps_params;", text, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        ctype, names = decl.split(None, 1)
        for n in names.split(","):
            fields.append((n.strip(), ctype))
    want = [(n, {ctypes.c_int: "int", ctypes.c_double: "double"}[t]) for n, t in vfps.VfpsParams._fields_]
    assert fields == want


def test_version_and_error_strings_without_gpu(vfps):
    L = vfps.load()
    assert b"sm_100a" in L.vfps_version()
    h = ctypes.c_void_p()
    P = vfps.VfpsParams(7, -6, 6, -6, 6, 100, 1e-3, 4, 2, 1, 1)
    assert L.vfps_create(ctypes.byref(P), None, None, ctypes.byref(h)) == -1      # VFPS_ERR_ARG
    assert b"N must be" in L.vfps_last_error(None)
    P = vfps.VfpsParams(8192, -6, 6, -6, 6, 100000, 1e-3, 4, 2, 1, 1)
    assert L.vfps_create(ctypes.byref(P), None, None, ctypes.byref(h)) == -5      # UNSUPPORTED (FFT length)
    P = vfps.VfpsParams(64, -6, 6, -6, 6, 100, 1e-3, 4, 2, 1, 1 | 64)
    assert L.vfps_create(ctypes.byref(P), None, None, ctypes.byref(h)) == -1      # unknown flag
    assert L.vfps_destroy(None) == 0


def test_no_cpu_fallback(vfps):
    """Without a CUDA device create must fail with VFPS_ERR_CUDA -- never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    L = vfps.load()
    h = ctypes.c_void_p()
    P = vfps.VfpsParams(64, -6, 6, -6, 6, 100, 1e-3, 4, 2, 1, 1)
    assert L.vfps_create(ctypes.byref(P), None, None, ctypes.byref(h)) == -3
    assert not h.value
    with pytest.raises(vfps.VfpsError):
        vfps.Simulation(64, -6, 6, -6, 6, 100, 1e-3)


def test_product_does_not_import_oracle():
    """The product path and the oracle share no code and never import each other."""
    pkg = os.path.join(ROOT, "paper_1611_05293_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f"{f} mentions the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1611_05293_b200" not in src and "libvfps.so" not in src
