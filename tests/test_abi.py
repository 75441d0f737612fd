"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol
include/fargo.h declares, sizes its workspace without a device, validates its arguments, and refuses to
run without a GPU (no CPU fallback).  No compute calls here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_1602_02359_b200 import binding, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _mesh_params(w, precision=64):
    m = binding.FargoMesh()
    ye = np.ascontiguousarray(w.mesh.yedges, dtype=np.float64)
    ze = np.ascontiguousarray(w.mesh.zedges, dtype=np.float64)
    m.nx, m.ny, m.nz = w.mesh.nx, w.mesh.ny, w.mesh.nz
    m.xmin, m.xmax = w.mesh.xmin, w.mesh.xmax
    m.yedges = ye.ctypes.data_as(C.POINTER(C.c_double))
    m.zedges = ze.ctypes.data_as(C.POINTER(C.c_double))
    for d in range(3):
        for s in range(2):
            m.bc[d][s] = w.mesh.bc[d][s]
    p = binding.FargoParams()
    for name in ("gamma", "cfl", "cvnr2", "nu", "fargo_on", "omega_frame", "gm_star", "planet_mass", "planet_r",
                 "planet_phi0", "planet_omega", "planet_eps", "shear_c0", "t_stop", "dt_fixed"):
        setattr(p, name, getattr(w.params, name))
    p.precision = precision
    p.use_graph = 1
    return m, p, (ye, ze)


def test_library_exports_every_declared_symbol():
    L = binding.load()
    header = open(os.path.join(ROOT, "include", "fargo.h")).read()
    declared = sorted(set(re.findall(r"\b(fargo_[a-z_]+)\s*\(", header)))
    assert declared == sorted(binding.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name


def test_library_is_sm100a_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", binding.library_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_workspace_bytes_scales_with_the_mesh_and_precision():
    L = binding.load()
    w = W.noise_box(64)
    m, p, keep = _mesh_params(w)
    b64 = L.fargo_workspace_bytes(C.byref(m), w.geometry, w.eos, C.byref(p))
    narr = 64 * 70 * 70 * 8           # X wrapped: no ghosts; Y, Z: 3 layers per side
    assert 25 * narr <= b64 <= 25 * narr + (1 << 20)
    p.precision = 32
    b32 = L.fargo_workspace_bytes(C.byref(m), w.geometry, w.eos, C.byref(p))
    assert 0.45 * b64 < b32 < 0.55 * b64
    w4 = W.disk3d(1536, 512, 128, nsteps=1) if False else None   # full size is checked on the GPU only
    assert w4 is None


def test_invalid_arguments_are_rejected_without_a_device():
    L = binding.load()
    w = W.noise_box(16)
    m, p, keep = _mesh_params(w)
    assert L.fargo_workspace_bytes(C.byref(m), 7, w.eos, C.byref(p)) == 0
    p.precision = 16
    assert L.fargo_workspace_bytes(C.byref(m), w.geometry, w.eos, C.byref(p)) == 0
    p.precision = 64
    p.fargo_on = 1
    m.bc[0][0] = W.OUTFLOW   # orbital advection needs whole periodic rings
    assert L.fargo_workspace_bytes(C.byref(m), w.geometry, w.eos, C.byref(p)) == 0
    h = C.c_void_p()
    assert L.fargo_init(C.byref(h), C.byref(m), w.geometry, w.eos, C.byref(p)) == -1
    assert not h.value
    assert b"periodic X" in L.fargo_last_error(None)


def test_no_cpu_fallback():
    """Without a CUDA device fargo_init fails with FARGO_ECUDA and the Python class raises."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    L = binding.load()
    w = W.noise_box(16)
    m, p, keep = _mesh_params(w)
    h = C.c_void_p()
    assert L.fargo_init(C.byref(h), C.byref(m), w.geometry, w.eos, C.byref(p)) == -3
    with pytest.raises(RuntimeError):
        binding.Fargo(w.mesh, w.geometry, w.eos, w.params)


def test_product_never_touches_the_oracle():
    """The product package must not import, link or read anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1602_02359_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                code = "\n".join(l for l in text.splitlines() if "oracle" in l and not l.strip().startswith(("//", "#", "*", '"')))
                assert not re.search(r"(import|include|from)\s+[\"<.]*oracle|liboracle", code), (f, code)
