"""ctypes binding of libfargo_b200.so (include/fargo.h): argument marshalling only.

Every step of the hydrodynamic update runs in the CUDA kernels of csrc/; this module allocates the
device workspace as one torch.uint8 tensor, hands over the current torch CUDA stream, and converts
numpy / torch arrays to pointers.  There is no CPU fallback: without the built library or without a
CUDA device, construction raises.  Nothing here imports oracle/.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from . import build as _build

_DP = C.POINTER(C.c_double)
STAGES = ["BC1", "VMEAN", "POT", "DT", "SRC_A", "SRC_B", "SRC_C", "SRC_D", "BC2", "MOM",
          "SWEEP_X", "SWEEP_Y", "SWEEP_Z", "ORB_FRAC", "ORB_SHIFT", "NEWVEL"]
EXPORTS = ["fargo_workspace_bytes", "fargo_init", "fargo_destroy", "fargo_set_fields", "fargo_get_fields",
           "fargo_step", "fargo_get_time", "fargo_kernel_launches", "fargo_step_until", "fargo_dims",
           "fargo_get_array", "fargo_last_error", "fargo_profile", "fargo_profile_report", "fargo_selftest_div",
           "fargo_set_planets", "fargo_get_planets", "fargo_set_omega_frame", "fargo_diagnostics", "fargo_diagnostics_noalloc",
           "fargo_update_phase", "fargo_halo_bytes", "fargo_halo", "fargo_dt_device_ptr", "fargo_set_bfield", "fargo_get_bfield", "fargo_dt_min_with"]


class FargoMesh(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("xmin", C.c_double), ("xmax", C.c_double),
                ("yedges", _DP), ("zedges", _DP),
                ("ymin", C.c_double), ("ymax", C.c_double), ("zmin", C.c_double), ("zmax", C.c_double),
                ("bc", (C.c_int * 2) * 3)]


class FargoParams(C.Structure):
    _fields_ = [("gamma", C.c_double), ("cfl", C.c_double), ("cvnr2", C.c_double), ("nu", C.c_double),
                ("fargo_on", C.c_int),
                ("omega_frame", C.c_double), ("gm_star", C.c_double), ("planet_mass", C.c_double),
                ("planet_r", C.c_double), ("planet_phi0", C.c_double), ("planet_omega", C.c_double),
                ("planet_eps", C.c_double),
                ("shear_c0", C.c_double), ("t_stop", C.c_double), ("dt_fixed", C.c_double), ("oort_a", C.c_double),
                ("precision", C.c_int), ("use_graph", C.c_int), ("mhd", C.c_int), ("kernel_plan", C.c_int),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t), ("cuda_stream", C.c_void_p)]


PLAN_UNFUSED_SOURCE, PLAN_UNFUSED_VISC, PLAN_UNFUSED_DT, PLAN_SEAM_ABOVE = 1, 2, 4, 8   # fargo_params.kernel_plan flags (include/fargo.h)

_lib = None


def library_path() -> str:
    return _build.LIB


def load():
    """Load (building first if the sources are newer) the C-ABI library and declare its signatures."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.build()
    L = C.CDLL(path)
    vp = C.c_void_p
    L.fargo_workspace_bytes.argtypes = [C.POINTER(FargoMesh), C.c_int, C.c_int, C.POINTER(FargoParams)]
    L.fargo_workspace_bytes.restype = C.c_size_t
    L.fargo_init.argtypes = [C.POINTER(vp), C.POINTER(FargoMesh), C.c_int, C.c_int, C.POINTER(FargoParams)]
    L.fargo_destroy.argtypes = [vp]
    L.fargo_set_fields.argtypes = [vp] + [vp] * 5
    L.fargo_get_fields.argtypes = [vp] + [vp] * 5
    L.fargo_step.argtypes = [vp, C.c_int]
    L.fargo_get_time.argtypes = [vp, _DP, _DP, C.POINTER(C.c_longlong)]
    L.fargo_kernel_launches.argtypes = [vp]
    L.fargo_kernel_launches.restype = C.c_longlong
    L.fargo_step_until.argtypes = [vp, C.c_int]
    L.fargo_dims.argtypes = [vp] + [C.POINTER(C.c_int)] * 6
    L.fargo_get_array.argtypes = [vp, C.c_char_p, vp]
    L.fargo_profile.argtypes = [vp, C.c_int]
    L.fargo_profile_report.argtypes = [vp, C.c_char_p, C.c_size_t]
    L.fargo_last_error.argtypes = [vp]
    L.fargo_set_planets.argtypes = [vp, C.c_int, _DP, _DP, _DP, _DP, C.c_int, C.c_double]
    L.fargo_get_planets.argtypes = [vp, _DP, _DP, _DP]
    L.fargo_set_omega_frame.argtypes = [vp, C.c_double]
    L.fargo_diagnostics.argtypes = [vp, _DP]
    L.fargo_diagnostics_noalloc.argtypes = [vp, vp]
    L.fargo_set_bfield.argtypes = [vp, vp, vp, vp, C.c_double, C.c_double, C.c_int]
    L.fargo_get_bfield.argtypes = [vp, vp, vp, vp]
    L.fargo_update_phase.argtypes = [vp, C.c_int]
    L.fargo_halo_bytes.argtypes = [vp, C.c_int, C.c_int]
    L.fargo_halo_bytes.restype = C.c_size_t
    L.fargo_halo.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, vp]
    L.fargo_dt_min_with.argtypes = [vp, vp]
    L.fargo_dt_device_ptr.argtypes = [vp]
    L.fargo_dt_device_ptr.restype = vp
    L.fargo_selftest_div.argtypes = [vp, vp, vp, C.c_longlong, vp]
    L.fargo_selftest_div.restype = C.c_int
    L.fargo_last_error.restype = C.c_char_p
    _lib = L
    return L


def _ptr(a) -> Optional[int]:
    """Raw address of a numpy array (host) or a torch tensor (host or device); None passes through."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return a.ctypes.data
    return a.data_ptr()


class Fargo:
    """One simulation context on the current CUDA device.

    `mesh` / `params` are the plain dataclasses of workloads.py (any objects with the same attributes).
    """

    def __init__(self, mesh, geometry: int, eos: int, params, precision: int = 64, use_graph: bool = True,
                 device: Optional[str] = None, kernel_plan: int = 0, mhd: bool = False, guard_bytes: int = 0):
        import torch
        L = load()
        if not torch.cuda.is_available():
            raise RuntimeError("fargo_b200 needs a CUDA device (there is no CPU fallback)")
        self._torch = torch
        self.device = torch.device(device or "cuda:%d" % torch.cuda.current_device())
        self.dtype = np.float64 if precision == 64 else np.float32
        self.tdtype = torch.float64 if precision == 64 else torch.float32
        self._ye = np.ascontiguousarray(mesh.yedges, dtype=np.float64)
        ext = getattr(mesh, "yedges_ext", None)
        if ext is not None:   # a slab: the neighbours' edges beyond the cut faces travel with the active ones
            self._ye = np.ascontiguousarray(np.concatenate([np.asarray(a, dtype=np.float64) for a in (ext[0], mesh.yedges, ext[1])
                                                            if a is not None]))
        self._ze = np.ascontiguousarray(mesh.zedges, dtype=np.float64)
        zext = getattr(mesh, "zedges_ext", None)
        if zext is not None:
            self._ze = np.ascontiguousarray(np.concatenate([np.asarray(a, dtype=np.float64) for a in (zext[0], mesh.zedges, zext[1])
                                                            if a is not None]))
        m = FargoMesh()
        m.nx, m.ny, m.nz = mesh.nx, mesh.ny, mesh.nz
        m.xmin, m.xmax = mesh.xmin, mesh.xmax
        m.yedges = self._ye.ctypes.data_as(_DP)
        m.zedges = self._ze.ctypes.data_as(_DP)
        m.ymin, m.ymax = float(mesh.yedges[0]), float(mesh.yedges[-1])
        m.zmin, m.zmax = float(mesh.zedges[0]), float(mesh.zedges[-1])
        for d in range(3):
            for s in range(2):
                m.bc[d][s] = mesh.bc[d][s]
        p = FargoParams()
        for name in ("gamma", "cfl", "cvnr2", "nu", "fargo_on", "omega_frame", "gm_star", "planet_mass", "planet_r",
                     "planet_phi0", "planet_omega", "planet_eps", "shear_c0", "t_stop", "dt_fixed", "oort_a"):
            setattr(p, name, getattr(params, name))
        p.precision = precision
        p.use_graph = 1 if use_graph else 0
        p.mhd = 1 if mhd else 0            # reserve the arrays of the MHD substeps (NEXT-4); set_bfield switches them on
        p.kernel_plan = int(kernel_plan)   # PLAN_* flags: the unfused kernel sequences (measurements, tests)
        nbytes = L.fargo_workspace_bytes(C.byref(m), geometry, eos, C.byref(p))
        if nbytes == 0:
            raise ValueError("fargo_workspace_bytes rejected the mesh / parameters")
        with torch.cuda.device(self.device):
            self.stream = torch.cuda.current_stream(self.device)
            if self.stream.cuda_stream == 0:
                # the legacy default stream cannot be captured into a CUDA graph: give the context its own
                self.stream = torch.cuda.Stream(self.device)
                torch.cuda.current_stream(self.device).synchronize()
            # guard_bytes > 0: a canary region before and after the workspace (check_guards(); compute-sanitizer is closed
            # on this pool, so out-of-bounds writes next to the workspace are looked for this way)
            self._guard = (int(guard_bytes) + 255) // 256 * 256
            with torch.cuda.stream(self.stream):   # the caching allocator ties the block to the stream that uses it
                self.workspace = torch.empty(nbytes + 256 + 2 * self._guard, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr() + self._guard
            off = (-base) % 256
            self._ws_off, self._ws_len = self._guard + off, nbytes
            if self._guard:   # (a torch fill, on request only: no library kernel runs on the default path)
                with torch.cuda.stream(self.stream):
                    self.workspace[:self._ws_off].fill_(0xA5)
                    self.workspace[self._ws_off + nbytes:].fill_(0xA5)
            p.workspace = base + off
            p.workspace_bytes = nbytes
            p.cuda_stream = self.stream.cuda_stream
            self._h = C.c_void_p()
            rc = L.fargo_init(C.byref(self._h), C.byref(m), geometry, eos, C.byref(p))
        if rc != 0:
            raise RuntimeError("fargo_init failed (%d): %s" % (rc, L.fargo_last_error(None).decode()))
        self.mesh_bc_y, self.mesh_bc_z = tuple(mesh.bc[1]), tuple(mesh.bc[2])
        self.shape = (mesh.nz, mesh.ny, mesh.nx)
        self.ncells = mesh.nx * mesh.ny * mesh.nz
        self.hasy, self.hasz = mesh.ny > 1, mesh.nz > 1
        d = [C.c_int() for _ in range(6)]
        L.fargo_dims(self._h, *[C.byref(x) for x in d])
        self.TX, self.TY, self.TZ, self.ngx, self.ngy, self.ngz = [x.value for x in d]

    # -- lifetime ------------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None):
            self.stream.synchronize()   # queued kernels still use the workspace
            load().fargo_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def check_guards(self) -> bool:
        """True when no byte of the canary regions around the workspace (guard_bytes) was written."""
        assert self._guard > 0, "the context was created without guard_bytes"
        self.stream.synchronize()
        lo = self.workspace[:self._ws_off]                      # the guard and the alignment slack before the workspace
        hi = self.workspace[self._ws_off + self._ws_len:]       # everything after it
        return bool((lo == 0xA5).all().item()) and bool((hi == 0xA5).all().item())

    def _check(self, rc, what):
        if rc != 0:
            raise RuntimeError("%s failed (%d): %s" % (what, rc, load().fargo_last_error(self._h).decode()))

    # -- the four calls of the north star ---------------------------------------------------------
    def set_fields(self, rho, e, vx, vy=None, vz=None):
        """Host numpy arrays or torch tensors (host or device) of the context's precision, shape (nz, ny, nx)."""
        arrs = []
        for a in (rho, e, vx, vy, vz):
            if isinstance(a, np.ndarray):
                a = np.ascontiguousarray(a, dtype=self.dtype)
            elif a is not None:
                a = a.to(self.tdtype).contiguous()
            if a is not None:
                n = a.size if isinstance(a, np.ndarray) else a.numel()
                assert n == self.ncells, "field size does not match the mesh"
            arrs.append(a)
        self._keep = arrs
        with self._torch.cuda.device(self.device):
            self._torch.cuda.current_stream(self.device).synchronize()   # device inputs made on another stream
            self._check(load().fargo_set_fields(self._h, *[_ptr(a) for a in arrs]), "fargo_set_fields")

    def step(self, n: int = 1):
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_step(self._h, int(n)), "fargo_step")

    def get_fields(self, out=None):
        """Returns (rho, e, vx, vy, vz) as host numpy arrays, or fills `out` (5 arrays / tensors / None)."""
        if out is None:
            out = [np.empty(self.shape, dtype=self.dtype) for _ in range(5)]
            if not self.hasy:
                out[3][...] = 0
            if not self.hasz:
                out[4][...] = 0
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_get_fields(self._h, *[_ptr(a) for a in out]), "fargo_get_fields")
        return tuple(out)

    def time(self):
        t, dt, n = C.c_double(), C.c_double(), C.c_longlong()
        self._check(load().fargo_get_time(self._h, C.byref(t), C.byref(dt), C.byref(n)), "fargo_get_time")
        return t.value, dt.value, n.value

    # -- slab decomposition in Y (NEXT-3; driven by slabs.SlabRun) -------------------------------------
    def update_phase(self, phase: int):
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_update_phase(self._h, phase), "fargo_update_phase")

    def halo_bytes(self, which: int, direction: int = 1) -> int:
        return int(load().fargo_halo_bytes(self._h, which, direction))

    def halo(self, which: int, direction: int, side: int, pack: bool, buf):
        """buf: a contiguous CUDA uint8 tensor of halo_bytes(which, direction) bytes on this context's device."""
        assert buf.is_cuda and buf.is_contiguous() and buf.numel() * buf.element_size() >= self.halo_bytes(which, direction)
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_halo(self._h, which, direction, side, 1 if pack else 0, buf.data_ptr()), "fargo_halo")

    def dt_device_ptr(self) -> int:
        return int(load().fargo_dt_device_ptr(self._h))

    def dt_min_with(self, other: "Fargo"):
        """dt <- min(dt, other's dt): one tiny kernel on this context's stream (sub-domains on one device)."""
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_dt_min_with(self._h, other.dt_device_ptr()), "fargo_dt_min_with")

    def dt_tensor(self):
        """The device-resident time step as a 1-element float64 tensor VIEW (for an in-place all-reduce)."""
        ptr = load().fargo_dt_device_ptr(self._h)

        class _View:
            __cuda_array_interface__ = {"shape": (1,), "typestr": "<f8", "data": (int(ptr), False), "version": 2}
        return self._torch.as_tensor(_View(), device=self.device)

    # -- MHD (NEXT-4; the context must have been created with mhd=True) ---------------------------------------
    def set_bfield(self, bx, by, bz, mu0: float = 1.0, eta: float = 0.0, passive: bool = False):
        """Face-centred field, shape (nz, ny, nx) each (bx[k, j, i] on the lower X face of cell (i, j, k))."""
        arrs = []
        for a in (bx, by, bz):
            if isinstance(a, np.ndarray) or np.isscalar(a):
                a = np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=self.dtype), self.shape))
            else:
                a = a.to(self.tdtype).contiguous()
            arrs.append(a)
        self._keep_b = arrs
        with self._torch.cuda.device(self.device):
            self._torch.cuda.current_stream(self.device).synchronize()
            self._check(load().fargo_set_bfield(self._h, *[_ptr(a) for a in arrs], float(mu0), float(eta), 1 if passive else 0),
                        "fargo_set_bfield")

    def get_bfield(self):
        out = [np.empty(self.shape, dtype=self.dtype) for _ in range(3)]
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_get_bfield(self._h, *[_ptr(a) for a in out]), "fargo_get_bfield")
        return tuple(out)

    # -- live planets (NEXT-2) ------------------------------------------------------------------------
    def set_planets(self, gm, eps, pos, vel, force_mode: int = 1, gconst: float = 1.0):
        a = [np.ascontiguousarray(np.atleast_1d(x), dtype=np.float64).ravel() for x in (gm, eps, pos, vel)]
        n = len(a[0])
        if len(a[1]) != n or len(a[2]) != 3 * n or len(a[3]) != 3 * n:
            raise ValueError("gm, eps need n entries, pos and vel 3 n")
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_set_planets(self._h, n, *[x.ctypes.data_as(_DP) for x in a], force_mode, float(gconst)),
                        "fargo_set_planets")
        self._npl = n

    def diagnostics(self):
        """(mass, X, Y, Z momentum of Tab. 2, internal energy): sums over the active cells, reduced on the device."""
        out = np.zeros(5)
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_diagnostics(self._h, out.ctypes.data_as(_DP)), "fargo_diagnostics")
        return out

    def diagnostics_noalloc(self, out):
        """fargo_diagnostics_noalloc: the same five sums into `out` (a CUDA float64 tensor of 5 elements on this device),
        asynchronously on the context's stream; allocates nothing (ny * nz <= 524288).  Returns `out`."""
        t = self._torch
        if not (isinstance(out, t.Tensor) and out.is_cuda and out.dtype == t.float64 and out.numel() >= 5 and out.is_contiguous()):
            raise ValueError("out: a contiguous CUDA float64 tensor of at least 5 elements")
        with t.cuda.device(self.device):
            self._check(load().fargo_diagnostics_noalloc(self._h, C.c_void_p(out.data_ptr())), "fargo_diagnostics_noalloc")
        return out

    def set_omega_frame(self, omega_new: float):
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_set_omega_frame(self._h, float(omega_new)), "fargo_set_omega_frame")

    def get_planets(self):
        n = getattr(self, "_npl", 0)
        pos, vel, acc = (np.zeros((n, 3)) for _ in range(3))
        with self._torch.cuda.device(self.device):
            rc = load().fargo_get_planets(self._h, *[x.ctypes.data_as(_DP) for x in (pos, vel, acc)])
        if rc < 0:
            self._check(rc, "fargo_get_planets")
        return pos, vel, acc

    def kernel_launches(self) -> int:
        return int(load().fargo_kernel_launches(self._h))

    # -- measurement -------------------------------------------------------------------------------
    def profile(self, enable: bool = True):
        self._check(load().fargo_profile(self._h, 1 if enable else 0), "fargo_profile")

    def profile_report(self) -> dict:
        """{launcher name: (kernel launches, total ms)} since profile(True), CUDA-event timed on the stream."""
        buf = C.create_string_buffer(1 << 14)
        self._check(load().fargo_profile_report(self._h, buf, len(buf)), "fargo_profile_report")
        out = {}
        for line in buf.value.decode().splitlines():
            name, n, ms = line.split()
            out[name] = (int(n), float(ms))
        return out

    # -- inspection ----------------------------------------------------------------------------------
    def step_until(self, stage: str):
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_step_until(self._h, STAGES.index(stage)), "fargo_step_until")

    def array(self, name: str) -> np.ndarray:
        ring = name in ("v0", "nshift")
        out = np.empty((self.TZ, self.TY) if ring else (self.TZ, self.TY, self.TX), dtype=self.dtype)
        with self._torch.cuda.device(self.device):
            self._check(load().fargo_get_array(self._h, name.encode(), out.ctypes.data), "fargo_get_array")
        return out


def selftest_div(a, b=None):
    """out = rdiv(a, b) elementwise on the GPU (torch.float64 CUDA tensors): the kernels' division; b = None
    selects their division by the constant six (rdiv6)."""
    import torch
    assert a.is_cuda and a.dtype == torch.float64
    a = a.contiguous()
    if b is not None:
        assert b.is_cuda and b.dtype == torch.float64 and a.numel() == b.numel()
        b = b.contiguous()
    out = torch.empty_like(a)
    torch.cuda.synchronize()
    rc = load().fargo_selftest_div(a.data_ptr(), None if b is None else b.data_ptr(), out.data_ptr(), a.numel(), None)
    if rc != 0:
        raise RuntimeError("fargo_selftest_div failed with code %d" % rc)
    return out
