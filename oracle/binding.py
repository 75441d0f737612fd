"""ctypes binding of the CPU oracle (oracle/liboracle.so).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It marshals arguments only; all
arithmetic is in the C++ sources beside it.  Nothing here imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_OMP_PATH = os.path.join(_HERE, "liboracle_omp.so")   # same sources + OpenMP on the outer loops; bit-identical (tests)
_lock = threading.Lock()
_libs = {}

STAGES = ["BC1", "VMEAN", "POT", "DT", "SRC_A", "SRC_B", "SRC_C", "SRC_D", "BC2", "MOM",
          "SWEEP_X", "SWEEP_Y", "SWEEP_Z", "ORB_FRAC", "ORB_SHIFT", "NEWVEL"]
_DP = C.POINTER(C.c_double)


class _Mesh(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("xmin", C.c_double), ("xmax", C.c_double),
                ("yedges", _DP), ("zedges", _DP),
                ("ymin", C.c_double), ("ymax", C.c_double), ("zmin", C.c_double), ("zmax", C.c_double),
                ("bc", (C.c_int * 2) * 3), ("nghost", C.c_int)]


class _Params(C.Structure):
    _fields_ = [("gamma", C.c_double), ("cfl", C.c_double), ("cvnr2", C.c_double), ("nu", C.c_double),
                ("fargo_on", C.c_int),
                ("omega_frame", C.c_double), ("gm_star", C.c_double), ("planet_mass", C.c_double),
                ("planet_r", C.c_double), ("planet_phi0", C.c_double), ("planet_omega", C.c_double),
                ("planet_eps", C.c_double),
                ("shear_c0", C.c_double), ("t_stop", C.c_double), ("dt_fixed", C.c_double),
                ("oort_a", C.c_double)]


def build(force: bool = False) -> str:
    """Compile liboracle.so and liboracle_omp.so with g++ (make) if missing or older than their sources."""
    srcs = [os.path.join(_HERE, f) for f in os.listdir(_HERE) if f.endswith((".cpp", ".hpp", ".h")) or f == "Makefile"]
    for path in (_LIB_PATH, _OMP_PATH):
        stale = force or not os.path.exists(path) or any(os.path.getmtime(s) > os.path.getmtime(path) for s in srcs)
        if stale:
            r = subprocess.run(["make", "-C", _HERE, "-B", os.path.basename(path)], capture_output=True, text=True)
            if r.returncode != 0:
                raise RuntimeError("building %s failed:\n%s%s" % (os.path.basename(path), r.stdout, r.stderr))
    return _LIB_PATH


def lib(omp: bool = False):
    """The one-thread library (the reference of every parity test) or, with omp=True, the OpenMP build of the same
    sources (full-length references at 512^3 and config 4 only)."""
    with _lock:
        if omp not in _libs:
            build()
            L = C.CDLL(_OMP_PATH if omp else _LIB_PATH)
            vp = C.c_void_p
            L.oracle_init.argtypes = [C.POINTER(vp), C.POINTER(_Mesh), C.c_int, C.c_int, C.POINTER(_Params)]
            L.oracle_destroy.argtypes = [vp]
            L.oracle_set_fields.argtypes = [vp] + [_DP] * 5
            L.oracle_get_fields.argtypes = [vp] + [_DP] * 5
            L.oracle_step.argtypes = [vp, C.c_int]
            L.oracle_step_until.argtypes = [vp, C.c_int]
            L.oracle_run_stage.argtypes = [vp, C.c_int]
            L.oracle_set_dt.argtypes = [vp, C.c_double]
            L.oracle_get_time.argtypes = [vp, _DP, _DP, C.POINTER(C.c_longlong)]
            L.oracle_get_array.argtypes = [vp, C.c_char_p, _DP]
            L.oracle_set_array.argtypes = [vp, C.c_char_p, _DP]
            L.oracle_dims.argtypes = [vp] + [C.POINTER(C.c_int)] * 6
            L.oracle_geometry.argtypes = [vp, C.c_int, C.c_int] + [_DP] * 7
            L.oracle_set_planets.argtypes = [vp, C.c_int, _DP, _DP, _DP, _DP, C.c_int, C.c_double]
            L.oracle_get_planets.argtypes = [vp, _DP, _DP, _DP]
            L.oracle_planets_rk5.argtypes = [vp, C.c_double]
            L.oracle_gas_force.argtypes = [vp, C.c_int, _DP]
            L.oracle_set_omega_frame.argtypes = [vp, C.c_double]
            L.oracle_diagnostics.argtypes = [vp, _DP]
            L.oracle_set_bfield.argtypes = [vp, _DP, _DP, _DP, C.c_double, C.c_double, C.c_int]
            L.oracle_get_bfield.argtypes = [vp, _DP, _DP, _DP]
            L.oracle_run_mhd_stage.argtypes = [vp, C.c_int]
            L.oracle_max_divb.argtypes = [vp]
            L.oracle_max_divb.restype = C.c_double
            L.oracle_vanleer_slopes.argtypes = [C.c_int, _DP, _DP, _DP]
            L.oracle_vanleer_slopes.restype = None
            L.oracle_vanleer_star.argtypes = [C.c_int, _DP, _DP, _DP, _DP, C.c_double, _DP]
            L.oracle_vanleer_star.restype = None
            L.oracle_ppa_star.argtypes = [C.c_int, _DP, C.c_double, _DP]
            L.oracle_ppa_star.restype = None
            L.oracle_ppa_interfaces.argtypes = [C.c_int, _DP, _DP, _DP]
            L.oracle_ppa_interfaces.restype = None
            _libs[omp] = L
    return _libs[omp]


def _p(a):
    return None if a is None else a.ctypes.data_as(_DP)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """One oracle context.  `mesh` and `params` are the plain dataclasses of workloads.py
    (any objects with the same attribute names work)."""

    def __init__(self, mesh, geometry: int, eos: int, params, nghost: int = 3, omp: bool = False):
        L = self._L = lib(omp)
        self._ye = _f64(mesh.yedges)
        self._ze = _f64(mesh.zedges)
        m = _Mesh()
        m.nx, m.ny, m.nz = mesh.nx, mesh.ny, mesh.nz
        m.xmin, m.xmax = mesh.xmin, mesh.xmax
        m.yedges, m.zedges = _p(self._ye), _p(self._ze)
        m.ymin, m.ymax = float(self._ye[0]), float(self._ye[-1])
        m.zmin, m.zmax = float(self._ze[0]), float(self._ze[-1])
        for d in range(3):
            for s in range(2):
                m.bc[d][s] = mesh.bc[d][s]
        m.nghost = nghost
        p = _Params()
        for name, _ in _Params._fields_:
            setattr(p, name, getattr(params, name))
        self._h = C.c_void_p()
        rc = L.oracle_init(C.byref(self._h), C.byref(m), geometry, eos, C.byref(p))
        if rc != 0:
            raise ValueError("oracle_init failed (%d)" % rc)
        self.shape = (mesh.nz, mesh.ny, mesh.nx)
        d = [C.c_int() for _ in range(6)]
        L.oracle_dims(self._h, *[C.byref(x) for x in d])
        self.TX, self.TY, self.TZ, self.ngx, self.ngy, self.ngz = [x.value for x in d]

    def close(self):
        if self._h:
            self._L.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_fields(self, rho, e, vx, vy=None, vz=None):
        a = [_f64(x) for x in (rho, e, vx, vy, vz)]
        for x in a:
            assert x is None or x.size == int(np.prod(self.shape))
        if self._L.oracle_set_fields(self._h, *[_p(x) for x in a]) != 0:
            raise ValueError("oracle_set_fields failed")

    def get_fields(self):
        out = [np.empty(self.shape, dtype=np.float64) for _ in range(5)]
        self._L.oracle_get_fields(self._h, *[_p(x) for x in out])
        return tuple(out)

    def step(self, n: int = 1):
        if self._L.oracle_step(self._h, n) != 0:
            raise RuntimeError("oracle_step failed")

    def step_until(self, stage: str):
        if self._L.oracle_step_until(self._h, STAGES.index(stage)) != 0:
            raise RuntimeError("oracle_step_until failed")

    def run_stage(self, stage: str):
        if self._L.oracle_run_stage(self._h, STAGES.index(stage)) != 0:
            raise RuntimeError("oracle_run_stage failed")

    def set_dt(self, dt: float):
        self._L.oracle_set_dt(self._h, float(dt))

    def time(self):
        t, dt, n = C.c_double(), C.c_double(), C.c_longlong()
        self._L.oracle_get_time(self._h, C.byref(t), C.byref(dt), C.byref(n))
        return t.value, dt.value, n.value

    # ---- MHD (NEXT-4; Cartesian meshes) ----
    def set_bfield(self, bx, by, bz, mu0: float = 1.0, eta: float = 0.0, passive: bool = False):
        """Face-centred field, shape (nz, ny, nx) each (bx[k, j, i] on the lower X face of cell (i, j, k)); switches MHD on."""
        b = [_f64(np.broadcast_to(a, self.shape)) for a in (bx, by, bz)]
        if self._L.oracle_set_bfield(self._h, _p(b[0]), _p(b[1]), _p(b[2]), float(mu0), float(eta), 1 if passive else 0) != 0:
            raise ValueError("oracle_set_bfield failed (MHD needs a Cartesian mesh without orbital advection)")

    def get_bfield(self):
        out = [np.empty(self.shape, dtype=np.float64) for _ in range(3)]
        if self._L.oracle_get_bfield(self._h, *[_p(x) for x in out]) != 0:
            raise RuntimeError("no magnetic field set")
        return tuple(out)

    def run_mhd_stage(self, name: str):
        """One MHD substep on the arrays as they stand: BC_B, EMF, TENSION, CT or ORBITAL (cell 11)."""
        if self._L.oracle_run_mhd_stage(self._h, ["BC_B", "EMF", "TENSION", "CT", "ORBITAL"].index(name)) != 0:
            raise RuntimeError("oracle_run_mhd_stage failed")

    def max_divb(self) -> float:
        return float(self._L.oracle_max_divb(self._h))

    # ---- live planets (NEXT-2) ----
    def set_planets(self, gm, eps, pos, vel, force_mode: int = 1, gconst: float = 1.0):
        gm, eps, pos, vel = (_f64(np.atleast_1d(a)).ravel() for a in (gm, eps, pos, vel))
        n = len(gm)
        assert len(eps) == n and len(pos) == 3 * n and len(vel) == 3 * n
        if self._L.oracle_set_planets(self._h, n, _p(gm), _p(eps), _p(pos), _p(vel), force_mode, float(gconst)) != 0:
            raise ValueError("oracle_set_planets failed")
        self._npl = n

    def get_planets(self):
        n = getattr(self, "_npl", 0)
        pos, vel, acc = (np.zeros((n, 3)) for _ in range(3))
        self._L.oracle_get_planets(self._h, _p(pos), _p(vel), _p(acc))
        return pos, vel, acc

    def set_omega_frame(self, omega_new: float):
        if self._L.oracle_set_omega_frame(self._h, float(omega_new)) != 0:
            raise ValueError("oracle_set_omega_frame failed")

    def diagnostics(self):
        """(mass, X, Y, Z momentum of Tab. 2, internal energy): sums over the active cells."""
        out = np.zeros(5)
        if self._L.oracle_diagnostics(self._h, _p(out)) != 0:
            raise RuntimeError("oracle_diagnostics failed")
        return out

    def planets_rk5(self, h: float):
        if self._L.oracle_planets_rk5(self._h, float(h)) != 0:
            raise RuntimeError("oracle_planets_rk5 failed")

    def gas_force(self, p: int = 0):
        F = np.zeros(3)
        if self._L.oracle_gas_force(self._h, p, _p(F)) != 0:
            raise RuntimeError("oracle_gas_force failed")
        return F

    def array(self, name: str) -> np.ndarray:
        """Ghost-inclusive copy of an internal array, shape (TZ, TY, TX) or (TZ, TY) for ring arrays."""
        ring = name in ("v0", "nshift", "xi")
        shape = (self.TZ, self.TY) if ring else (self.TZ, self.TY, self.TX)
        out = np.empty(shape, dtype=np.float64)
        if self._L.oracle_get_array(self._h, name.encode(), _p(out)) != 0:
            raise KeyError(name)
        return out

    def set_array(self, name: str, a):
        a = _f64(a)
        if self._L.oracle_set_array(self._h, name.encode(), _p(a)) != 0:
            raise KeyError(name)

    def active(self, a: np.ndarray) -> np.ndarray:
        nz, ny, nx = self.shape
        return a[self.ngz:self.ngz + nz, self.ngy:self.ngy + ny, self.ngx:self.ngx + nx]

    def geometry(self, j: int, k: int):
        v = [C.c_double() for _ in range(7)]
        if self._L.oracle_geometry(self._h, j, k, *[C.byref(x) for x in v]) != 0:
            raise IndexError((j, k))
        return dict(zip(("sx", "sy", "sz", "invv", "lx", "ly", "lz"), [x.value for x in v]))


# ---- 1-D primitives (pinned to the paper's formulas in tests/) ---------------------------------
def vanleer_slopes(f, invd):
    f, invd = _f64(f), _f64(invd)
    a = np.empty_like(f)
    lib().oracle_vanleer_slopes(len(f), _p(f), _p(invd), _p(a))
    return a


def vanleer_star(f, a, length, w, dt):
    f, a, length, w = _f64(f), _f64(a), _f64(length), _f64(w)
    out = np.empty_like(f)
    lib().oracle_vanleer_star(len(f), _p(f), _p(a), _p(length), _p(w), float(dt), _p(out))
    return out


def ppa_star(f, xi):
    f = _f64(f)
    out = np.empty_like(f)
    lib().oracle_ppa_star(len(f), _p(f), float(xi), _p(out))
    return out


def ppa_interfaces(f):
    f = _f64(f)
    fl, fr = np.empty_like(f), np.empty_like(f)
    lib().oracle_ppa_interfaces(len(f), _p(f), _p(fl), _p(fr))
    return fl, fr
