"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle and the CUDA library and therefore holds
none of the method's arithmetic: it only builds meshes, parameter dictionaries
and initial fields (numpy, fp64).  Neither `oracle/` nor the CUDA path contains
a random generator; the counter-based deviate below is the only one.

Array layout everywhere: shape (nz, ny, nx), X (index i) fastest, ACTIVE cells
only.  Staggered velocities live on the LOWER face of the cell in their own
direction (Eqs. 49-50 at PAPER.md:345-350).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

# geometry / eos / bc codes: must match include/fargo.h and oracle/fargo_oracle.h
CARTESIAN, CYLINDRICAL, SPHERICAL, SHEARING_SHEET = 0, 1, 2, 3
ISOTHERMAL, ADIABATIC = 0, 1
PERIODIC, OUTFLOW, REFLECTING = 0, 1, 2

SEED = 160202359


@dataclasses.dataclass
class Mesh:
    nx: int
    ny: int
    nz: int
    xmin: float
    xmax: float
    yedges: np.ndarray  # ny+1 active edges
    zedges: np.ndarray  # nz+1 active edges
    bc: tuple = ((PERIODIC, PERIODIC), (PERIODIC, PERIODIC), (PERIODIC, PERIODIC))
    zedges_ext: Optional[tuple] = None   # sub-domains only: the same for cut Z faces
    yedges_ext: Optional[tuple] = None   # slabs only: (3 edges beyond a cut lower Y face or None, 3 beyond a cut upper face or None)

    @property
    def dx(self) -> float:
        return (self.xmax - self.xmin) / self.nx

    @property
    def ncells(self) -> int:
        return self.nx * self.ny * self.nz

    def xc(self):
        return self.xmin + (np.arange(self.nx) + 0.5) * self.dx

    def xf(self):
        return self.xmin + np.arange(self.nx) * self.dx

    def yc(self):
        return 0.5 * (self.yedges[:-1] + self.yedges[1:])

    def zc(self):
        return 0.5 * (self.zedges[:-1] + self.zedges[1:])


@dataclasses.dataclass
class Params:
    gamma: float = 1.4
    cfl: float = 0.44
    cvnr2: float = 2.0          # C_q^2 of the von Neumann-Richtmyer viscosity (reading G8)
    nu: float = 0.0
    fargo_on: int = 0
    omega_frame: float = 0.0
    gm_star: float = 0.0
    planet_mass: float = 0.0    # G*m_p
    planet_r: float = 1.0
    planet_phi0: float = 0.0
    planet_omega: float = 0.0
    planet_eps: float = 0.0
    shear_c0: float = 0.5
    t_stop: float = 0.0         # <= 0: none
    dt_fixed: float = 0.0       # <= 0: CFL
    oort_a: float = 0.0         # Oort constant A of Eq. 29 (shearing sheet only; Keplerian -0.75 Omega_f)


@dataclasses.dataclass
class Workload:
    name: str
    mesh: Mesh
    geometry: int
    eos: int
    params: Params
    rho: np.ndarray
    e: np.ndarray               # internal energy density, or c_s when isothermal
    vx: np.ndarray
    vy: Optional[np.ndarray]
    vz: Optional[np.ndarray]
    nsteps: int
    planets: Optional[dict] = None   # live planets (NEXT-2): keyword arguments of set_planets, or None
    bfield: Optional[dict] = None    # MHD (NEXT-4): keyword arguments of set_bfield (bx, by, bz, mu0, eta, passive), or None

    def fields(self):
        return self.rho, self.e, self.vx, self.vy, self.vz


def uedges(lo: float, hi: float, n: int) -> np.ndarray:
    """Uniform edges lo + j*(hi-lo)/n, j = 0..n (same formula on both sides)."""
    return lo + np.arange(n + 1, dtype=np.float64) * ((hi - lo) / n)


# ---------------------------------------------------------------- deviates ---
_M64 = (1 << 64) - 1


def _splitmix64(x: np.ndarray) -> np.ndarray:
    x = (x + np.uint64(0x9E3779B97F4A7C15))
    z = x
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def uniform_pm1(field: int, n: int, seed: int = SEED, chunk: int = 1 << 24) -> np.ndarray:
    """U(seed, field, m) in [-1, 1), m = 0..n-1 (linear active-cell index, i fastest).

    U = 2 * (splitmix64(seed ^ (field << 56) ^ m) >> 11) * 2^-53 - 1
    """
    out = np.empty(n, dtype=np.float64)
    base = np.uint64((seed ^ (field << 56)) & _M64)
    with np.errstate(over="ignore"):
        for s in range(0, n, chunk):
            m = np.arange(s, min(n, s + chunk), dtype=np.uint64)
            bits = _splitmix64(base ^ m) >> np.uint64(11)
            out[s:s + len(m)] = 2.0 * (bits.astype(np.float64) * (2.0 ** -53)) - 1.0
    return out


# ----------------------------------------------------------------- configs ---
def sound_wave(n: int = 32, amp: float = 1e-6, nsteps: int = 200) -> Workload:
    """Config 1: linear sound wave along (1,1,1) in a periodic Cartesian box."""
    gamma = 1.4
    mesh = Mesh(n, n, n, 0.0, 1.0, uedges(0.0, 1.0, n), uedges(0.0, 1.0, n))
    xc, yc, zc = mesh.xc(), mesh.yc(), mesh.zc()
    xf, yf, zf = mesh.xf(), mesh.yedges[:-1], mesh.zedges[:-1]
    two_pi = 2.0 * math.pi

    def psi(x, y, z):
        return two_pi * (x[None, None, :] + y[None, :, None] + z[:, None, None])

    rho0, p0, c = 1.0, 1.0 / gamma, 1.0
    cpsi = np.cos(psi(xc, yc, zc))
    rho = rho0 * (1.0 + amp * cpsi)
    p = p0 + c * c * rho0 * amp * cpsi
    e = p / (gamma - 1.0)
    a = amp * c / math.sqrt(3.0)
    vx = a * np.cos(psi(xf, yc, zc))
    vy = a * np.cos(psi(xc, yf, zc))
    vz = a * np.cos(psi(xc, yc, zf))
    return Workload("sound_wave_%d" % n, mesh, CARTESIAN, ADIABATIC, Params(gamma=gamma),
                    rho, e, vx, vy, vz, nsteps)


def sod(nx: int = 512, nyz: int = 4, t_stop: float = 0.2) -> Workload:
    """Config 2: Sod shock tube along X, outflow in X, periodic in Y and Z."""
    gamma = 1.4
    w = nyz / nx
    bc = ((OUTFLOW, OUTFLOW), (PERIODIC, PERIODIC), (PERIODIC, PERIODIC))
    mesh = Mesh(nx, nyz, nyz, 0.0, 1.0, uedges(0.0, w, nyz), uedges(0.0, w, nyz), bc)
    left = (mesh.xc() < 0.5)[None, None, :]
    shape = (nyz, nyz, nx)
    rho = np.where(left, 1.0, 0.125) * np.ones(shape)
    p = np.where(left, 1.0, 0.1) * np.ones(shape)
    e = p / (gamma - 1.0)
    z = np.zeros(shape)
    return Workload("sod_%d" % nx, mesh, CARTESIAN, ADIABATIC,
                    Params(gamma=gamma, t_stop=t_stop), rho, e, z.copy(), z.copy(), z.copy(), 2000)


def _disk_params(nu: float) -> Params:
    h = 0.05
    return Params(gamma=1.4, nu=nu, fargo_on=1, omega_frame=1.0, gm_star=1.0, planet_mass=1e-3,
                  planet_r=1.0, planet_phi0=0.0, planet_omega=1.0, planet_eps=0.6 * h * 1.0)


def disk2d(nphi: int = 768, nr: int = 256, nsteps: int = 500) -> Workload:
    """Config 3: 2-D cylindrical locally isothermal disk, FARGO on, nu = 1e-5, planet q = 1e-3."""
    h = 0.05
    bc = ((PERIODIC, PERIODIC), (REFLECTING, REFLECTING), (PERIODIC, PERIODIC))
    mesh = Mesh(nphi, nr, 1, -math.pi, math.pi, uedges(0.4, 2.5, nr), np.array([-0.5, 0.5]), bc)
    prm = _disk_params(1e-5)
    n = mesh.ncells
    shape = (1, nr, nphi)
    rc = mesh.yc()[None, :, None] * np.ones(shape)
    rf = mesh.yedges[:-1][None, :, None] * np.ones(shape)
    rho = rc ** -0.5
    cs = h * rc ** -0.5
    vphi = rc ** -0.5 * math.sqrt(1.0 - 1.5 * h * h) - rc * prm.omega_frame
    vx = vphi + 1e-4 * cs * uniform_pm1(2, n).reshape(shape)
    vy = 1e-4 * (h * rf ** -0.5) * uniform_pm1(3, n).reshape(shape)
    return Workload("disk2d_%dx%d" % (nphi, nr), mesh, CYLINDRICAL, ISOTHERMAL, prm,
                    rho, cs, vx, vy, None, nsteps)


def disk3d(nphi: int = 1536, nr: int = 512, nth: int = 128, nsteps: int = 100) -> Workload:
    """Config 4: 3-D spherical locally isothermal disk, FARGO on, planet q = 1e-3, nu = 0."""
    h = 0.05
    bc = ((PERIODIC, PERIODIC), (REFLECTING, REFLECTING), (REFLECTING, REFLECTING))
    mesh = Mesh(nphi, nr, nth, -math.pi, math.pi, uedges(0.4, 2.5, nr),
                uedges(0.5 * math.pi - 0.15, 0.5 * math.pi + 0.15, nth), bc)
    prm = _disk_params(0.0)
    n = mesh.ncells
    shape = (nth, nr, nphi)
    r = mesh.yc()[None, :, None]
    th = mesh.zc()[:, None, None]
    R = r * np.sin(th)
    z = r * np.cos(th)
    H = h * R
    ones = np.ones(shape)
    rho = (R ** -1.5 * np.exp(-z * z / (2.0 * H * H))) * ones
    cs = (h * R ** -0.5) * ones
    vx = (R ** -0.5 * math.sqrt(1.0 - 2.5 * h * h) - R * prm.omega_frame) * ones
    vx = vx + 1e-4 * cs * uniform_pm1(2, n).reshape(shape)
    vy = 1e-4 * cs * uniform_pm1(3, n).reshape(shape)
    vz = 1e-4 * cs * uniform_pm1(4, n).reshape(shape)
    return Workload("disk3d_%dx%dx%d" % (nphi, nr, nth), mesh, SPHERICAL, ISOTHERMAL, prm,
                    rho, cs, vx, vy, vz, nsteps)


def sheet3d(nx: int = 1024, ny: int = 512, nz: int = 128, nsteps: int = 20) -> Workload:
    """NEXT-1 workload (no BASELINE.json config): 3-D adiabatic Keplerian shearing sheet (Tab. 1, Eqs. 28-30),
    X along the flow (periodic, 4 H long), Y along the shear (2 H, reflecting walls), Z periodic (H/2); Omega_f = 1,
    A = -3/4, c_s = H Omega_f = 1 so that lengths are in scale heights; v_x = 2 A y plus noise of 1e-2 c_s on the three
    components, rho = 1 + 0.01 U; orbital advection on."""
    gamma, om, A = 5.0 / 3.0, 1.0, -0.75
    bc = ((PERIODIC, PERIODIC), (REFLECTING, REFLECTING), (PERIODIC, PERIODIC))
    mesh = Mesh(nx, ny, nz, -2.0, 2.0, uedges(-1.0, 1.0, ny), uedges(-0.25, 0.25, nz), bc)
    prm = Params(gamma=gamma, fargo_on=1, omega_frame=om, oort_a=A)
    n = mesh.ncells
    shape = (nz, ny, nx)
    rho = (1.0 + 0.01 * uniform_pm1(0, n)).reshape(shape)
    e = rho / (gamma * (gamma - 1.0))                       # c_s^2 = gamma P / rho = 1
    vx = 2.0 * A * mesh.yc()[None, :, None] * np.ones(shape) + 1e-2 * uniform_pm1(2, n).reshape(shape)
    vy = 1e-2 * uniform_pm1(3, n).reshape(shape)
    vz = 1e-2 * uniform_pm1(4, n).reshape(shape)
    return Workload("sheet3d_%dx%dx%d" % (nx, ny, nz), mesh, SHEARING_SHEET, ADIABATIC, prm, rho, e, vx, vy, vz, nsteps)


def disk3d_live(nphi: int = 1536, nr: int = 512, nth: int = 128, nsteps: int = 100) -> Workload:
    """NEXT-2 workload (no BASELINE.json config): config 4 with its planet LIVE (section 3.8): same mass, softening and
    starting point (r, phi) = (1, 0), at rest in the corotating frame, feeling the gas by direct summation."""
    w = disk3d(nphi, nr, nth, nsteps)
    w.name = w.name.replace("disk3d", "disk3d_live")
    w.planets = dict(gm=[w.params.planet_mass], eps=[w.params.planet_eps], pos=[w.params.planet_r, 0.0, 0.0],
                     vel=[0.0, 0.0, 0.0], force_mode=1, gconst=1.0)
    return w


def noise_box(n: int = 64, nsteps: int = 50, shape3: Optional[tuple] = None) -> Workload:
    """Config 5: periodic Cartesian box with cell-scale white noise, gamma = 5/3."""
    gamma = 5.0 / 3.0
    nx, ny, nz = shape3 if shape3 is not None else (n, n, n)
    mesh = Mesh(nx, ny, nz, 0.0, 1.0, uedges(0.0, ny / nx, ny), uedges(0.0, nz / nx, nz))
    m = mesh.ncells
    shape = (nz, ny, nx)
    rho = (1.0 + 0.01 * uniform_pm1(0, m)).reshape(shape)
    e = np.full(shape, 1.0 / (gamma - 1.0))
    vx = (0.1 * uniform_pm1(2, m)).reshape(shape)
    vy = (0.1 * uniform_pm1(3, m)).reshape(shape)
    vz = (0.1 * uniform_pm1(4, m)).reshape(shape)
    return Workload("noise_box_%dx%dx%d" % (nx, ny, nz), mesh, CARTESIAN, ADIABATIC,
                    Params(gamma=gamma), rho, e, vx, vy, vz, nsteps)


def mhd_box(n: int = 64, nsteps: int = 20, shape3: Optional[tuple] = None) -> Workload:
    """NEXT-4: the noise box of config 5 threaded by a magnetic field: a uniform field (0.3, -0.2, 0.1) plus the discrete
    curl of a seeded edge-centred vector potential (divergence-free to rounding), |B| ~ 0.4, beta ~ 10."""
    w = noise_box(n, nsteps, shape3)
    m = w.mesh
    shape = (m.nz, m.ny, m.nx)
    dx, dy, dz = m.dx, float(m.yedges[1] - m.yedges[0]), float(m.zedges[1] - m.zedges[0])
    ax, ay, az = (0.02 * min(dx, dy, dz) * 8.0 * uniform_pm1(5 + f, m.ncells).reshape(shape) for f in range(3))
    up = lambda a, axis: np.roll(a, -1, axis=axis)
    bx = 0.3 + (up(az, 1) - az) / dy - (up(ay, 0) - ay) / dz
    by = -0.2 + (up(ax, 0) - ax) / dz - (up(az, 2) - az) / dx
    bz = 0.1 + (up(ay, 2) - ay) / dx - (up(ax, 1) - ax) / dy
    w.name = w.name.replace("noise_box", "mhd_box")
    w.bfield = dict(bx=bx, by=by, bz=bz, mu0=1.0, eta=0.0, passive=False)
    return w
