"""Small seeded workloads for the GPU parity tests: every geometry / EOS / boundary kind / dimension
combination the hot path supports, at sizes the CPU oracle finishes in seconds and that span several
kernel tiles plus a ragged tail.  No method arithmetic here (inputs only)."""
import math

import numpy as np

from paper_1602_02359_b200 import workloads as W

P, O, R = W.PERIODIC, W.OUTFLOW, W.REFLECTING


def _noise(shape, field, amp, seed=7):
    n = int(np.prod(shape))
    return amp * W.uniform_pm1(field, n, seed=seed).reshape(shape)


def cart_adi_periodic(nx=37, ny=29, nz=11, nsteps=6):
    w = W.noise_box(shape3=(nx, ny, nz), nsteps=nsteps)
    w.e = w.e * (1.0 + _noise(w.e.shape, 1, 0.05))
    return w


def cart_adi_periodic_even(nx=130, ny=29, nz=37, nsteps=5):
    """Even wrapped nx: the path bench.py times (two-cell X sweep, fused source pass, two-cell dt) at a size that
    spans three 60-cell warp tiles with a ragged tail, a row count that is no multiple of the block's 4 rows and
    strong compressions so that 7b fires."""
    w = W.noise_box(shape3=(nx, ny, nz), nsteps=nsteps)
    w.e = w.e * (1.0 + _noise(w.e.shape, 1, 0.3))
    w.vx, w.vy, w.vz = (6.0 * v for v in (w.vx, w.vy, w.vz))
    return w


def cart_iso_periodic(nx=66, ny=10, nz=9, nsteps=5):
    """Isothermal Cartesian box (the `e` slot carries c_s): the fused source pass without 7c."""
    w = W.noise_box(shape3=(nx, ny, nz), nsteps=nsteps)
    cs = 0.8 * (1.0 + _noise(w.e.shape, 1, 0.2))
    return W.Workload("cart_iso_periodic", w.mesh, W.CARTESIAN, W.ISOTHERMAL, W.Params(gamma=1.4), w.rho, cs,
                      4.0 * w.vx, 4.0 * w.vy, 4.0 * w.vz, nsteps)


def sph3d_iso_fargo_odd(nphi=45, nr=20, nth=10, nsteps=5):
    """Odd ring length: the one-cell-per-lane X sweep, the shared-memory orbital kernel and the unfused source."""
    return W.disk3d(nphi, nr, nth, nsteps)


def cart_adi_mixed_bc(nx=70, ny=9, nz=40, nsteps=5):
    """Non-periodic X (ghosted X), reflecting Y, outflow/reflecting Z; strong compressions so 7b fires."""
    bc = ((R, O), (R, R), (O, R))
    mesh = W.Mesh(nx, ny, nz, 0.0, 1.4, W.uedges(0.0, 0.3, ny), W.uedges(-0.2, 0.9, nz), bc)
    shape = (nz, ny, nx)
    rho = 1.0 + _noise(shape, 0, 0.3)
    e = 1.5 * (1.0 + _noise(shape, 1, 0.3))
    vx, vy, vz = (_noise(shape, f, 0.6) for f in (2, 3, 4))
    return W.Workload("cart_adi_mixed_bc", mesh, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4), rho, e, vx, vy, vz, nsteps)


def sod_small(nx=96, nsteps=40):
    w = W.sod(nx=nx, nyz=4, t_stop=0.05)
    w.nsteps = nsteps
    return w


def cyl2d_iso_fargo_visc(nphi=84, nr=40, nsteps=8):
    return W.disk2d(nphi, nr, nsteps)


def sph3d_iso_fargo(nphi=72, nr=33, nth=14, nsteps=6):
    return W.disk3d(nphi, nr, nth, nsteps)


def sph3d_iso_fargo_quad():
    """Longer rings: five 56-cell tiles of the orbital kernel with a ragged tail, shifts of several cells."""
    return W.disk3d(248, 12, 8, 5)


def cyl3d_adi_fargo_quad():
    """The orbital kernel with the adiabatic quantity list (7 quantities) over three tiles."""
    return cyl3d_adi_fargo(nphi=128, nr=14, nz=8, nsteps=4)


def cyl3d_adi_fargo(nphi=64, nr=30, nz=12, nsteps=5):
    """3-D cylindrical (phi, r, z): in north_star's geometry list, in no config (SURVEY.md 8(a) note)."""
    h = 0.1
    bc = ((P, P), (R, O), (P, P))
    mesh = W.Mesh(nphi, nr, nz, 0.0, 2.0 * math.pi, W.uedges(0.5, 2.0, nr), W.uedges(-0.3, 0.3, nz), bc)
    prm = W.Params(gamma=1.4, fargo_on=1, omega_frame=0.7, gm_star=1.0, planet_mass=2e-3, planet_r=1.1,
                   planet_phi0=0.4, planet_omega=0.7, planet_eps=0.05)
    shape = (nz, nr, nphi)
    r = mesh.yc()[None, :, None] * np.ones(shape)
    rho = r ** -1.0 * (1.0 + _noise(shape, 0, 0.05))
    cs = h * r ** -0.5
    e = rho * cs * cs / (1.4 - 1.0) * (1.0 + _noise(shape, 1, 0.05))
    vx = r ** -0.5 - r * prm.omega_frame + _noise(shape, 2, 0.02)
    vy = _noise(shape, 3, 0.02)
    vz = _noise(shape, 4, 0.02)
    return W.Workload("cyl3d_adi_fargo", mesh, W.CYLINDRICAL, W.ADIABATIC, prm, rho, e, vx, vy, vz, nsteps)


def sph3d_adi_nofargo(nphi=40, nr=21, nth=18, nsteps=5):
    """Spherical, adiabatic, FARGO off, inertial frame, outflow in r, reflecting/outflow in theta."""
    bc = ((P, P), (O, O), (R, O))
    mesh = W.Mesh(nphi, nr, nth, 0.0, 2.0 * math.pi, W.uedges(0.8, 1.6, nr),
                  W.uedges(0.5 * math.pi - 0.3, 0.5 * math.pi + 0.2, nth), bc)
    prm = W.Params(gamma=5.0 / 3.0, gm_star=1.0)
    shape = (nth, nr, nphi)
    r = mesh.yc()[None, :, None] * np.ones(shape)
    rho = 1.0 + _noise(shape, 0, 0.2)
    e = 0.02 * (1.0 + _noise(shape, 1, 0.2))
    vx = r ** -0.5 * (1.0 + _noise(shape, 2, 0.1))
    vy = _noise(shape, 3, 0.1)
    vz = _noise(shape, 4, 0.1)
    return W.Workload("sph3d_adi_nofargo", mesh, W.SPHERICAL, W.ADIABATIC, prm, rho, e, vx, vy, vz, nsteps)


def x_only_1d(nx=300, nsteps=10):
    mesh = W.Mesh(nx, 1, 1, 0.0, 1.0, np.array([0.0, 1.0]), np.array([0.0, 1.0]))
    shape = (1, 1, nx)
    rho = 1.0 + _noise(shape, 0, 0.2)
    e = 1.5 + _noise(shape, 1, 0.3)
    vx = _noise(shape, 2, 0.5)
    return W.Workload("x_only_1d", mesh, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4), rho, e, vx, None, None, nsteps)


def yz_only_2d(ny=45, nz=50, nsteps=6):
    bc = ((P, P), (O, R), (P, P))
    mesh = W.Mesh(1, ny, nz, 0.0, 1.0, W.uedges(0.0, 1.0, ny), W.uedges(0.0, 1.0, nz), bc)
    shape = (nz, ny, 1)
    rho = 1.0 + _noise(shape, 0, 0.2)
    e = 1.5 + _noise(shape, 1, 0.3)
    vx = _noise(shape, 2, 0.3)
    vy = _noise(shape, 3, 0.5)
    vz = _noise(shape, 4, 0.5)
    return W.Workload("yz_only_2d", mesh, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4), rho, e, vx, vy, vz, nsteps)


def nonuniform_cyl2d(nphi=50, nr=36, nsteps=6):
    """Logarithmic radial spacing: exercises centre distances vs cell widths (readings G5, G6)."""
    bc = ((P, P), (R, R), (P, P))
    yed = 0.4 * (2.5 / 0.4) ** (np.arange(nr + 1) / nr)
    mesh = W.Mesh(nphi, nr, 1, -math.pi, math.pi, yed, np.array([-0.5, 0.5]), bc)
    prm = W.Params(gamma=1.4, nu=2e-4, fargo_on=1, omega_frame=0.0, gm_star=1.0, planet_mass=0.0)
    shape = (1, nr, nphi)
    r = mesh.yc()[None, :, None] * np.ones(shape)
    rho = r ** -0.5 * (1.0 + _noise(shape, 0, 0.1))
    cs = 0.07 * r ** -0.5
    vx = r ** -0.5 * (1.0 + _noise(shape, 2, 0.03))
    vy = _noise(shape, 3, 0.02)
    return W.Workload("nonuniform_cyl2d", mesh, W.CYLINDRICAL, W.ISOTHERMAL, prm, rho, cs, vx, vy, None, nsteps)


def _with_nu(w, nu, name):
    import dataclasses
    return W.Workload(name, w.mesh, w.geometry, w.eos, dataclasses.replace(w.params, nu=nu), w.rho, w.e, w.vx, w.vy,
                      w.vz, w.nsteps)


def cart3d_visc_mixed_bc():
    """3-D Cartesian viscous stress (B1, B4) with ghosted X, walls and outflow; nu large enough to matter in 5 steps."""
    return _with_nu(cart_adi_mixed_bc(nx=34, ny=9, nz=20), 3e-3, "cart3d_visc_mixed_bc")


def cyl3d_visc_fargo():
    """3-D cylindrical viscous stress (B2, B5) with orbital advection and a planet."""
    return _with_nu(cyl3d_adi_fargo(nphi=48, nr=22, nz=10), 2e-3, "cyl3d_visc_fargo")


def sph3d_visc_fargo():
    """3-D spherical viscous stress (B3, B6) on the config-4 recipe."""
    return _with_nu(sph3d_iso_fargo(nphi=48, nr=24, nth=12), 1e-3, "sph3d_visc_fargo")


def _sheet(name, nx, ny, nz, eos, fargo, nsteps, nu=0.0):
    """Shearing sheet (NEXT-1, reading G32): Keplerian shear v_x = 2 A y plus cell-scale noise, reflecting Y walls."""
    om, A = 1.0, -0.75
    bc = ((P, P), (R, R), (P, P))
    mesh = W.Mesh(nx, ny, nz, 0.0, 2.0, W.uedges(-0.5, 0.5, ny), W.uedges(-0.25, 0.25, max(nz, 1)), bc)
    prm = W.Params(gamma=1.4, fargo_on=fargo, omega_frame=om, oort_a=A, nu=nu)
    shape = (nz, ny, nx)
    y = mesh.yc()[None, :, None] * np.ones(shape)
    rho = 1.0 + _noise(shape, 0, 0.2)
    cs = 0.3
    e = (cs * (1.0 + _noise(shape, 1, 0.1))) if eos == W.ISOTHERMAL else rho * cs * cs / 0.4 * (1.0 + _noise(shape, 1, 0.2))
    vx = 2.0 * A * y + _noise(shape, 2, 0.3)
    vy = _noise(shape, 3, 0.3)
    vz = _noise(shape, 4, 0.3) if nz > 1 else None
    return W.Workload(name, mesh, W.SHEARING_SHEET, eos, prm, rho, e, vx, vy, vz, nsteps)


def sheet3d_adi_fargo():
    """Even nx: fused source pass (GEO_SHEAR variant), two-cell X sweep and orbital kernel."""
    return _sheet("sheet3d_adi_fargo", 66, 21, 10, W.ADIABATIC, 1, 5)


def sheet3d_iso_nofargo_odd():
    """Odd nx: unfused source kernels (k_source_a carries Eq. 29), one-cell X sweep, no orbital advection."""
    return _sheet("sheet3d_iso_nofargo_odd", 45, 18, 9, W.ISOTHERMAL, 0, 5)


def sheet2d_adi_fargo():
    return _sheet("sheet2d_adi_fargo", 70, 33, 1, W.ADIABATIC, 1, 6)


def sheet3d_visc():
    """Sheet with the 3-D Cartesian viscous stress (B1, B4) on top."""
    return _sheet("sheet3d_visc", 40, 16, 8, W.ADIABATIC, 1, 4, nu=2e-3)


ALL = [sph3d_iso_fargo_quad, cyl3d_adi_fargo_quad, sheet3d_adi_fargo, sheet3d_iso_nofargo_odd, sheet2d_adi_fargo, sheet3d_visc, cart3d_visc_mixed_bc, cyl3d_visc_fargo, sph3d_visc_fargo, cart_adi_periodic, cart_adi_periodic_even, cart_iso_periodic, sph3d_iso_fargo_odd, cart_adi_mixed_bc, sod_small, cyl2d_iso_fargo_visc, sph3d_iso_fargo, cyl3d_adi_fargo,
       sph3d_adi_nofargo, x_only_1d, yz_only_2d, nonuniform_cyl2d]
