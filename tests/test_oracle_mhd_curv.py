"""Pins of the MHD oracle on CURVILINEAR meshes (oracle/mhd.cpp; reading G38; Eqs. 76, 86-91; section 3.7), against what
the physics fixes:

* constrained transport with the edge lengths and face areas of Tab. 5 keeps (sum of B S over the faces) / V of every
  zone to rounding, in cylindrical and spherical geometry, with and without orbital advection;
* current-free fields exert no force, so a gas at rest stays at rest up to the truncation error, which must fall at
  second order: a uniform Cartesian field written in cylindrical components (tension + Eq. 87 + Eq. 88 + pressure), the
  field of a line current B_phi = C/r (Eq. 88 against the pressure gradient), and on the sphere B_phi = C/(r sin theta)
  and B_theta = C/(r sin theta) (Eqs. 90, 91);
* a torsional Alfven wave on a cylindrical shell travels along z at B_z/sqrt(mu0 rho);
* orbital advection of B in a disk: rigid rotation by whole zones is an exact circular shift; Keplerian shear winds
  B_r = C/r up into B_phi at the closed-form rate r Omega' B_r (Eq. 94 in a disk), second order."""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W

P, O, R = W.PERIODIC, W.OUTFLOW, W.REFLECTING


def cyl(nphi, nr, nz, r0=1.0, r1=2.0, z0=-0.25, z1=0.25, bcy=(O, O), bcz=(P, P)):
    return W.Mesh(nphi, nr, nz, 0.0, 2 * math.pi, W.uedges(r0, r1, nr), W.uedges(z0, z1, nz), ((P, P), bcy, bcz))


def sph(nphi, nr, nth, r0=1.0, r1=2.0, th0=1.0, th1=2.0):
    return W.Mesh(nphi, nr, nth, 0.0, 2 * math.pi, W.uedges(r0, r1, nr), W.uedges(th0, th1, nth), ((P, P), (O, O), (O, O)))


def start(mesh, geometry, rho, e, v, b, **kw):
    passive = kw.pop("passive", False)
    o = Oracle(mesh, geometry, W.ADIABATIC, W.Params(gamma=5.0 / 3.0, **kw))
    shape = (mesh.nz, mesh.ny, mesh.nx)
    full = lambda a: np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), shape))
    o.set_fields(full(rho), full(e), full(v[0]), full(v[1]), full(v[2]))
    o.set_bfield(full(b[0]), full(b[1]), full(b[2]), passive=passive)
    return o


def coords(m):
    """phi, r, z|theta at faces and centres, shaped for broadcasting over (nz, ny, nx)."""
    dx = (m.xmax - m.xmin) / m.nx
    xf = (m.xmin + np.arange(m.nx) * dx)[None, None, :]
    xc = xf + 0.5 * dx
    ye, ze = np.asarray(m.yedges), np.asarray(m.zedges)
    yf, yc = ye[:-1][None, :, None], (0.5 * (ye[:-1] + ye[1:]))[None, :, None]
    zf, zc = ze[:-1][:, None, None], (0.5 * (ze[:-1] + ze[1:]))[:, None, None]
    return xf, xc, yf, yc, zf, zc


def div_b(o, m):
    """(sum of B S over the six faces) / V of every active zone that has all its faces inside the active mesh."""
    o.run_mhd_stage("BC_B")
    bx, by, bz = (o.array(n) for n in ("bx", "by", "bz"))
    ngy, ngz = o.ngy, o.ngz
    out = np.zeros((m.nz, m.ny, m.nx))
    for k in range(m.nz):
        for j in range(m.ny):
            J, K = j + ngy, k + ngz
            g = o.geometry(J, K)
            sx, sy, sz, invv = g["sx"], g["sy"], g["sz"], g["invv"]
            sy1 = o.geometry(J + 1, K)["sy"]
            sz1 = o.geometry(J, K + 1)["sz"] if m.nz > 1 else sz
            fx = (np.roll(bx[K, J, :], -1) - bx[K, J, :]) * sx
            fy = by[K, J + 1, :] * sy1 - by[K, J, :] * sy
            fz = (bz[K + 1, J, :] * sz1 - bz[K, J, :] * sz) if m.nz > 1 else 0.0
            out[k, j, :] = (fx + fy + fz) * invv
    return out


@pytest.mark.parametrize("geo,fargo", [("cyl", 0), ("cyl", 1), ("sph", 0)])
def test_div_b_is_kept_to_rounding_on_curvilinear_meshes(geo, fargo):
    r = np.random.default_rng(8)
    m = cyl(24, 10, 6, bcz=(P, P)) if geo == "cyl" else sph(24, 10, 8)
    shape = (m.nz, m.ny, m.nx)
    xf, xc, yf, yc, zf, zc = coords(m)
    b = tuple(0.3 * r.uniform(-1, 1, shape) + s for s in (0.2, 0.4, 0.3))
    vk = yc ** -0.5 * (np.sin(zc) if geo == "sph" else 1.0) * np.ones(shape)
    v = (vk + 0.05 * r.uniform(-1, 1, shape), 0.05 * r.uniform(-1, 1, shape), 0.05 * r.uniform(-1, 1, shape))
    o = start(m, W.CYLINDRICAL if geo == "cyl" else W.SPHERICAL, 1.0 + 0.2 * r.uniform(-1, 1, shape), 1.5, v, b, fargo_on=fargo, gm_star=1.0)
    d0 = div_b(o, m)
    o.step(5)
    d1 = div_b(o, m)
    scale = 0.5 * max(m.nx, m.ny, m.nz) * 10
    inner = (slice(1, -1) if m.nz > 2 else slice(None), slice(1, -1), slice(None))   # faces on an outflow wall are re-filled
    assert np.max(np.abs(d0)) > 1e-3                                                  # a random field: div B is what it is ...
    assert np.max(np.abs((d1 - d0)[inner])) <= 1e-13 * scale, np.max(np.abs((d1 - d0)[inner]))   # ... and stays so
    assert not np.array_equal(o.get_bfield()[0], b[0])


def _rest_acceleration(m, geometry, b):
    """max |v| / dt after one tiny update of a gas at rest with uniform pressure, over the middle half of the mesh in Y and Z
    (the same physical region at every resolution, away from the walls)."""
    dt = 1e-6
    z = np.zeros((m.nz, m.ny, m.nx))
    o = start(m, geometry, 1.0, 1.5, (z, z, z), b, dt_fixed=dt)
    o.step(1)
    f = o.get_fields()
    ys = slice(m.ny // 4, m.ny - m.ny // 4)
    zs = slice(m.nz // 4, m.nz - m.nz // 4) if m.nz > 6 else slice(None)
    return max(float(np.max(np.abs(f[c][zs, ys, :]))) for c in (2, 3, 4)) / dt


def test_uniform_cartesian_field_in_cylindrical_components_exerts_no_force():
    acc = []
    for n in (1, 2):
        m = cyl(32 * n, 16 * n, 1, bcz=(P, P))
        xf, xc, yf, yc, zf, zc = coords(m)
        b0 = 0.8
        bphi = -b0 * np.sin(xf) + 0 * yc          # on the phi faces: (phi face, r centre)
        br = b0 * np.cos(xc) + 0 * yf             # on the r faces: (phi centre, r face)
        acc.append(_rest_acceleration(m, W.CYLINDRICAL, (bphi, br, 0.0 * xc)))
    scale = 0.8 ** 2 / 1.0                        # B^2 / (rho r): what each single term of the balance amounts to
    assert acc[0] < 0.02 * scale and acc[1] < acc[0] / 3.0, (acc, scale)


def test_line_current_field_is_force_free_in_cylindrical_and_spherical_geometry():
    acc = []
    for n in (1, 2):
        m = cyl(8, 16 * n, 4)
        xf, xc, yf, yc, zf, zc = coords(m)
        acc.append(_rest_acceleration(m, W.CYLINDRICAL, (0.7 / yc + 0 * xf, 0.0 * xc, 0.0 * xc)))     # B_phi = C / r: Eq. 88
    # (with B_phi averaged before it is squared and 1/r taken at the face, the two terms cancel identically on a uniform mesh)
    assert acc[0] < 1e-9 and acc[1] < 1e-9, acc
    for comp in (0, 2):                            # B_phi = C / (r sin theta), then B_theta = C / (r sin theta): Eqs. 90, 91
        acc = []
        for n in (1, 2):
            m = sph(8, 16 * n, 16 * n)
            xf, xc, yf, yc, zf, zc = coords(m)
            zero = 0.0 * xc * yc * zc
            f = (0.7 / (yc * np.sin(zc)) + zero) if comp == 0 else (0.7 / (yc * np.sin(zf)) + zero)
            b = (f, zero, zero) if comp == 0 else (zero, zero, f)
            acc.append(_rest_acceleration(m, W.SPHERICAL, b))
        assert acc[0] < 0.02 * 0.49 and acc[1] < max(acc[0] / 3.0, 1e-9), (comp, acc)   # (B_theta: cancels identically)


def test_torsional_alfven_wave_on_a_cylindrical_shell():
    n = 64
    m = cyl(4, 4, n, r0=10.0, r1=10.4, z0=0.0, z1=1.0, bcy=(R, R), bcz=(P, P))
    xf, xc, yf, yc, zf, zc = coords(m)
    shape = (n, 4, 4)
    bz0, rho0, amp = 0.5, 1.0, 1e-6
    prof = amp * np.sin(2 * math.pi * zc) * np.ones(shape)
    z = np.zeros(shape)
    o = start(m, W.CYLINDRICAL, rho0, 0.9, (prof, z, z), (-math.sqrt(rho0) * prof, z, z + bz0), t_stop=0.5 / (bz0 / math.sqrt(rho0)))
    o.step(100000)
    bphi = o.get_bfield()[0][:, 1, 0]
    c = np.sum(bphi * np.exp(-2j * math.pi * zc[:, 0, 0])) * 2.0 / n
    c0 = np.sum(-prof[:, 1, 0] * np.exp(-2j * math.pi * zc[:, 0, 0])) * 2.0 / n
    lag = (np.angle(c) - np.angle(c0) + math.pi) % (2 * math.pi) - math.pi       # half a period: the phase turns by -pi
    assert abs(abs(lag) - math.pi) < 0.03 and 0.95 < abs(c) / abs(c0) < 1.05


def test_orbital_advection_of_b_in_a_disk():
    # rigid rotation by exactly N zones per update: a circular shift of all three components
    nphi, nr, nz = 32, 8, 4
    m = cyl(nphi, nr, nz)
    xf, xc, yf, yc, zf, zc = coords(m)
    shape = (nz, nr, nphi)
    r = np.random.default_rng(3)
    # a divergence-free field (Eq. 107 uses div B = 0): B_phi, B_r from A_z on the z edges, B_z any function of (phi, r)
    az = 0.05 * r.standard_normal((nr + 1, nphi))
    dx, ye = 2 * math.pi / nphi, np.asarray(m.yedges)
    bphi = (az[1:, :] - az[:-1, :]) / np.diff(ye)[:, None]
    br = -(np.roll(az, -1, axis=1) - az)[:-1, :] / (ye[:-1, None] * dx)
    b = (bphi[None] * np.ones(shape), br[None] * np.ones(shape), (0.3 * r.uniform(-1, 1, (nr, nphi)))[None] * np.ones(shape))
    om, N = 0.9, 3
    dt = N * (2 * math.pi / nphi) / om
    o = start(m, W.CYLINDRICAL, 1.0, 1.5, (om * yc * np.ones(shape), 0, 0), b, passive=True, fargo_on=1)
    o.run_stage("BC1"); o.run_mhd_stage("BC_B"); o.run_stage("VMEAN"); o.set_dt(dt); o.run_mhd_stage("ORBITAL")
    for a, a0 in zip(o.get_bfield(), b):
        assert np.allclose(a[1:-1, 1:-1, :], np.roll(a0, N, axis=2)[1:-1, 1:-1, :], rtol=0, atol=1e-14)
    # Keplerian shear winds B_r = C / r up: dB_phi/dt = r Omega' B_r = -1.5 C r^-2.5
    errs = []
    for n in (1, 2):
        m = cyl(16, 16 * n, 1, bcz=(P, P))
        xf, xc, yf, yc, zf, zc = coords(m)
        shape = (1, 16 * n, 16)
        C, dt = 0.4, 1e-3
        o = start(m, W.CYLINDRICAL, 1.0, 1.5, (yc ** -0.5 * np.ones(shape), 0, 0), (np.zeros(shape), C / yf * np.ones(shape), np.zeros(shape)),
                  passive=True, fargo_on=1)
        o.run_stage("BC1"); o.run_mhd_stage("BC_B"); o.run_stage("VMEAN"); o.set_dt(dt); o.run_mhd_stage("ORBITAL")
        bx = o.get_bfield()[0][0, 3:-3, 0]
        exact = dt * (-1.5 * C) * yc[0, 3:-3, 0] ** -2.5
        errs.append(float(np.max(np.abs(bx - exact))) / float(np.max(np.abs(exact))))
    assert errs[0] < 0.02 and errs[1] < errs[0] / 3.0, errs
