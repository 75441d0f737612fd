"""Pins of the oracle's 3-D viscous sub-step (oracle/viscosity3d.cpp; App. B, Eqs. B1-B6) against
what the mathematics fixes, independent of the oracle's own code:

* Cartesian, exact: a discrete shear wave v_a = A sin(kappa x_b) (a != b) decays by the factor
  1 - dt nu (2 - 2 cos(kappa D)) / D^2 per sub-step, a compressive wave (a == b) by 4/3 of that (B1, B4);
* every geometry: a uniform translation and a rigid rotation about ANY axis are stress free, and a uniform
  shear has a constant stress tensor whose divergence vanishes; written in cylindrical / spherical components
  these fields exercise every curvature term of B2/B3 and B5/B6 (a dropped or mis-signed term leaves an O(1)
  residual), while the discrete residual falls as h^2;
* every geometry: for the divergence-free quadratic field u = (y^2, z^2, x^2) and uniform density the force is
  nu Laplacian(u) = nu (2, 2, 2): pins the sign and the magnitude of the force in curvilinear components;
* 3-D cylindrical with no z dependence reproduces the (pinned) 2-D cylindrical routine.
"""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W

NG = 3
P_, O_ = W.PERIODIC, W.OUTFLOW


def _ghosted(edges):
    e = np.asarray(edges, dtype=np.float64)
    lo = e[0] - (np.arange(NG, 0, -1)) * (e[1] - e[0])
    hi = e[-1] + (np.arange(1, NG + 1)) * (e[-1] - e[-2])
    return np.concatenate([lo, e, hi])


class Setup:
    """An oracle context plus the coordinates of every stored position (ghost-inclusive, shape (TZ, TY, TX))."""

    def __init__(self, geometry, nx, ny, nz, xr, yr, zr, nu, bc):
        mesh = W.Mesh(nx, ny, nz, xr[0], xr[1], W.uedges(yr[0], yr[1], ny), W.uedges(zr[0], zr[1], nz), bc)
        self.o = Oracle(mesh, geometry, W.ISOTHERMAL, W.Params(nu=nu))
        self.geometry, self.nu = geometry, nu
        o = self.o
        ngx = o.ngx
        dx = mesh.dx
        xf = xr[0] + (np.arange(o.TX) - ngx) * dx
        ye, ze = _ghosted(mesh.yedges), _ghosted(mesh.zedges)
        self.xf, self.xc = xf[None, None, :], (xf + 0.5 * dx)[None, None, :]
        self.ye, self.yc = ye[:-1][None, :, None], (0.5 * (ye[:-1] + ye[1:]))[None, :, None]
        self.ze, self.zc = ze[:-1][None, None].reshape(-1, 1, 1), (0.5 * (ze[:-1] + ze[1:])).reshape(-1, 1, 1)
        self.shape = (o.TZ, o.TY, o.TX)
        self.h = max(dx, ye[1] - ye[0], ze[1] - ze[0])

    def cart_of(self, X, Y, Z):
        """Cartesian position and local unit vectors (e_X, e_Y, e_Z) of the point with coordinates (X, Y, Z)."""
        X, Y, Z = np.broadcast_arrays(X, Y, Z)
        zero, one = np.zeros(X.shape), np.ones(X.shape)
        if self.geometry == W.CARTESIAN:
            return (X, Y, Z), ((one, zero, zero), (zero, one, zero), (zero, zero, one))
        if self.geometry == W.CYLINDRICAL:     # X = phi, Y = r, Z = z
            c, s = np.cos(X), np.sin(X)
            return (Y * c, Y * s, Z), ((-s, c, zero), (c, s, zero), (zero, zero, one))
        c, s, ct, st = np.cos(X), np.sin(X), np.cos(Z), np.sin(Z)   # X = phi, Y = r, Z = theta
        return (Y * st * c, Y * st * s, Y * ct), ((-s, c, zero), (st * c, st * s, ct), (ct * c, ct * s, -st))

    def components(self, field):
        """Staggered components of the Cartesian vector field `field(x, y, z) -> (ux, uy, uz)`."""
        out = []
        for comp, pos in enumerate(((self.xf, self.yc, self.zc), (self.xc, self.ye, self.zc), (self.xc, self.yc, self.ze))):
            x, e = self.cart_of(*pos)
            u = field(*x)
            out.append(sum(u[a] * e[comp][a] for a in range(3)) * np.ones(self.shape))
        return out

    def substep(self, v, dt, rho=None):
        o = self.o
        o.set_array("rho", np.ones(self.shape) if rho is None else rho)
        for name, a in zip(("vxc", "vyc", "vzc"), v):
            o.set_array(name, np.ascontiguousarray(a))
        o.set_dt(dt)
        o.run_stage("SRC_D")
        return [o.array(n) for n in ("vxd", "vyd", "vzd")]

    def interior(self, a, m=2):
        sx = slice(None) if self.o.ngx == 0 else slice(m, -m)
        return a[m:-m, m:-m, sx]


# ---------------------------------------------------------------- Cartesian: exact discrete decay ---------
@pytest.mark.parametrize("comp", [0, 1, 2])
@pytest.mark.parametrize("along", [0, 1, 2])
def test_cartesian_wave_decays_by_the_discrete_laplacian(comp, along):
    n = (16, 12, 10)
    L = (1.0, 0.75, 0.5)
    nu, dt, amp, mode = 3e-3, 0.02, 0.7, 2
    bc = ((P_, P_), (P_, P_), (P_, P_))
    s = Setup(W.CARTESIAN, n[0], n[1], n[2], (0.0, L[0]), (0.0, L[1]), (0.0, L[2]), nu, bc)
    kappa = 2.0 * math.pi * mode / L[along]
    D = L[along] / n[along]
    # coordinate of the velocity component `comp` along direction `along` (its own direction: the face)
    coords = [(s.xf, s.yc, s.zc), (s.xc, s.ye, s.zc), (s.xc, s.yc, s.ze)][comp]
    v = [np.zeros(s.shape) for _ in range(3)]
    v[comp] = amp * np.sin(kappa * coords[along]) * np.ones(s.shape)
    # ghost layers must hold the periodic continuation: the analytic field already does (uniform ghost spacing)
    out = s.substep(v, dt)
    lam = (2.0 - 2.0 * math.cos(kappa * D)) / (D * D)
    factor = 1.0 - dt * nu * lam * (4.0 / 3.0 if comp == along else 1.0)
    for c in range(3):
        got, ref = s.interior(out[c]), s.interior(v[c]) * (factor if c == comp else 1.0)
        assert np.max(np.abs(got - ref)) <= 1e-13 * amp, (comp, along, c)


def test_cartesian_force_is_divided_by_the_face_mean_density():
    """Reading G24: with rho = 2 everywhere the velocity change halves... it does not: tau carries rho, so the
    change is the same; with a density jump the face-mean density of the two cells divides the force."""
    bc = ((P_, P_), (P_, P_), (P_, P_))
    s = Setup(W.CARTESIAN, 16, 8, 8, (0.0, 1.0), (0.0, 0.5), (0.0, 0.5), 1e-2, bc)
    kappa, D = 2.0 * math.pi, 0.5 / 8
    v = [0.3 * np.sin(kappa / 0.5 * s.yc) * np.ones(s.shape), np.zeros(s.shape), np.zeros(s.shape)]
    a = s.substep(v, 0.01)[0]
    b = s.substep(v, 0.01, rho=np.full(s.shape, 2.0))[0]
    assert np.max(np.abs(s.interior(a) - s.interior(b))) <= 1e-15


# ---------------------------------------------------------------- curvilinear: stress-free fields ---------
def _make(geometry, n):
    if geometry == W.CARTESIAN:
        bc = ((O_, O_), (O_, O_), (O_, O_))
        return Setup(geometry, n, n, n, (0.3, 1.1), (-0.2, 0.6), (0.1, 0.9), 1.0, bc)
    bc = ((P_, P_), (O_, O_), (O_, O_))
    if geometry == W.CYLINDRICAL:
        return Setup(geometry, 2 * n, n, n, (0.0, 2.0 * math.pi), (0.6, 1.4), (-0.4, 0.4), 1.0, bc)
    return Setup(geometry, 2 * n, n, n, (0.0, 2.0 * math.pi), (0.6, 1.4), (0.9, 1.9), 1.0, bc)


def _residual(geometry, n, field, expect=None):
    """max over the interior of |dv/dt - expected force component| for the Cartesian vector field `field`."""
    s = _make(geometry, n)
    v = s.components(field)
    dt = 1e-3
    out = s.substep(v, dt)
    exp = s.components(expect) if expect is not None else [np.zeros(s.shape)] * 3
    return max(float(np.max(np.abs(s.interior((o - a) / dt - e, 3)))) for o, a, e in zip(out, v, exp))


GEOS = [W.CARTESIAN, W.CYLINDRICAL, W.SPHERICAL]
OMEGA = (0.3, -0.7, 0.5)
FIELDS = {
    "translation": lambda x, y, z: (0.4 + 0 * x, -0.9 + 0 * x, 0.6 + 0 * x),
    "rotation": lambda x, y, z: (OMEGA[1] * z - OMEGA[2] * y, OMEGA[2] * x - OMEGA[0] * z, OMEGA[0] * y - OMEGA[1] * x),
    "shear": lambda x, y, z: (0.8 * y - 0.5 * z, 0.3 * z + 0 * x, -0.6 * x + 0.2 * y),   # traceless gradient, constant stress
}


@pytest.mark.parametrize("geometry", GEOS)
@pytest.mark.parametrize("name", sorted(FIELDS))
def test_stress_free_and_constant_stress_fields_feel_no_force(geometry, name):
    r1, r2 = _residual(geometry, 12, FIELDS[name]), _residual(geometry, 24, FIELDS[name])
    # |u| ~ 1, nu = 1, lengths ~ 1: a dropped or mis-signed term leaves a residual of order 1
    assert r2 < 0.02, (name, r1, r2)
    if geometry != W.CARTESIAN:
        assert r2 < r1 / 3.0, (name, r1, r2)          # second order
    else:
        assert r2 < 1e-11, (name, r2)                 # linear fields are differenced exactly on a Cartesian mesh


@pytest.mark.parametrize("geometry", GEOS)
def test_quadratic_field_feels_nu_times_its_laplacian(geometry):
    field = lambda x, y, z: (y * y, z * z, x * x)     # divergence free, Laplacian = (2, 2, 2)
    lap = lambda x, y, z: (2.0 + 0 * x, 2.0 + 0 * x, 2.0 + 0 * x)
    r1, r2 = _residual(geometry, 12, field, lap), _residual(geometry, 24, field, lap)
    assert r2 < 0.05, (r1, r2)                        # against a force of magnitude 2 sqrt(3)
    if geometry != W.CARTESIAN:
        assert r2 < r1 / 3.0, (r1, r2)
    else:
        assert r2 < 1e-10, r2


@pytest.mark.parametrize("geometry", GEOS)
def test_compressive_field_feels_the_bulk_term(geometry):
    """u = (x^2, 0, 0): force = nu (Laplacian u + grad(div u) / 3) = nu (2 + 2/3, 0, 0)  (B1 with the -2/3 div term)."""
    field = lambda x, y, z: (x * x, 0 * x, 0 * x)
    force = lambda x, y, z: (8.0 / 3.0 + 0 * x, 0 * x, 0 * x)
    r1, r2 = _residual(geometry, 12, field, force), _residual(geometry, 24, field, force)
    assert r2 < 0.05, (r1, r2)
    if geometry != W.CARTESIAN:
        assert r2 < r1 / 3.0, (r1, r2)


# ---------------------------------------------------------------- 3-D cylindrical vs the pinned 2-D routine --
def test_cylindrical_3d_without_z_dependence_matches_the_2d_routine():
    nphi, nr, nz, nu, dt = 24, 14, 5, 2e-3, 0.05
    bc3 = ((P_, P_), (O_, O_), (P_, P_))
    s3 = Setup(W.CYLINDRICAL, nphi, nr, nz, (0.0, 2.0 * math.pi), (0.5, 1.5), (-0.1, 0.1), nu, bc3)
    m2 = W.Mesh(nphi, nr, 1, 0.0, 2.0 * math.pi, W.uedges(0.5, 1.5, nr), np.array([-0.5, 0.5]), bc3)
    o2 = Oracle(m2, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(nu=nu))
    rng = np.random.default_rng(5)
    plane = lambda: rng.uniform(-1.0, 1.0, (1, s3.shape[1], s3.shape[2]))
    rho2, vx2, vy2 = 1.0 + 0.3 * plane(), plane(), plane()
    v3 = [np.repeat(vx2, s3.shape[0], 0), np.repeat(vy2, s3.shape[0], 0), np.zeros(s3.shape)]
    out3 = s3.substep(v3, dt, rho=np.repeat(rho2, s3.shape[0], 0))
    o2.set_array("rho", rho2); o2.set_array("vxc", vx2); o2.set_array("vyc", vy2)
    o2.set_dt(dt); o2.run_stage("SRC_D")
    kmid = s3.shape[0] // 2
    # the 2-D routine starts its radial force at j = 2; compare where both are defined
    for got, ref in ((out3[0][kmid, 2:-2], o2.array("vxd")[0, 2:-2]), (out3[1][kmid, 2:-2], o2.array("vyd")[0, 2:-2])):
        assert np.max(np.abs(got - ref)) <= 1e-13
    assert np.max(np.abs(s3.interior(out3[2]))) <= 1e-15
