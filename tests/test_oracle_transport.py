"""Pins of the oracle's transport step, orbital advection and 7d viscosity. CPU only."""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W
from helpers import mesh, rng_fields

PER = (W.PERIODIC,) * 2
OUT = (W.OUTFLOW,) * 2
REF = (W.REFLECTING,) * 2


def _volumes(o):
    V = np.empty((o.TZ, o.TY))
    for k in range(o.TZ):
        for j in range(o.TY):
            V[k, j] = 1.0 / o.geometry(j, k)["invv"]
    return V[:, :, None]


# ---------------------------------------------------------------- momenta and Eq. 51
@pytest.mark.parametrize("geometry", [W.CARTESIAN, W.CYLINDRICAL, W.SPHERICAL])
def test_eq51_on_untransported_momenta_returns_old_velocity(geometry):
    """Eq. 51 applied to the momenta of Eqs. 49-50 before any transport gives back v."""
    z = (0.0, 1.0) if geometry != W.SPHERICAL else (1.0, 1.8)
    m = mesh(8, 6, 5, x=(-math.pi, math.pi), y=(1.0, 2.0), z=z, bc=(PER, OUT, OUT))
    o = Oracle(m, geometry, W.ADIABATIC, W.Params(omega_frame=0.6))
    f = rng_fields((5, 6, 8), 5)
    o.set_fields(*f)
    o.step_until("BC1")
    o.run_stage("MOM")
    o.run_stage("NEWVEL")
    for name, v in (("vx", f[2]), ("vy", f[3]), ("vz", f[4])):
        assert np.allclose(o.active(o.array(name)), v, rtol=0, atol=2e-15)


def test_momenta_table2():
    """Tab. 2: Pi_x = rho r sin(theta) (v_phi + r sin(theta) Omega_f) in spherical geometry
    (angular momentum), Pi_y = rho v_r, Pi_z = rho r v_theta."""
    m = mesh(4, 3, 3, x=(-math.pi, math.pi), y=(1.0, 2.0), z=(1.0, 1.6), bc=(PER, OUT, OUT))
    om = 0.4
    o = Oracle(m, W.SPHERICAL, W.ISOTHERMAL, W.Params(omega_frame=om))
    rho, e, vx, vy, vz = rng_fields((3, 3, 4), 8)
    o.set_fields(rho, e, vx, vy, vz)
    o.step_until("BC1")
    o.run_stage("MOM")
    R = (m.yc()[None, :, None] * np.sin(m.zc())[:, None, None]) * np.ones((3, 3, 4))
    r = m.yc()[None, :, None] * np.ones((3, 3, 4))
    assert np.allclose(o.active(o.array("pxm")), rho * R * (vx + R * om), rtol=1e-14)
    assert np.allclose(o.active(o.array("pxp")), rho * R * (np.roll(vx, -1, axis=2) + R * om), rtol=1e-14)
    assert np.allclose(o.active(o.array("pym")), rho * vy, rtol=1e-15)
    assert np.allclose(o.active(o.array("pzm")), rho * r * vz, rtol=1e-15)
    assert np.allclose(o.active(o.array("pyp"))[:, :-1], rho[:, :-1] * vy[:, 1:], rtol=1e-15)
    assert np.allclose(o.active(o.array("pzp"))[:-1], (rho * r)[:-1] * vz[1:], rtol=1e-15)


# ---------------------------------------------------------------- sweeps (Eqs. 40-48)
def test_uniform_state_is_preserved_bitwise():
    n = 6
    m = mesh(n, n, n)
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4))
    s = (n, n, n)
    f = (np.full(s, 1.3), np.full(s, 0.7), np.full(s, 0.25), np.full(s, -0.5), np.full(s, 0.125))
    o.set_fields(*f)
    o.step(3)
    for a, b in zip(o.get_fields(), f):
        assert np.max(np.abs(a - b)) <= 4e-16      # momenta/rho round trip only
    assert np.array_equal(o.get_fields()[0], f[0])


@pytest.mark.parametrize("direction", [0, 1, 2])
@pytest.mark.parametrize("wv", [0.6, -0.6])
def test_sweep_translates_linear_profile_exactly(direction, wv):
    """Uniform velocity w, rho = 1, e linear along the sweep: e_new = e(x - w dt) in interior cells."""
    n, dt = 12, 0.02
    m = mesh(n, n, n, bc=(OUT, OUT, OUT))
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4, dt_fixed=dt))
    s = (n, n, n)
    c = [m.zc()[:, None, None], m.yc()[None, :, None], m.xc()[None, None, :]][2 - direction] * np.ones(s)
    e = 2.0 + 0.5 * c
    v = [np.zeros(s), np.zeros(s), np.zeros(s)]
    v[direction] = np.full(s, wv)
    o.set_fields(np.ones(s), e, *v)
    o.step_until("BC1")
    o.set_dt(dt)
    o.run_stage("MOM")
    o.run_stage(("SWEEP_X", "SWEEP_Y", "SWEEP_Z")[direction])
    got = o.active(o.array("e"))[2:-2, 2:-2, 2:-2]
    assert np.allclose(got, (2.0 + 0.5 * (c - wv * dt))[2:-2, 2:-2, 2:-2], rtol=1e-14)
    assert np.allclose(o.active(o.array("rho"))[2:-2, 2:-2, 2:-2], 1.0, rtol=1e-15)


def test_sweeps_conserve_mass_momenta_energy_in_periodic_box():
    """every transported quantity is conserved to rounding by each sweep."""
    n = 8
    m = mesh(n, n, n)
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4))
    o.set_fields(*rng_fields((n, n, n), 6, vamp=0.5))
    o.step_until("MOM")
    names = ("rho", "e", "pxm", "pxp", "pym", "pyp", "pzm", "pzp")
    before = {a: o.active(o.array(a)).sum() for a in names}
    for st in ("SWEEP_X", "SWEEP_Y", "SWEEP_Z"):
        o.run_stage(st)
        for a in names:
            assert o.active(o.array(a)).sum() == pytest.approx(before[a], rel=1e-13, abs=1e-13)
    assert np.max(np.abs(o.active(o.array("rho")) - 1.0)) > 1e-3     # not vacuous


@pytest.mark.parametrize("geometry", [W.CYLINDRICAL, W.SPHERICAL])
def test_full_step_conserves_mass_and_angular_momentum_with_walls(geometry):
    """Reflecting walls in r (and theta), periodic phi, FARGO on: total mass and total angular
    momentum sum((Pi_x- + Pi_x+)/2 V) are conserved to rounding by transport + orbital advection
    ("conserves mass and angular momentum to computer accuracy")."""
    nz = 1 if geometry == W.CYLINDRICAL else 6
    z = (-0.5, 0.5) if geometry == W.CYLINDRICAL else (math.pi / 2 - 0.2, math.pi / 2 + 0.2)
    m = mesh(24, 10, nz, x=(-math.pi, math.pi), y=(0.6, 1.8), z=z, bc=(PER, REF, REF))
    prm = W.Params(fargo_on=1, omega_frame=0.3, gm_star=1.0)
    o = Oracle(m, geometry, W.ISOTHERMAL, prm)
    s = (nz, 10, 24)
    rng = np.random.default_rng(9)
    rc = m.yc()[None, :, None] * np.ones(s)
    rho = 1.0 + 0.3 * rng.uniform(-1, 1, s)
    vx = rc ** -0.5 - 0.3 * rc + 0.05 * rng.uniform(-1, 1, s)
    vy = 0.05 * rng.uniform(-1, 1, s)
    vz = 0.05 * rng.uniform(-1, 1, s) if nz > 1 else None
    o.set_fields(rho, np.full(s, 0.05), vx, vy, vz)
    o.step_until("MOM")
    V = _volumes(o)

    def totals():
        mass = (o.active(o.array("rho") * V)).sum()
        ang = (o.active(0.5 * (o.array("pxm") + o.array("pxp")) * V)).sum()
        return mass, ang
    m0, a0 = totals()
    for st in ("SWEEP_X", "SWEEP_Y", "SWEEP_Z", "ORB_FRAC", "ORB_SHIFT"):
        o.run_stage(st)
        m1, a1 = totals()
        assert m1 == pytest.approx(m0, rel=2e-14), st
        assert a1 == pytest.approx(a0, rel=2e-14), st
    assert np.abs(o.array("nshift")).max() >= 1 or np.abs(o.array("xi")).max() > 0.05


# ---------------------------------------------------------------- orbital advection
def _shift_setup(s_cells, n=16):
    """Cartesian periodic box, uniform pressure, v_x = v0 uniform, dx = 1/16, dt = 1/32 (exact in
    binary): the ring moves by s_cells = v0 dt / dx cells."""
    m = mesh(n, 4, 4, y=(0, 0.25), z=(0, 0.25))
    dt = 1.0 / 32.0
    v0 = s_cells * (1.0 / n) / dt
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4, fargo_on=1, dt_fixed=dt))
    s = (4, 4, n)
    return o, m, s, v0


def test_integer_shift_is_exact():
    """"The circular permutation of Eq. (69) does not introduce numerical errors": residual
    velocity 0 and v0 dt / dx = 3 exactly => rho, e are the input rotated by 3 cells, bit for bit,
    towards +x (Q_i <- Q_{i-N})."""
    for N in (3, -5, 16 + 2):
        o, m, s, v0 = _shift_setup(float(N))
        rho = rng_fields(s, 12)[0]
        z = np.zeros(s)
        o.set_fields(rho, np.full(s, 2.5), np.full(s, v0), z, z)
        o.step(1)
        r1, e1, vx1, _, _ = o.get_fields()
        assert np.array_equal(r1, np.roll(rho, N, axis=2))
        assert np.array_equal(e1, np.full(s, 2.5))
        assert np.allclose(vx1, v0, rtol=1e-15)


def test_fractional_shift_moves_smooth_profile_the_right_way():
    """s = 2.3 cells: N = 2, xi = 0.3; s = 2.5: N = floor(3.0) = 3, xi = -0.5 (reading G11).
    A smooth profile must land on its analytic translate; a sign error in xi would be off by
    O(amplitude * 2 pi * 0.6 / n)."""
    n = 64
    for sc, N, xi in ((2.3, 2, 0.3), (2.5, 3, -0.5), (-1.75, -2, 0.25)):
        o, m, s, v0 = _shift_setup(sc, n)
        x = m.xc()[None, None, :] * np.ones(s)
        rho = 1.0 + 0.1 * np.sin(2 * np.pi * x)
        z = np.zeros(s)
        o.set_fields(rho, np.full(s, 2.5), np.full(s, v0), z, z)
        o.step(1)
        assert np.all(o.array("nshift") == N)
        assert np.allclose(o.array("xi"), xi, atol=1e-12)
        r1 = o.get_fields()[0]
        exact = 1.0 + 0.1 * np.sin(2 * np.pi * (x - sc / n))
        assert np.max(np.abs(r1 - exact)) < 3e-4      # limiter clips the extrema; a sign error gives 6e-3
        assert r1.sum() == pytest.approx(rho.sum(), rel=1e-14)


def test_fargo_on_and_off_agree_for_smooth_flow():
    """Operator splitting v = v0 + dv (Eqs. 60-63) changes truncation errors only: with and without
    orbital advection a smooth 2-D disk state evolves to the same result within discretisation error."""
    res = []
    for fargo in (0, 1):
        m = mesh(64, 24, 1, x=(-math.pi, math.pi), y=(0.8, 1.6), z=(-0.5, 0.5), bc=(PER, REF, PER))
        prm = W.Params(fargo_on=fargo, gm_star=1.0, dt_fixed=2e-3)
        o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, prm)
        s = (1, 24, 64)
        rc = m.yc()[None, :, None] * np.ones(s)
        ph = m.xc()[None, None, :] * np.ones(s)
        rho = 1.0 + 0.05 * np.cos(2 * ph) * np.exp(-((rc - 1.2) / 0.15) ** 2)
        o.set_fields(rho, np.full(s, 0.05), rc ** -0.5, np.zeros(s), None)
        o.step(40)
        res.append(o.get_fields())
    for a, b, tol in zip(res[0][:4], res[1][:4], (2e-3, 0, 2e-3, 2e-3)):
        assert np.max(np.abs(a - b)) <= tol


# ---------------------------------------------------------------- ghost budget
@pytest.mark.parametrize("case", ["disk3d", "sod3d", "disk2d"])
def test_three_ghost_layers_suffice(case):
    """Indiscernibility test: the active-zone result does not depend on the number of ghost
    layers once there are enough: NG = 3 and NG = 4 give bit-identical fields."""
    if case == "disk3d":
        w = W.disk3d(24, 8, 6, nsteps=3)
    elif case == "disk2d":
        w = W.disk2d(32, 12, nsteps=3)
    else:
        w = W.sod(24, 4)
    out = []
    for ng in (3, 4):
        o = Oracle(w.mesh, w.geometry, w.eos, w.params, nghost=ng)
        o.set_fields(*w.fields())
        o.step(3)
        out.append(o.get_fields() + (o.time()[0],))
    for a, b in zip(*out):
        assert np.array_equal(a, b)


# ---------------------------------------------------------------- 7d viscosity (App. B)
def test_viscosity_rigid_rotation_has_no_stress():
    m = mesh(16, 12, 1, x=(-math.pi, math.pi), y=(0.5, 1.5), z=(-0.5, 0.5), bc=(PER, OUT, PER))
    o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(nu=0.1, dt_fixed=0.1))
    s = (1, 12, 16)
    rc = m.yc()[None, :, None] * np.ones(s)
    rho = rng_fields(s, 2)[0]
    o.set_fields(rho, np.full(s, 1e-9), 0.7 * rc, np.zeros(s), None)
    o.step_until("BC1")
    vxc, vyc = o.array("vx").copy(), o.array("vy").copy()     # feed 7d the rigid rotation itself
    o.set_array("vxc", vxc)
    o.set_array("vyc", vyc)
    o.set_dt(0.1)
    o.run_stage("SRC_D")
    sl = (0, slice(o.ngy + 2, o.ngy + 10))
    assert np.max(np.abs(o.array("vxd")[sl] - vxc[sl])) < 1e-14
    assert np.max(np.abs(o.array("vyd")[sl] - vyc[sl])) < 1e-14


def test_viscosity_shear_flow_closed_form():
    """v_phi = A r^p, v_r = 0, uniform rho: tau_phi_r = -rho nu A (p-1) r^(p-1) and
    dv_phi/dt = nu A (p^2 - 1) r^(p-2)  (B2, B5).  Keplerian p = -1/2: -3/4 nu A r^-5/2."""
    nr, nu, A, p = 128, 0.05, 1.0, -0.5
    m = mesh(8, nr, 1, x=(-math.pi, math.pi), y=(1.0, 2.0), z=(-0.5, 0.5), bc=(PER, OUT, PER))
    o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(nu=nu, dt_fixed=1.0))
    s = (1, nr, 8)
    rc = m.yc()[None, :, None] * np.ones(s)
    o.set_fields(np.ones(s), np.full(s, 1e-9), A * rc ** p, np.zeros(s), None)
    o.step_until("BC1")
    full = lambda a: np.ascontiguousarray(a)
    for nm, src in (("vxc", "vx"), ("vyc", "vy")):
        o.set_array(nm, full(o.array(src)))
    o.set_dt(1.0)
    o.run_stage("SRC_D")
    acc = (o.active(o.array("vxd")) - o.active(o.array("vx")))[0, 4:-4, 0]
    r = m.yc()[4:-4]
    assert np.allclose(acc, nu * A * (p * p - 1.0) * r ** (p - 2.0), rtol=2e-3)
    assert np.max(np.abs(o.active(o.array("vyd"))[0, 4:-4])) < 1e-12
