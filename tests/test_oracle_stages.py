"""Pins of the oracle's stages (source step, momenta, sweeps, orbital advection, time step) against
closed forms, invariants and hand-computed stencils.  CPU only."""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W
from helpers import mesh, rng_fields

PER = (W.PERIODIC,) * 2
OUT = (W.OUTFLOW,) * 2
REF = (W.REFLECTING,) * 2


def _box(n=8, eos=W.ADIABATIC, seed=1, **kw):
    m = mesh(n, n, n)
    o = Oracle(m, W.CARTESIAN, eos, W.Params(gamma=1.4, **kw))
    f = rng_fields((n, n, n), seed)
    o.set_fields(*f)
    return o, m, f


# ---------------------------------------------------------------------------- time step (Eq. 59)
def test_dt_uniform_state_at_rest_closed_form():
    """Only the sound-speed limit is active: dt = C * min_d(L_d) / c, c = sqrt(gamma P / rho)."""
    m = mesh(8, 4, 2, x=(0, 1), y=(0, 1), z=(0, 1))       # L = 1/8, 1/4, 1/2
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4, cfl=0.44))
    s = (2, 4, 8)
    rho, P = 2.0, 3.0
    o.set_fields(np.full(s, rho), np.full(s, P / 0.4), np.zeros(s), np.zeros(s), np.zeros(s))
    o.step_until("DT")
    assert o.time()[1] == pytest.approx(0.44 * (1.0 / 8.0) / math.sqrt(1.4 * P / rho), rel=1e-15)


def test_dt_single_limits():
    """Each of the limits of P:409-413 alone, on a state where it is the only one that matters."""
    m = mesh(8, 8, 8)
    s = (8, 8, 8)
    z = np.zeros(s)
    # (2) fluid motion: uniform v, cold gas: dt = C L / |v| combined with sound in quadrature
    o = Oracle(m, W.CARTESIAN, W.ISOTHERMAL, W.Params(cfl=0.5))
    o.set_fields(np.ones(s), np.full(s, 0.3), np.full(s, 0.4), z, z)
    o.step_until("DT")
    assert o.time()[1] == pytest.approx(0.5 * 0.125 / math.hypot(0.3, 0.4), rel=1e-14)
    # (4) viscosity: dt4 = L^2 / (4 nu)
    o = Oracle(m, W.CARTESIAN, W.ISOTHERMAL, W.Params(cfl=0.5, nu=0.7))
    o.set_fields(np.ones(s), np.full(s, 1e-9), z, z, z)
    o.step_until("DT")
    assert o.time()[1] == pytest.approx(0.5 * 0.125 ** 2 / (4 * 0.7), rel=1e-12)
    # (3) artificial viscosity: one compressed cell with dv = -0.2: dt3 = L / (4 Cq^2 |dv|) (reading G8)
    vx = z.copy()
    vx[:, :, 4:] = -0.2      # v jumps down between face 3 and face 4: cell 3 is compressed
    o = Oracle(m, W.CARTESIAN, W.ISOTHERMAL, W.Params(cfl=1.0, cvnr2=2.0))
    o.set_fields(np.ones(s), np.full(s, 1e-9), vx, z, z)
    o.step_until("DT")
    i3 = 4 * 2.0 * 0.2 / 0.125
    i2 = 0.2 / 0.125          # cells 4..7 move at -0.2; cell 3 at -0.1 but has the I3 term
    expect = 1.0 / max(math.hypot(i3, 0.1 / 0.125), i2)
    assert o.time()[1] == pytest.approx(expect, rel=1e-9)


def test_dt_fargo_uses_residual_velocity_and_shear_limit():
    """v0 is removed from the CFL; Eq. 73 adds the shear limit C0 / |v0_j/LX_j - v0_j+1/LX_j+1|."""
    bc = (PER, REF, PER)
    m = mesh(16, 6, 1, x=(-math.pi, math.pi), y=(1.0, 2.2), bc=bc)
    prm = W.Params(cfl=0.44, fargo_on=1, gm_star=0.0, shear_c0=0.5)
    o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, prm)
    s = (1, 6, 16)
    rc = m.yc()[None, :, None] * np.ones(s)
    o.set_fields(np.ones(s), np.full(s, 1e-6), 3.0 / rc, np.zeros(s), None)   # huge uniform rotation per ring
    o.step_until("DT")
    lx = rc[0, :, 0] * m.dx
    shear = np.max(np.abs(np.diff((3.0 / rc[0, :, 0]) / lx)))
    assert o.time()[1] == pytest.approx(0.44 * 0.5 / shear, rel=1e-13)
    assert np.allclose(o.active(o.array("v0")[:, :, None])[0, :, 0], 3.0 / rc[0, :, 0], rtol=1e-15)


def test_vmean_is_half_max_plus_min():
    m = mesh(16, 4, 1, x=(-math.pi, math.pi), y=(1.0, 2.0), bc=(PER, REF, PER))
    o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(fargo_on=1))
    r = np.random.default_rng(2)
    vx = r.normal(size=(1, 4, 16))
    o.set_fields(np.ones((1, 4, 16)), np.ones((1, 4, 16)), vx, np.zeros((1, 4, 16)), None)
    o.step_until("VMEAN")
    v0 = o.array("v0")[0, o.ngy:o.ngy + 4]
    assert np.array_equal(v0, 0.5 * (vx[0].max(axis=1) + vx[0].min(axis=1)))   # Eq. 72


# ---------------------------------------------------------------------------- source 7a
def test_src_a_uniform_pressure_leaves_velocity_bitwise():
    o, m, (rho, e, vx, vy, vz) = _box(6)
    o.set_fields(rho, np.full_like(e, 2.5), vx, vy, vz)
    o.step_until("SRC_A")
    for a, b in (("vxb", vx), ("vyb", vy), ("vzb", vz)):
        assert np.array_equal(o.active(o.array(a)), b)


def test_src_a_linear_pressure_closed_form():
    """rho = 1, P = P0 + g*y: dv_y = -dt * g exactly (pins the factor 2/(rho_i + rho_i-1) and the sign)."""
    n = 8
    m = mesh(4, n, 4, bc=(PER, OUT, PER))
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.5, dt_fixed=0.01))
    s = (4, n, 4)
    P = 2.0 + 0.75 * m.yc()[None, :, None] * np.ones(s)
    z = np.zeros(s)
    o.set_fields(np.ones(s), P / 0.5, z, z, z)
    o.step_until("SRC_A")
    vyb = o.active(o.array("vyb"))
    assert np.allclose(vyb[:, 1:, :], -0.01 * 0.75, rtol=1e-12)
    assert np.all(o.active(o.array("vxb")) == 0.0) and np.all(o.active(o.array("vzb")) == 0.0)


def test_src_a_conserves_momentum_along_periodic_direction():
    """Eq. 58: sum_i (rho_i + rho_i-1)/2 * dv_i telescopes to zero for arbitrary P and rho."""
    o, m, (rho, e, vx, vy, vz) = _box(8, seed=4)
    o.step_until("SRC_A")
    for name, v, ax in (("vxb", vx, 2), ("vyb", vy, 1), ("vzb", vz, 0)):
        dv = o.active(o.array(name)) - v
        rbar = 0.5 * (rho + np.roll(rho, 1, axis=ax))
        tot = np.sum(rbar * dv, axis=ax)
        assert np.max(np.abs(tot)) < 1e-13 * np.max(np.abs(rbar * dv)) * 8 + 1e-18
        assert np.max(np.abs(dv)) > 1e-6      # the test is not vacuous


def test_src_a_keplerian_balance_cylindrical():
    """Centrifugal term (Eq. 33, 38) against the star's potential gradient: for v_phi^2 = GM/r and no
    pressure the radial acceleration cancels to second order in dr; each term alone is O(1)."""
    nr = 64
    m = mesh(8, nr, 1, x=(-math.pi, math.pi), y=(0.5, 2.0), z=(-0.5, 0.5), bc=(PER, OUT, PER))
    s = (1, nr, 8)
    rc = m.yc()[None, :, None] * np.ones(s)
    for omf in (0.0, 0.7):
        prm = W.Params(gm_star=1.0, omega_frame=omf, dt_fixed=1.0)
        o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, prm)
        o.set_fields(np.ones(s), np.full(s, 1e-8), rc ** -0.5 - omf * rc, np.zeros(s), None)
        o.step_until("SRC_A")
        acc = o.active(o.array("vyb"))[0, 2:-2, 0]          # dt = 1: the acceleration itself
        rf = m.yedges[2:nr - 2]
        assert np.max(np.abs(acc) * rf ** 2) < 2e-3         # |g| = 1/r^2: cancels to O(dr^2)
        # and the potential term alone has the right sign and size: switch the rotation off
        o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(gm_star=1.0, dt_fixed=1.0))
        o.set_fields(np.ones(s), np.full(s, 1e-8), np.zeros(s), np.zeros(s), None)
        o.step_until("SRC_A")
        acc = o.active(o.array("vyb"))[0, 2:-2, 0]
        assert np.allclose(acc, -1.0 / rf ** 2, rtol=2e-3)


def test_src_a_spherical_balance():
    """Spherical: rigid rotation Omega about the axis, no gravity, frame at rest: the centrifugal
    acceleration is Omega^2 R along cylindrical R, i.e. a_r = Omega^2 r sin^2(theta),
    a_theta = Omega^2 r sin(theta) cos(theta)  (Eqs. 36-37)."""
    nr, nt = 12, 10
    m = mesh(8, nr, nt, x=(-math.pi, math.pi), y=(1.0, 2.0), z=(0.9, 1.5), bc=(PER, OUT, OUT))
    s = (nt, nr, 8)
    r = m.yc()[None, :, None] * np.ones(s)
    th = m.zc()[:, None, None] * np.ones(s)
    Om = 0.8
    o = Oracle(m, W.SPHERICAL, W.ISOTHERMAL, W.Params(dt_fixed=1.0))
    o.set_fields(np.ones(s), np.full(s, 1e-9), Om * r * np.sin(th), np.zeros(s), np.zeros(s))
    o.step_until("SRC_A")
    ar = o.active(o.array("vyb"))[1:-1, 1:-1, 0]
    at = o.active(o.array("vzb"))[1:-1, 1:-1, 0]
    rf = m.yedges[:-1][None, 1:-1]
    thc = m.zc()[1:-1, None]
    rcc = m.yc()[None, 1:-1]
    thf = m.zedges[:-1][1:-1, None]
    assert np.allclose(ar, Om ** 2 * rf * np.sin(thc) ** 2, rtol=5e-3)
    assert np.allclose(at, Om ** 2 * rcc * np.sin(thf) * np.cos(thf), rtol=5e-3, atol=1e-4)
    # same flow seen from the frame rotating at Omega: v = 0, frame term alone must give the same
    o = Oracle(m, W.SPHERICAL, W.ISOTHERMAL, W.Params(dt_fixed=1.0, omega_frame=Om))
    o.set_fields(np.ones(s), np.full(s, 1e-9), np.zeros(s), np.zeros(s), np.zeros(s))
    o.step_until("SRC_A")
    assert np.allclose(o.active(o.array("vyb"))[1:-1, 1:-1, 0], ar, rtol=5e-3)
    assert np.allclose(o.active(o.array("vzb"))[1:-1, 1:-1, 0], at, rtol=5e-3, atol=1e-4)


def test_potential_planet_and_star():
    m = mesh(16, 4, 1, x=(-math.pi, math.pi), y=(0.8, 1.2), z=(-0.5, 0.5), bc=(PER, REF, PER))
    prm = W.Params(gm_star=1.0, planet_mass=1e-3, planet_r=1.0, planet_phi0=0.3, planet_omega=1.0,
                   omega_frame=1.0, planet_eps=0.03, fargo_on=1)
    o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, prm)
    s = (1, 4, 16)
    o.set_fields(np.ones(s), np.ones(s), np.zeros(s), np.zeros(s), None)
    o.step_until("POT")
    phi = o.active(o.array("phi"))[0]
    r = m.yc()[:, None]
    ph = m.xc()[None, :]
    d2 = r ** 2 + 1.0 - 2 * r * np.cos(ph - 0.3)
    assert np.allclose(phi, -1.0 / r - 1e-3 / np.sqrt(d2 + 0.03 ** 2), rtol=1e-13)


# ---------------------------------------------------------------------------- source 7b
def test_src_b_expansion_everywhere_is_a_no_op():
    n = 6
    m = mesh(n, n, n, bc=(OUT, OUT, OUT))
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4, dt_fixed=1e-3))
    s = (n, n, n)
    X = m.xf()[None, None, :] * np.ones(s)
    Y = m.yedges[:-1][None, :, None] * np.ones(s)
    Z = m.zedges[:-1][:, None, None] * np.ones(s)
    rho = rng_fields(s, 3)[0]
    e = np.full(s, 1.7)                                  # uniform pressure: 7a leaves v alone
    o.set_fields(rho, e, 0.3 * X, 0.2 * Y, 0.1 * Z)      # dv >= 0 everywhere (zero in outflow ghosts)
    o.step_until("SRC_B")
    for a, b in (("vxc", "vxb"), ("vyc", "vyb"), ("vzc", "vzb")):
        assert np.array_equal(o.active(o.array(a)), o.active(o.array(b)))
    assert np.array_equal(o.active(o.array("ec")), e)


def test_src_b_hand_stencil():
    """One compressed cell in x: rho = 2, dv = -0.5 in cell 3 -> q = Cq^2 rho dv^2 = 2*2*0.25 = 1.
    Faces 3 and 4 get -+ dt * 2 (q_i - q_i-1)/((rho_i + rho_i-1) dx); cell 3 is heated by dt*q*|dv|/dx."""
    n = 8
    m = mesh(n, 4, 4)
    dt, dx = 1e-2, 1.0 / n
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.0 + 1e-12, dt_fixed=dt, cvnr2=2.0))
    s = (4, 4, n)
    vx = np.zeros(s)
    vx[:, :, 4:] = -0.5
    vx[:, :, 0] = -0.5          # periodic: make the jump back up happen between face 7.. and 0 smoothly
    vx[:, :, 0] = 0.0
    # profile along x faces: 0 0 0 0 -.5 -.5 -.5 -.5 ; wraps -0.5 -> 0 between face 7 and face 0 (expansion)
    z = np.zeros(s)
    o.set_fields(np.full(s, 2.0), np.full(s, 3.0), vx, z, z)
    o.step_until("SRC_B")
    # gamma ~ 1: no pressure; uniform P anyway so 7a changes nothing
    assert np.array_equal(o.active(o.array("vxb")), vx)
    vxc, ec = o.active(o.array("vxc"))[0, 0], o.active(o.array("ec"))[0, 0]
    q = 2.0 * 2.0 * 0.25
    expect_v = vx[0, 0].copy()
    expect_v[3] -= dt * 2.0 * (q - 0.0) / (4.0 * dx)
    expect_v[4] -= dt * 2.0 * (0.0 - q) / (4.0 * dx)
    assert np.allclose(vxc, expect_v, rtol=1e-14, atol=0)
    expect_e = np.full(n, 3.0)
    expect_e[3] -= dt * q * (-0.5) / dx
    assert np.allclose(ec, expect_e, rtol=1e-15)


# ---------------------------------------------------------------------------- source 7c
def test_src_c_uniform_divergence():
    """v = D/3 * (x, y, z) (zero-gradient ghosts; interior cells only): e_d = e_c (1 - a)/(1 + a),
    a = dt (gamma - 1) D / 2 (time-centred -P div v for a gamma law)."""
    n, D, dt, g = 8, 0.9, 0.05, 1.4
    m = mesh(n, n, n, bc=(OUT, OUT, OUT))
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=g, dt_fixed=dt))
    s = (n, n, n)
    X = m.xf()[None, None, :] * np.ones(s)
    Y = m.yedges[:-1][None, :, None] * np.ones(s)
    Z = m.zedges[:-1][:, None, None] * np.ones(s)
    o.set_fields(np.ones(s), np.full(s, 2.0), D / 3 * X, D / 3 * Y, D / 3 * Z)
    o.step_until("SRC_C")
    a = 0.5 * dt * (g - 1.0) * D
    ed = o.active(o.array("ed"))[1:-1, 1:-1, 1:-1]
    assert np.allclose(ed, 2.0 * (1 - a) / (1 + a), rtol=1e-13)


def test_src_c_divergence_uses_exact_surfaces_in_spherical_geometry():
    """v_r = A r in spherical geometry has div v = 3A exactly, and the finite-volume divergence built
    from Tab. 5's exact surfaces and volumes reproduces it to rounding: sum(S v)/V =
    A (r1^3 - r0^3) dphi dcos / ((r1^3 - r0^3)/3 dphi dcos)."""
    nr, nt, A, dt, g = 10, 6, 0.4, 0.02, 1.4
    m = mesh(8, nr, nt, x=(-math.pi, math.pi), y=(1.0, 2.0), z=(1.0, 1.6), bc=(PER, OUT, OUT))
    s = (nt, nr, 8)
    rf = m.yedges[:-1][None, :, None] * np.ones(s)
    o2 = Oracle(m, W.SPHERICAL, W.ADIABATIC, W.Params(gamma=g, dt_fixed=dt))
    o2.set_fields(np.ones(s), np.full(s, 2.0), np.zeros(s), A * rf, np.zeros(s))
    o2.step_until("SRC_C")
    # uniform pressure, no rotation, v_theta = 0: 7a and 7b leave v_r alone
    assert np.allclose(o2.active(o2.array("vyc")), A * rf, rtol=1e-14)
    a = 0.5 * dt * (g - 1.0) * 3 * A
    ed = o2.active(o2.array("ed"))[:, 1:-1, :]
    assert np.allclose(ed, 2.0 * (1 - a) / (1 + a), rtol=1e-12)


# ---------------------------------------------------------------------------- Eq. 36: the v_theta^2 / r term
def _sph_src_a(nphi, nr, nth, vphi, vth, om=0.0):
    """One 7a sub-step (dt = 1, uniform pressure, no potential) on a spherical mesh with v_phi(phi, r, theta) and
    v_theta(phi, r, theta) sampled at their own faces; returns the mesh and the radial / polar accelerations."""
    m = mesh(nphi, nr, nth, x=(-math.pi, math.pi), y=(1.0, 2.0), z=(0.5 * math.pi - 0.6, 0.5 * math.pi + 0.4),
             bc=(PER, OUT, OUT))
    s = (nth, nr, nphi)
    one = np.ones(s)
    pf, pc = m.xf()[None, None, :] * one, m.xc()[None, None, :] * one
    rc = m.yc()[None, :, None] * one
    tc, tf = m.zc()[:, None, None] * one, m.zedges[:-1][:, None, None] * one
    o = Oracle(m, W.SPHERICAL, W.ISOTHERMAL, W.Params(dt_fixed=1.0, omega_frame=om))
    vz_in = vth(pc, rc, tf)
    o.set_fields(one, np.full(s, 1e-9), vphi(pf, rc, tc), np.zeros(s), vz_in)
    o.step_until("SRC_A")
    return m, o.active(o.array("vyb")), o.active(o.array("vzb")) - vz_in   # dt = 1, v_r = 0: the accelerations


def _eq36_error(n, vphi, vth, om=0.0):
    """max |a_r - (v_phi^t^2 + v_theta^2)/r| over the interior radial faces, relative to max |a_r| (Eq. 36),
    and the same for Eq. 37's (v_phi^t)^2 cot(theta) / r on the polar faces; v^t = v + Omega_f r sin(theta)."""
    m, ar, at = _sph_src_a(2 * n, n, n, vphi, vth, om)
    P = m.xc()[None, None, :]
    rf, rc = m.yedges[:-1][None, :, None], m.yc()[None, :, None]
    tc, tf = m.zc()[:, None, None], m.zedges[:-1][:, None, None]
    ex_r = ((vphi(P, rf, tc) + om * rf * np.sin(tc)) ** 2 + vth(P, rf, tc) ** 2) / rf
    ex_t = (vphi(P, rc, tf) + om * rc * np.sin(tf)) ** 2 / (np.tan(tf) * rc)
    I = (slice(1, -1), slice(1, -1), slice(None))
    return (np.max(np.abs(ar[I] - ex_r[I])) / np.max(np.abs(ex_r[I])),
            np.max(np.abs(at[I] - ex_t[I])) / max(np.max(np.abs(ex_t[I])), 1e-300))


def test_src_a_eq36_rigid_rotation_about_a_perpendicular_axis():
    """Rigid rotation Omega about the x axis (perpendicular to the polar axis): v_r = 0, v_theta = -Omega r sin(phi),
    v_phi = -Omega r cos(theta) cos(phi).  The radial equation (Eq. 36) must then supply the centripetal term
    |v|^2 / r = Omega^2 r (1 - sin^2(theta) cos^2(phi)) = Omega^2 times the distance to the axis, projected on r;
    Eq. 37 supplies v_phi^2 cot(theta) / r.  Second-order in the mesh spacing: the 4-point averages of Eq. 38 are
    centred on the face.  A dropped v_theta^2, a radius taken at the cell centre or a one-sided average leaves an
    O(1) or first-order error and fails the bounds and the convergence order below."""
    Om = 0.7
    vphi = lambda p, r, t: -Om * r * np.cos(t) * np.cos(p)
    vth = lambda p, r, t: -Om * r * np.sin(p) + 0.0 * t
    e1, e2 = _eq36_error(16, vphi, vth), _eq36_error(32, vphi, vth)
    assert e2[0] < 1.5e-3 and e2[1] < 3e-3, (e1, e2)          # second-order truncation only
    assert 3.0 < e1[0] / e2[0] < 5.0 and 3.0 < e1[1] / e2[1] < 5.0, (e1, e2)   # first-order mistakes give 2
    # physical reading at one face: centripetal acceleration of the rotation about x
    m, ar, _ = _sph_src_a(64, 32, 32, vphi, vth)
    k, j, i = 9, 11, 20
    r, t, p = m.yedges[j], m.zc()[k], m.xc()[i]
    x = np.array([r * math.sin(t) * math.cos(p), r * math.sin(t) * math.sin(p), r * math.cos(t)])
    perp = x - np.array([x[0], 0.0, 0.0])                      # from the x axis to the point
    assert ar[k, j, i] == pytest.approx(Om ** 2 * float(perp @ x) / r, rel=2e-3)


def test_src_a_eq36_v_theta_alone_on_a_meridian_flow():
    """v_phi = 0 everywhere, frame at rest: the only term left in Eq. 36 is v_theta^2 / r.  v_theta varies with r,
    theta AND phi, so each leg of the 4-point average (j, j-1) x (k, k+1) and the position of 1/r (the radial FACE)
    matters: a_r -> v_theta(phi_c, r_face, theta_c)^2 / r_face at second order; Eq. 37 gives exactly zero."""
    vphi = lambda p, r, t: 0.0 * (p + r + t)
    vth = lambda p, r, t: 0.3 * r ** 1.5 * (1.0 + 0.5 * np.sin(3.0 * t)) * (1.0 + 0.4 * np.cos(p))
    e1, e2 = _eq36_error(16, vphi, vth)[0], _eq36_error(32, vphi, vth)[0]
    assert e2 < 2e-3, (e1, e2)
    assert 3.0 < e1 / e2 < 5.0, (e1, e2)
    _, _, at = _sph_src_a(16, 8, 8, vphi, vth)
    assert not np.any(at[1:-1, 1:-1])   # v_theta untouched bit for bit: no v_phi, uniform P


def test_src_a_eq36_with_both_terms_and_a_rotating_frame():
    """Both terms together with Omega_f != 0: (v_phi + Omega_f r sin(theta))^2 + v_theta^2 over r (Eqs. 36, 38)."""
    vphi = lambda p, r, t: 0.2 * r ** -0.5 * np.sin(t) * (1.0 + 0.3 * np.sin(p))
    vth = lambda p, r, t: 0.25 * r * np.cos(2.0 * t) * (1.0 + 0.3 * np.cos(2.0 * p))
    e1, e2 = _eq36_error(16, vphi, vth, om=0.35), _eq36_error(32, vphi, vth, om=0.35)
    assert e2[0] < 2e-3 and e2[1] < 4e-3, (e1, e2)
    assert 3.0 < e1[0] / e2[0] < 5.0 and 3.0 < e1[1] / e2[1] < 5.0, (e1, e2)
