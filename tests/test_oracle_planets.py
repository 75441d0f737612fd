"""Pins of the oracle's live planets (section 3.8, Eq. 109, Tab. 3 P:754-764;
DESIGN.md reading G33).  CPU only.  Each pin is something the paper or mechanics fixes, not the oracle's own formula:
* Cash-Karp is fifth order: on an eccentric Kepler orbit the error against the exact solution (Kepler's equation
  solved here) falls by ~2^5 when h is halved -- one wrong entry of Tab. 3 lowers the order;
* a body on the circular orbit whose rate is the frame's stays at rest; in a slower frame it drifts at Omega_K - Omega_f
  (Coriolis and centrifugal signs);
* two equal masses without a star circle their centre of mass at omega^2 = G (2m) / d^3 (planet-planet term);
* gas force: one loaded cell gives G dm (x_c - x_p) / (d^2 + eps^2)^(3/2) with Tab. 5's volume; a ring seen from its
  axis gives M dz / d^3 exactly; an axisymmetric disk gives no torque, and no force at all once its axisymmetric
  part is removed.
"""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W

PER = (W.PERIODIC,) * 2
REF = (W.REFLECTING,) * 2


def _disk_mesh(nphi=32, nr=16, nz=1, r=(0.5, 2.0), z=(-0.5, 0.5)):
    return W.Mesh(nphi, nr, nz, -math.pi, math.pi, W.uedges(r[0], r[1], nr), W.uedges(z[0], z[1], nz), (PER, REF, REF if nz > 1 else PER))


def _ctx(om=0.0, gm_star=1.0, mesh=None, geometry=W.CYLINDRICAL):
    m = mesh or _disk_mesh()
    o = Oracle(m, geometry, W.ISOTHERMAL, W.Params(omega_frame=om, gm_star=gm_star))
    shape = (m.nz, m.ny, m.nx)
    o.set_fields(np.ones(shape), np.full(shape, 0.05), np.zeros(shape), np.zeros(shape), np.zeros(shape) if m.nz > 1 else None)
    return m, o


def _kepler_exact(a, e, t, gm=1.0):
    """Position on a Kepler ellipse (pericentre on +x at t = 0), Kepler's equation by Newton iteration."""
    n = math.sqrt(gm / a ** 3)
    M = n * t
    E = M
    for _ in range(50):
        E -= (E - e * math.sin(E) - M) / (1.0 - e * math.cos(E))
    return a * (math.cos(E) - e), a * math.sqrt(1 - e * e) * math.sin(E)


def _integrate_kepler(nsteps, e=0.3, a=1.0):
    _, o = _ctx()
    rp = a * (1 - e)
    vp = math.sqrt((1 + e) / (a * (1 - e)))
    o.set_planets([1e-30], [0.0], [rp, 0, 0], [0, vp, 0], force_mode=0)
    T = 2 * math.pi * a ** 1.5
    tend = 0.7 * T
    h = tend / nsteps
    for _ in range(nsteps):
        o.planets_rk5(h)
    pos, vel, _ = o.get_planets()
    xe, ye = _kepler_exact(a, e, tend)
    return math.hypot(pos[0, 0] - xe, pos[0, 1] - ye), pos, vel


def test_cash_karp_is_fifth_order_on_an_eccentric_kepler_orbit():
    e1, _, _ = _integrate_kepler(100)
    e2, _, _ = _integrate_kepler(200)
    e3, pos, vel = _integrate_kepler(400)
    assert e1 < 1e-4 and e3 < 1e-7
    assert 20.0 < e1 / e2 < 45.0 and 20.0 < e2 / e3 < 45.0          # 2^5 = 32
    # energy and angular momentum of the end state
    r = math.hypot(pos[0, 0], pos[0, 1])
    en = 0.5 * (vel[0, 0] ** 2 + vel[0, 1] ** 2) - 1.0 / r
    assert abs(en + 0.5) < 1e-8
    assert abs(pos[0, 0] * vel[0, 1] - pos[0, 1] * vel[0, 0] - math.sqrt(1 - 0.09)) < 1e-8


def test_weights_sum_to_one_free_motion_is_exact():
    """No forces (no star, massless frame at rest): x advances by exactly h v (sum b_i = 1, k_i = v for all i)."""
    _, o = _ctx(gm_star=0.0)
    o.set_planets([1e-30], [0.0], [1.0, 2.0, 3.0], [0.25, -0.5, 0.125], force_mode=0)
    o.planets_rk5(0.5)
    pos, vel, _ = o.get_planets()
    assert np.allclose(pos[0], [1.125, 1.75, 3.0625], rtol=0, atol=1e-15) and np.array_equal(vel[0], [0.25, -0.5, 0.125])


def test_corotating_planet_stays_at_rest_and_drifts_in_a_slower_frame():
    rp = 1.3
    omk = rp ** -1.5
    _, o = _ctx(om=omk)
    o.set_planets([1e-30], [0.0], [rp, 0, 0], [0, 0, 0], force_mode=0)
    for _ in range(200):
        o.planets_rk5(0.05)
    pos, vel, _ = o.get_planets()
    assert np.max(np.abs(pos[0] - [rp, 0, 0])) < 1e-12 and np.max(np.abs(vel[0])) < 1e-12
    omf = 0.4 * omk
    _, o = _ctx(om=omf)
    o.set_planets([1e-30], [0.0], [rp, 0, 0], [0, rp * (omk - omf), 0], force_mode=0)
    n, h = 300, 0.02
    for _ in range(n):
        o.planets_rk5(h)
    pos, _, _ = o.get_planets()
    ang = (omk - omf) * n * h
    assert abs(pos[0, 0] - rp * math.cos(ang)) < 1e-9 and abs(pos[0, 1] - rp * math.sin(ang)) < 1e-9


def test_two_equal_masses_circle_their_centre_of_mass():
    gm, d = 0.5, 2.0
    w = math.sqrt(2 * gm / d ** 3)
    _, o = _ctx(gm_star=0.0)
    o.set_planets([gm, gm], [0.0, 0.0], [1, 0, 0, -1, 0, 0], [0, w, 0, 0, -w, 0], force_mode=0)
    n, h = 400, 0.01
    for _ in range(n):
        o.planets_rk5(h)
    pos, _, _ = o.get_planets()
    ang = w * n * h
    assert np.max(np.abs(pos[0] - [math.cos(ang), math.sin(ang), 0])) < 1e-10
    assert np.max(np.abs(pos[0] + pos[1])) < 1e-13


def test_gas_force_of_one_loaded_cell_by_hand():
    m, o = _ctx(mesh=_disk_mesh(nphi=24, nr=10, nz=4, z=(-0.2, 0.2)))
    shape = (m.nz, m.ny, m.nx)
    rho = np.zeros(shape)
    k, j, i = 2, 6, 5
    rho[k, j, i] = 3.0
    o.set_fields(rho, np.full(shape, 0.05), np.zeros(shape), np.zeros(shape), np.zeros(shape))
    xp, eps = np.array([0.9, -0.3, 0.07]), 0.11
    o.set_planets([1e-3], [eps], xp, [0, 0, 0], force_mode=1)
    r0, r1 = m.yedges[j], m.yedges[j + 1]
    vol = 0.5 * (r1 * r1 - r0 * r0) * m.dx * (m.zedges[k + 1] - m.zedges[k])          # Tab. 5, cylindrical
    rc, phic, zc = 0.5 * (r0 + r1), m.xc()[i], 0.5 * (m.zedges[k] + m.zedges[k + 1])
    dvec = np.array([rc * math.cos(phic), rc * math.sin(phic), zc]) - xp
    expect = 3.0 * vol * dvec / (dvec @ dvec + eps * eps) ** 1.5
    assert np.allclose(o.gas_force(0), expect, rtol=1e-13, atol=0)


def test_ring_seen_from_its_axis_spherical_mesh():
    """Every cell of a ring (fixed r, theta) is at the same distance from a planet on the axis: F_z = M dz / d^3,
    F_x = F_y = 0 by symmetry -- exact for the discrete sum too (spherical volumes of Tab. 5)."""
    nphi, nr, nth = 48, 8, 6
    m = W.Mesh(nphi, nr, nth, -math.pi, math.pi, W.uedges(0.8, 1.6, nr), W.uedges(1.2, 1.8, nth), (PER, REF, REF))
    o = Oracle(m, W.SPHERICAL, W.ISOTHERMAL, W.Params(gm_star=1.0))
    shape = (nth, nr, nphi)
    rho = np.zeros(shape)
    k, j = 1, 5
    rho[k, j, :] = 2.0
    o.set_fields(rho, np.full(shape, 0.05), np.zeros(shape), np.zeros(shape), np.zeros(shape))
    zp = 0.45
    o.set_planets([1e-3], [0.0], [0, 0, zp], [0, 0, 0], force_mode=1)
    r0, r1, t0, t1 = m.yedges[j], m.yedges[j + 1], m.zedges[k], m.zedges[k + 1]
    M = 2.0 * (r1 ** 3 - r0 ** 3) / 3.0 * (math.cos(t0) - math.cos(t1)) * 2 * math.pi
    rc, tc = 0.5 * (r0 + r1), 0.5 * (t0 + t1)
    R, z = rc * math.sin(tc), rc * math.cos(tc)
    F = o.gas_force(0)
    assert abs(F[2] - M * (z - zp) / (R * R + (z - zp) ** 2) ** 1.5) < 1e-13 * abs(F[2])
    assert abs(F[0]) < 1e-14 * abs(F[2]) * nphi and abs(F[1]) < 1e-14 * abs(F[2]) * nphi


@pytest.mark.parametrize("mode", [1, 2])
def test_axisymmetric_disk_exerts_no_torque_and_nothing_once_removed(mode):
    m, o = _ctx(mesh=_disk_mesh(nphi=64, nr=24))
    shape = (m.nz, m.ny, m.nx)
    rho = np.broadcast_to((m.yc() ** -1.5)[None, :, None], shape).copy()
    o.set_fields(rho, np.full(shape, 0.05), np.zeros(shape), np.zeros(shape), None)
    phi_p = m.xc()[20]                                   # on a cell-centre azimuth: the discrete disk is symmetric about it
    xp = np.array([1.1 * math.cos(phi_p), 1.1 * math.sin(phi_p), 0.0])
    o.set_planets([1e-3], [0.05], xp, [0, 0, 0], force_mode=mode)
    F = o.gas_force(0)
    scale = float(np.sum(rho[0] * 0.5 * (m.yedges[1:] ** 2 - m.yedges[:-1] ** 2)[:, None] * m.dx))   # total mass / r^2 ~ 1
    torque = xp[0] * F[1] - xp[1] * F[0]
    assert abs(torque) < 1e-13 * scale
    if mode == 1:
        assert abs(F @ xp) > 1e-3 * scale                # the radial pull of the (outer-heavy) disk is there ...
    else:
        assert np.max(np.abs(F)) < 1e-13 * scale         # ... and gone with the axisymmetric part


def test_live_planet_potential_is_the_fixed_orbit_one_at_the_same_place():
    m = _disk_mesh(nphi=40, nr=12, nz=6, z=(-0.3, 0.3))
    prm = W.Params(gm_star=1.0, planet_mass=2e-3, planet_r=1.2, planet_phi0=0.0, planet_omega=0.0, planet_eps=0.04)
    shape = (m.nz, m.ny, m.nx)
    f = (np.ones(shape), np.full(shape, 0.05), np.zeros(shape), np.zeros(shape), np.zeros(shape))
    a = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, prm); a.set_fields(*f); a.run_stage("POT")
    b = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(gm_star=1.0)); b.set_fields(*f)
    b.set_planets([2e-3], [0.04], [1.2, 0.0, 0.0], [0, 0, 0], force_mode=0); b.run_stage("POT")
    assert np.array_equal(a.array("phi"), b.array("phi"))


def test_one_update_kicks_the_planet_by_dt_times_the_gas_acceleration():
    m = _disk_mesh(nphi=48, nr=20)
    shape = (m.nz, m.ny, m.nx)
    r = m.yc()[None, :, None] * np.ones(shape)
    phi = m.xc()[None, None, :] * np.ones(shape)
    rho = 1e-2 * r ** -0.5 * (1.0 + 0.5 * np.cos(phi - 0.7))          # lopsided: a net force
    out = []
    for mode in (0, 1):
        o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(gm_star=1.0, dt_fixed=1e-3))
        o.set_fields(rho, 0.05 * r ** -0.5, r ** -0.5, np.zeros(shape), None)
        o.set_planets([1e-4], [0.05], [1.0, 0, 0], [0, 1.0, 0], force_mode=mode, gconst=1.0)
        F = o.gas_force(0)
        o.step(1)
        out.append(o.get_planets())
    dv = out[1][1][0] - out[0][1][0]
    assert np.allclose(dv[:2], 1e-3 * F[:2], rtol=2e-3, atol=1e-12) and np.allclose(out[1][2][0], F)
    assert np.max(np.abs(out[0][2])) == 0.0


# ---- cell 5b: change of the frame's rotation rate, Eq. 44 ---------------------------------------------
def test_eq44_leaves_the_inertial_azimuthal_velocity_and_angular_momentum_alone():
    nphi, nr, nth = 16, 10, 6
    m = W.Mesh(nphi, nr, nth, -math.pi, math.pi, W.uedges(0.6, 1.8, nr), W.uedges(1.3, 1.8, nth), (PER, REF, REF))
    om0, om1 = 0.35, 1.15
    o = Oracle(m, W.SPHERICAL, W.ISOTHERMAL, W.Params(gm_star=1.0, omega_frame=om0))
    shape = (nth, nr, nphi)
    rng = np.random.default_rng(4)
    rho = 1.0 + 0.3 * rng.uniform(-1, 1, shape)
    vx, vy, vz = (0.2 * rng.uniform(-1, 1, shape) for _ in range(3))
    o.set_fields(rho, np.full(shape, 0.05), vx, vy, vz)
    R = (m.yc()[None, :, None] * np.sin(m.zc())[:, None, None]) * np.ones(shape)      # r sin(theta) at the phi face
    before = vx + om0 * R
    o.set_omega_frame(om1)
    r1, _, vx1, vy1, vz1 = o.get_fields()
    assert np.max(np.abs((vx1 + om1 * R) - before)) < 1e-15 * np.max(np.abs(before))
    assert np.array_equal(vy1, vy) and np.array_equal(vz1, vz) and np.array_equal(r1, rho)
    # "trivially conserves angular momentum to machine accuracy": Tab. 2's momentum, face-mean density
    rf = 0.5 * (rho + np.roll(rho, 1, axis=2))
    L0, L1 = np.sum(rf * R * before), np.sum(rf * R * (vx1 + om1 * R))
    assert abs(L1 - L0) < 1e-15 * abs(L0) * 10


def test_a_disk_in_balance_stays_in_balance_across_a_change_of_frame():
    """Keplerian, cold, axisymmetric disk: three updates in the frame om1 reached through Eq. 44 from om0 give the
    fields of the same disk set up in the frame om1 directly (to rounding: the correction is one subtraction)."""
    m = _disk_mesh(nphi=24, nr=20)
    shape = (1, m.ny, m.nx)
    r = m.yc()[None, :, None] * np.ones(shape)
    om0, om1 = 0.2, 0.8
    out = []
    for start in (om0, om1):
        o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(gm_star=1.0, omega_frame=start, fargo_on=1))
        o.set_fields(r ** -0.5, 1e-3 * r ** -0.5, r ** -0.5 - start * r, np.zeros(shape), None)
        if start != om1:
            o.set_omega_frame(om1)
        o.step(3)
        out.append(o.get_fields())
    for a, b in zip(out[0][:4], out[1][:4]):
        assert np.max(np.abs(a - b)) < 1e-13 * max(1.0, np.max(np.abs(b)))
    assert np.max(np.abs(out[0][3][:, 3:-3])) < 2e-3          # and it is a balance up to the O(dr^2) of the 20-cell mesh


def test_live_planet_is_carried_into_the_new_frame():
    rp = 1.25
    omk = rp ** -1.5
    _, o = _ctx(om=omk)
    o.set_planets([1e-30], [0.0], [rp, 0, 0], [0, 0, 0], force_mode=0)       # at rest in its corotating frame
    for _ in range(50):
        o.planets_rk5(0.04)
    om1 = 0.3 * omk
    o.set_omega_frame(om1)
    n, h = 200, 0.03
    for _ in range(n):
        o.planets_rk5(h)
    pos, vel, _ = o.get_planets()
    ang = (omk - om1) * n * h
    assert abs(pos[0, 0] - rp * math.cos(ang)) < 1e-9 and abs(pos[0, 1] - rp * math.sin(ang)) < 1e-9


def test_fixed_orbit_planet_keeps_its_azimuth_when_the_frame_changes():
    m = _disk_mesh(nphi=32, nr=12)
    shape = (1, m.ny, m.nx)
    prm = W.Params(gm_star=1.0, planet_mass=1e-3, planet_r=1.1, planet_phi0=0.3, planet_omega=0.9, planet_eps=0.05,
                   omega_frame=0.5, dt_fixed=0.01)
    f = (np.ones(shape), np.full(shape, 0.05), np.zeros(shape), np.zeros(shape), None)
    a = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, prm); a.set_fields(*f); a.step(4)
    a.run_stage("POT"); phi_before = a.array("phi").copy()
    b = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, prm); b.set_fields(*f); b.step(4)
    b.set_omega_frame(0.1); b.run_stage("POT")
    assert np.max(np.abs(b.array("phi") - phi_before)) < 1e-14
    with pytest.raises(ValueError):
        Oracle(mesh_cart(), W.CARTESIAN, W.ADIABATIC, W.Params()).set_omega_frame(0.5)


def mesh_cart():
    return W.Mesh(8, 8, 1, 0.0, 1.0, W.uedges(0.0, 1.0, 8), np.array([0.0, 1.0]))
