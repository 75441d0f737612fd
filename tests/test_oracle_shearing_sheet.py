"""Pins of the oracle's shearing-sheet geometry (NEXT-1, second half): Tab. 1/Tab. 2 rows "Shearing sheet"
 and the source terms of Eqs. 28-30; reading G32 of DESIGN.md.  CPU only.

What fixes the implementation here is the physics the paper's equations state, not the oracle's own formula:
* Eq. 29 vanishes on v_x = 2 A y, v_y = 0: that flow is steady, for any A (pins the ratio 4 A Omega / 2 Omega, the
  y position of the term and the four-point average);
* a uniform kick on top of it oscillates at the epicyclic frequency kappa^2 = 4 Omega (Omega + A) with the
  amplitude ratio 2 Omega / kappa (pins the 2 Omega of Eq. 29 AND the 2 Omega y of Tab. 2, signs included);
* the sum of Tab. 2's X momentum rho (v_x + 2 Omega_f y) is conserved to rounding, that of rho v_x is not;
* with orbital advection a sheared profile is shifted by whole cells exactly (Eq. 69) in every row.
"""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W
from helpers import mesh, rng_fields

PER = (W.PERIODIC,) * 2
REF = (W.REFLECTING,) * 2


def _sheet(nx, ny, nz, A, om, eos=W.ADIABATIC, ybc=REF, x=(0.0, 1.0), y=(-0.5, 0.5), z=(0.0, 1.0), **kw):
    m = mesh(nx, ny, nz, x=x, y=y, z=z, bc=(PER, ybc, PER))
    p = W.Params(gamma=1.4, omega_frame=om, oort_a=A, **kw)
    return m, Oracle(m, W.SHEARING_SHEET, eos, p)


def _shear_flow(m, A):
    shape = (m.nz, m.ny, m.nx)
    return np.broadcast_to((2.0 * A * m.yc())[None, :, None], shape).copy()


@pytest.mark.parametrize("A,om", [(-0.75, 1.0), (-0.3, 1.7), (0.4, -0.9)])
@pytest.mark.parametrize("fargo", [0, 1])
def test_unperturbed_shear_flow_is_steady(A, om, fargo):
    """Away from the walls: a reflecting wall mirrors v_x, which breaks the linear profile in the ghost rows, so 7a
    leaves a velocity on the wall face until the ghost fill of cell 9 and 7b/7c heat the first row (the order of
    Fig. 2); that disturbance travels inward by at most 3 rows per update (stencils of 7a-7c and of one sweep)."""
    m, o = _sheet(8, 32, 4, A, om, fargo_on=fargo)
    shape = (m.nz, m.ny, m.nx)
    rho, e = np.full(shape, 1.3), np.full(shape, 0.9)
    vx = _shear_flow(m, A)
    z = np.zeros(shape)
    o.set_fields(rho, e, vx, z, z.copy())
    o.step(3)
    r1, e1, vx1, vy1, vz1 = o.get_fields()
    c = slice(10, 22)
    assert np.max(np.abs(vx1 - vx)[:, c]) < 1e-14 and np.max(np.abs(vy1[:, c])) < 1e-14 and np.max(np.abs(vz1)) == 0.0
    assert np.max(np.abs(r1 - rho)[:, c]) < 1e-14 and np.max(np.abs(e1 - e)[:, c]) < 1e-14
    assert np.max(np.abs(e1 - e)[:, :2]) > 1e-6          # ... and the wall rows do feel it


def test_a_different_shear_rate_is_not_steady():
    """The steadiness test has teeth: v_x = 2.2 A y is accelerated in y at the rate 2 Omega * 0.2 A y."""
    A, om = -0.75, 1.0
    m, o = _sheet(8, 16, 4, A, om, dt_fixed=1e-3)
    shape = (m.nz, m.ny, m.nx)
    vx = 1.1 * _shear_flow(m, A)
    z = np.zeros(shape)
    o.set_fields(np.ones(shape), np.ones(shape), vx, z, z.copy())
    o.step(1)
    vy = o.get_fields()[3]
    ye = m.yedges[:-1]
    expect = 1e-3 * 2.0 * om * (0.1 * 2.0 * A * ye)          # dt * (2 Om * 1.1 * 2 A y - 4 A Om y)
    assert np.allclose(vy[0, 2:-2, 0], expect[2:-2], rtol=1e-5, atol=1e-16)   # transport moves it at O(dt v_y)


def _epicycle(A, om, dt, u0=1e-3, ny=48):
    """Uniform kick u0 on the shear flow of a cold sheet; returns (t, u, w) at the central row after one period."""
    m, o = _sheet(4, ny, 1, A, om, eos=W.ISOTHERMAL, x=(0.0, 40.0), dt_fixed=dt)
    shape = (1, ny, 4)
    vx = _shear_flow(m, A) + u0
    o.set_fields(np.ones(shape), np.full(shape, 1e-4), vx, np.zeros(shape), np.zeros(shape))
    kappa = math.sqrt(4.0 * om * (om + A))
    n = int(round(2.0 * math.pi / kappa / dt))
    us, ws, ts = [], [], []
    j = ny // 2
    for q in range(4):                       # quarter periods
        o.step(n // 4)
        f = o.get_fields()
        t = o.time()[0]
        # v_y lives on the lower Y face of row j (y = ye[j]); v_x at the row centre
        us.append(f[2][0, j, 0] - 2.0 * A * m.yc()[j]); ws.append(f[3][0, j, 0]); ts.append(t)
    return kappa, np.array(ts), np.array(us), np.array(ws)


@pytest.mark.parametrize("A,om", [(-0.75, 1.0), (-0.5, 1.0), (-0.3, 1.6)])
def test_epicyclic_oscillation_frequency_and_amplitude(A, om):
    u0 = 1e-3
    errs = []
    for dt in (8e-3, 4e-3):
        kappa, t, u, w = _epicycle(A, om, dt, u0)
        ue = u0 * np.cos(kappa * t)
        we = (2.0 * om / kappa) * u0 * np.sin(kappa * t)
        errs.append(max(np.max(np.abs(u - ue)), np.max(np.abs(w - we))) / u0)
    assert errs[0] < 0.05 and errs[1] < 0.025          # the operator split is first order in dt ...
    assert errs[1] < 0.62 * errs[0]                    # ... and converges to the closed form


def test_wrong_sign_or_factor_would_fail_the_epicycle():
    """Sanity of the pin itself: the closed form with kappa^2 = 4 Om (Om - A) or amplitude Om/kappa is far off."""
    A, om, u0 = -0.5, 1.0, 1e-3
    kappa, t, u, w = _epicycle(A, om, 4e-3, u0)
    bad_k = math.sqrt(4.0 * om * (om - A))
    assert np.max(np.abs(u - u0 * np.cos(bad_k * t))) / u0 > 0.3
    assert np.max(np.abs(w - (om / kappa) * u0 * np.sin(kappa * t))) / u0 > 0.3


def test_tab2_x_momentum_is_conserved_to_rounding():
    A, om = -0.75, 1.3
    m, o = _sheet(8, 12, 6, A, om)
    shape = (m.nz, m.ny, m.nx)
    rho, e, vx, vy, vz = rng_fields(shape, seed=5, vamp=0.2)
    vx = vx + _shear_flow(m, A)
    o.set_fields(rho, e, vx, vy, vz)

    def sums():
        r, _, ux, _, _ = o.get_fields()
        uc = 0.5 * (ux + np.roll(ux, -1, axis=2))
        y = m.yc()[None, :, None]
        return float(np.sum(r * (uc + 2.0 * om * y))), float(np.sum(r * uc)), float(np.sum(r))

    p0, c0, m0 = sums()
    o.step(5)
    p1, c1, m1 = sums()
    scale = float(np.sum(np.abs(rho) * (np.abs(vx) + 2.0 * abs(om) * 0.5)))
    assert abs(m1 - m0) < 1e-13 * m0
    assert abs(p1 - p0) < 2e-14 * scale
    assert abs(c1 - c0) > 1e-6 * scale          # the plain Cartesian momentum is NOT what is conserved


def test_source_term_of_eq29_by_hand_on_a_small_mesh():
    """7a of the sheet minus 7a of the plain Cartesian mesh = dt (2 Om <v_x> - 4 A Om y) on the Y faces, nothing else."""
    A, om, dt = -0.6, 1.2, 0.01
    m, o = _sheet(4, 6, 4, A, om, ybc=PER)
    oc = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4))
    shape = (m.nz, m.ny, m.nx)
    f = rng_fields(shape, seed=9)
    out = []
    for c in (o, oc):
        c.set_fields(*f)
        c.run_stage("BC1"); c.set_dt(dt); c.run_stage("SRC_A")
        out.append([c.active(c.array(n)) for n in ("vxb", "vyb", "vzb")])
    vx = f[2]
    vxa = 0.25 * (vx + np.roll(vx, -1, 2) + np.roll(vx, 1, 1) + np.roll(np.roll(vx, -1, 2), 1, 1))
    ye = m.yedges[:-1][None, :, None]
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][2], out[1][2])      # Eqs. 28, 30
    assert np.allclose(out[0][1] - out[1][1], dt * (2 * om * vxa - 4 * A * om * ye), rtol=0, atol=1e-15)


def test_sheet_without_rotation_is_the_cartesian_mesh_bit_for_bit():
    m, o = _sheet(6, 8, 4, 0.0, 0.0, ybc=PER)
    oc = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4))
    f = rng_fields((m.nz, m.ny, m.nx), seed=3)
    for c in (o, oc):
        c.set_fields(*f); c.step(3)
    for a, b in zip(o.get_fields(), oc.get_fields()):
        assert np.array_equal(a, b)


def test_orbital_advection_shifts_every_row_by_whole_cells():
    """v_x = 2 A y with 2 A dy dt / dx = 2: row j moves by (2 j + 1 - ny) cells per update (Eq. 69), exactly
    (rows away from the walls, see test_unperturbed_shear_flow_is_steady)."""
    A, om, nx, ny = -0.75, 1.0, 32, 24
    dx, dy = 1.0 / nx, 1.0 / ny
    dt = 2.0 * dx / (2.0 * abs(A) * dy)
    m, o = _sheet(nx, ny, 1, A, om, fargo_on=1, dt_fixed=dt)
    shape = (1, ny, nx)
    rho = 1.0 + 0.3 * np.sin(2 * np.pi * m.xc())[None, None, :] * np.ones(shape)
    e = np.full(shape, 1.0)                                   # uniform pressure: no force
    vx = _shear_flow(m, A)
    o.set_fields(rho, e, vx, np.zeros(shape), np.zeros(shape))
    nstep = 2
    o.step(nstep)
    r1, e1, vx1, vy1, _ = o.get_fields()
    for j in range(8, 16):
        s = -(2 * j + 1 - ny) * nstep                          # A < 0: rows above the centre move to -x
        assert np.max(np.abs(r1[0, j] - np.roll(rho[0, j], s))) < 1e-11, j
        assert np.max(np.abs(r1[0, j] - np.roll(rho[0, j], s + 1))) > 1e-2, j
    assert np.max(np.abs(vx1 - vx)[:, 8:16]) < 1e-11 and np.max(np.abs(vy1[:, 8:16])) < 1e-11


def test_sheet_needs_a_periodic_x_axis():
    m = mesh(8, 8, 1, bc=((W.OUTFLOW,) * 2, REF, PER))
    with pytest.raises(ValueError):
        Oracle(m, W.SHEARING_SHEET, W.ADIABATIC, W.Params(omega_frame=1.0, oort_a=-0.75))
