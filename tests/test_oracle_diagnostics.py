"""Pins of the oracle's diagnostics (sum reductions over the mesh: "the mass or angular momentum"): closed-form
volumes of Tab. 5's cells summed over the mesh, rigid rotation, and the conservation to rounding that the paper
states for mass and (angular) momentum ("conserves mass and angular momentum to computer accuracy").  CPU only."""
import math

import numpy as np

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W
from helpers import mesh, rng_fields

PER = (W.PERIODIC,) * 2
REF = (W.REFLECTING,) * 2


def test_mass_and_energy_of_a_uniform_state_are_density_times_the_exact_volume():
    # Cartesian box
    m = mesh(6, 5, 4, x=(0.0, 2.0), y=(1.0, 1.5), z=(-1.0, 2.0))
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params())
    sh = (4, 5, 6)
    o.set_fields(np.full(sh, 1.7), np.full(sh, 0.6), np.zeros(sh), np.zeros(sh), np.zeros(sh))
    d = o.diagnostics()
    assert abs(d[0] - 1.7 * 2.0 * 0.5 * 3.0) < 1e-13 and abs(d[4] - 0.6 * 3.0) < 1e-13 and not d[1:4].any()
    # cylindrical annulus sector
    m = W.Mesh(12, 7, 3, -1.0, 2.0, W.uedges(0.5, 1.9, 7), W.uedges(-0.3, 0.6, 3), (PER, REF, REF))
    o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params())
    sh = (3, 7, 12)
    o.set_fields(np.full(sh, 2.0), np.full(sh, 0.1), np.zeros(sh), np.zeros(sh), np.zeros(sh))
    assert abs(o.diagnostics()[0] - 2.0 * 0.5 * (1.9 ** 2 - 0.5 ** 2) * 3.0 * 0.9) < 1e-13
    # spherical shell sector
    t0, t1 = 1.1, 1.9
    m = W.Mesh(10, 6, 5, 0.0, 2 * math.pi, W.uedges(0.7, 1.4, 6), W.uedges(t0, t1, 5), (PER, REF, REF))
    o = Oracle(m, W.SPHERICAL, W.ISOTHERMAL, W.Params())
    sh = (5, 6, 10)
    o.set_fields(np.full(sh, 0.5), np.full(sh, 0.1), np.zeros(sh), np.zeros(sh), np.zeros(sh))
    vol = (1.4 ** 3 - 0.7 ** 3) / 3.0 * (math.cos(t0) - math.cos(t1)) * 2 * math.pi
    assert abs(o.diagnostics()[0] - 0.5 * vol) < 1e-13


def test_angular_momentum_of_rigid_rotation_includes_the_frame():
    """v_phi = (w - Om_f) r in the frame rotating at Om_f: Tab. 2's X momentum is rho r^2 w whatever Om_f is."""
    nr = 40
    m = W.Mesh(8, nr, 1, -math.pi, math.pi, W.uedges(0.5, 1.5, nr), np.array([-0.5, 0.5]), (PER, REF, PER))
    sh = (1, nr, 8)
    r = m.yc()[None, :, None] * np.ones(sh)
    w = 0.7
    vals = []
    for omf in (0.0, 0.4, -1.3):
        o = Oracle(m, W.CYLINDRICAL, W.ISOTHERMAL, W.Params(omega_frame=omf))
        o.set_fields(np.full(sh, 1.2), np.full(sh, 0.1), (w - omf) * r, np.zeros(sh), None)
        vals.append(o.diagnostics()[1])
    exact = 1.2 * w * (1.5 ** 4 - 0.5 ** 4) / 4.0 * 2 * math.pi          # integral of rho w r^2 dV
    dr = 1.0 / nr
    assert abs(vals[0] - exact) < 0.6 * dr * dr * exact                   # r_c^2 V_j: second order in dr
    assert abs(vals[1] - vals[0]) < 1e-13 * exact and abs(vals[2] - vals[0]) < 1e-13 * exact


def test_mass_and_momenta_are_conserved_to_rounding_in_a_periodic_box():
    m = mesh(8, 6, 5)
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params(gamma=1.4))
    o.set_fields(*rng_fields((5, 6, 8), seed=2, vamp=0.3))
    d0 = o.diagnostics()
    o.step(6)
    d1 = o.diagnostics()
    scale = d0[0]
    assert np.max(np.abs(d1[:4] - d0[:4])) < 1e-14 * scale
    assert abs(d1[4] - d0[4]) > 1e-6                                       # internal energy is not (7b, 7c)


def test_angular_momentum_is_conserved_with_orbital_advection_and_walls():
    nphi, nr, nth = 16, 10, 6
    m = W.Mesh(nphi, nr, nth, -math.pi, math.pi, W.uedges(0.6, 1.8, nr), W.uedges(1.3, 1.8, nth), (PER, REF, REF))
    o = Oracle(m, W.SPHERICAL, W.ISOTHERMAL, W.Params(omega_frame=0.8, fargo_on=1))      # no potential: no torque
    sh = (nth, nr, nphi)
    rng = np.random.default_rng(8)
    r = m.yc()[None, :, None] * np.ones(sh)
    o.set_fields(1.0 + 0.3 * rng.uniform(-1, 1, sh), np.full(sh, 0.05), r ** -0.5 - 0.8 * r + 0.05 * rng.uniform(-1, 1, sh),
                 0.02 * rng.uniform(-1, 1, sh), 0.02 * rng.uniform(-1, 1, sh))
    d0 = o.diagnostics()
    o.step(5)
    d1 = o.diagnostics()
    assert abs(d1[0] - d0[0]) < 1e-14 * d0[0] and abs(d1[1] - d0[1]) < 1e-13 * abs(d0[1])
    assert abs(d1[2] - d0[2]) > 1e-8                                       # radial momentum has sources
