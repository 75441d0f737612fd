"""Pins of the oracle's 1-D primitives and tables against what the paper and the mathematics fix
(SURVEY.md 8(c.4)).  CPU only.  P:n = /root/reference/PAPER.md line n."""
import math

import numpy as np
import pytest

from oracle import binding as ob
from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W
from helpers import mesh


# ------------------------------------------------------------------ geometry (Tab. 5)
def _geom_oracle(geometry, y, z, nx=8, ny=5, nz=4, x=(0.0, 1.0)):
    bc = ((W.PERIODIC,) * 2, (W.OUTFLOW,) * 2, (W.OUTFLOW,) * 2)
    m = mesh(nx, ny, nz, x=x, y=y, z=z, bc=bc)
    return Oracle(m, geometry, W.ISOTHERMAL, W.Params()), m


@pytest.mark.parametrize("geometry", [W.CARTESIAN, W.CYLINDRICAL, W.SPHERICAL])
def test_geometry_tables_are_exact_areas_and_volumes(geometry):
    """"Left as an exercise" at P:1134: products of the Tab. 5 coefficients are the exact face
    areas and the exact cell volume in each geometry."""
    y, z = (0.5, 2.0), ((0.3, 0.9) if geometry != W.SPHERICAL else (1.0, 1.9))
    o, m = _geom_oracle(geometry, y, z, x=(0.0, 0.8))
    dx = m.dx
    tot = 0.0
    for k in range(o.ngz, o.ngz + m.nz):
        for j in range(o.ngy, o.ngy + m.ny):
            g = o.geometry(j, k)
            y0, y1 = m.yedges[j - o.ngy], m.yedges[j - o.ngy + 1]
            z0, z1 = m.zedges[k - o.ngz], m.zedges[k - o.ngz + 1]
            if geometry == W.CARTESIAN:
                sx, sy, sz = (y1 - y0) * (z1 - z0), dx * (z1 - z0), dx * (y1 - y0)
                vol = dx * (y1 - y0) * (z1 - z0)
                lx, lz = dx, z1 - z0
            elif geometry == W.CYLINDRICAL:      # X = phi, Y = r, Z = z
                sx, sy, sz = (y1 - y0) * (z1 - z0), y0 * dx * (z1 - z0), 0.5 * dx * (y1**2 - y0**2)
                vol = 0.5 * (y1**2 - y0**2) * dx * (z1 - z0)
                lx, lz = 0.5 * (y0 + y1) * dx, z1 - z0
            else:                                # X = phi, Y = r, Z = theta
                sx = 0.5 * (y1**2 - y0**2) * (z1 - z0)
                sy = y0**2 * dx * (math.cos(z0) - math.cos(z1))
                sz = 0.5 * dx * (y1**2 - y0**2) * math.sin(z0)
                vol = (y1**3 - y0**3) / 3.0 * dx * (math.cos(z0) - math.cos(z1))
                rc = 0.5 * (y0 + y1)
                lx, lz = rc * math.sin(0.5 * (z0 + z1)) * dx, rc * (z1 - z0)
            assert g["sx"] == pytest.approx(sx, rel=1e-14)
            assert g["sy"] == pytest.approx(sy, rel=1e-14)
            assert g["sz"] == pytest.approx(sz, rel=1e-14)
            assert 1.0 / g["invv"] == pytest.approx(vol, rel=1e-14)
            assert g["lx"] == pytest.approx(lx, rel=1e-14)
            assert g["ly"] == pytest.approx(y1 - y0, rel=1e-14)
            assert g["lz"] == pytest.approx(lz, rel=1e-14)
            tot += m.nx / g["invv"]
    X = m.xmax - m.xmin
    if geometry == W.CARTESIAN:
        exact = X * (y[1] - y[0]) * (z[1] - z[0])
    elif geometry == W.CYLINDRICAL:
        exact = 0.5 * (y[1]**2 - y[0]**2) * X * (z[1] - z[0])
    else:
        exact = (y[1]**3 - y[0]**3) / 3.0 * X * (math.cos(z[0]) - math.cos(z[1]))
    assert tot == pytest.approx(exact, rel=1e-13)


# ------------------------------------------------------------------ van Leer
def test_vanleer_worked_example():
    """f = (1,2,4,3), unit spacing: a_1 = 2*1*2/(1+2) = 4/3, a_2 = 0 (extremum);
    w = +0.5, dt = 0.4 -> f* between cells 1 and 2 = 2 + (4/3)(1 - 0.2)/2; w = -0.5 -> f* = 4."""
    f = np.array([1.0, 2.0, 4.0, 3.0])
    one = np.ones(4)
    a = ob.vanleer_slopes(f, one)
    assert a[0] == 0.0 and a[3] == 0.0 and a[2] == 0.0
    assert a[1] == pytest.approx(4.0 / 3.0, rel=1e-15)
    fs = ob.vanleer_star(f, a, one, 0.5 * one, 0.4)
    assert fs[2] == pytest.approx(2.0 + (4.0 / 3.0) * (1.0 - 0.2) / 2.0, rel=1e-15)
    fs = ob.vanleer_star(f, a, one, -0.5 * one, 0.4)
    assert fs[2] == 4.0          # a_2 = 0: upwind cell value
    assert fs[1] == pytest.approx(2.0 - (4.0 / 3.0) * (1.0 - 0.2) / 2.0, rel=1e-15)


def test_vanleer_slope_is_harmonic_mean_and_zero_at_extrema():
    r = np.random.default_rng(3)
    f = r.normal(size=64)
    c = np.cumsum(r.uniform(0.5, 1.5, 64))          # non-uniform centres (reading G5)
    invd = np.ones(64)
    invd[1:] = 1.0 / np.diff(c)
    a = ob.vanleer_slopes(f, invd)
    for m in range(1, 63):
        dm, dp = (f[m] - f[m - 1]) / (c[m] - c[m - 1]), (f[m + 1] - f[m]) / (c[m + 1] - c[m])
        if dm * dp <= 0:
            assert a[m] == 0.0
        else:
            assert 1.0 / a[m] == pytest.approx(0.5 * (1.0 / dm + 1.0 / dp), rel=1e-13)   # harmonic mean
            assert abs(a[m]) <= 2.0 * min(abs(dm), abs(dp)) * (1 + 1e-14)                  # monotone


def test_vanleer_star_is_time_centred_upwind_value_of_a_linear_profile():
    """For linear f the slope is exact, and Eq. 48 returns f at the point half a displacement upstream
    of the face: f(x_face - w dt / 2), whatever the sign of w."""
    n, dt = 16, 0.3
    x = np.arange(n) + 0.5
    f = 3.0 + 0.25 * x
    one = np.ones(n)
    a = ob.vanleer_slopes(f, one)
    for wv in (0.7, -0.7, 0.0):
        fs = ob.vanleer_star(f, a, one, wv * one, dt)
        for m in range(2, n - 1):
            assert fs[m] == pytest.approx(3.0 + 0.25 * (m - 0.5 * wv * dt), rel=1e-14)


# ------------------------------------------------------------------ PPA
def test_ppa_parabola_example():
    """cell averages of x^2 on unit cells [i-1/2, i+1/2] are i^2 + 1/12; for
    f_i = i^2 (interior of a long ring) the interface values are (i+-1/2)^2 - 1/12, no limiter fires,
    and for xi = 0.25 the star value on face 3+1/2 is the exact mean of x^2 - 1/12 over [3.25, 3.5]."""
    n = 32
    i = np.arange(n, dtype=float)
    f = i * i
    fl, fr = ob.ppa_interfaces(f)
    for c in range(3, 12):
        assert fr[c] == pytest.approx((c + 0.5) ** 2 - 1.0 / 12.0, rel=1e-14)
        assert fl[c] == pytest.approx((c - 0.5) ** 2 - 1.0 / 12.0, rel=1e-14)
    fs = ob.ppa_star(f, 0.25)
    exact = ((3.5 ** 3 - 3.25 ** 3) / 3.0) / 0.25 - 1.0 / 12.0
    assert exact == pytest.approx(11.3125, rel=1e-15)
    assert fs[3] == pytest.approx(exact, rel=1e-14)
    # negative displacement: the upwind cell is 4 and the swept interval is [3.5, 3.75]
    fs = ob.ppa_star(f, -0.25)
    exact = ((3.75 ** 3 - 3.5 ** 3) / 3.0) / 0.25 - 1.0 / 12.0
    assert fs[3] == pytest.approx(exact, rel=1e-14)


def test_ppa_monotonised_interfaces_bounded_and_flat_at_extrema():
    r = np.random.default_rng(5)
    f = r.normal(size=97)
    fl, fr = ob.ppa_interfaces(f)
    fm, fp = np.roll(f, 1), np.roll(f, -1)
    ext = (fp - f) * (f - fm) <= 0
    assert np.all(fl[ext] == f[ext]) and np.all(fr[ext] == f[ext])          # first test of P:484
    lo, hi = np.minimum(np.minimum(fm, fp), f), np.maximum(np.maximum(fm, fp), f)
    assert np.all(fl >= lo - 1e-13) and np.all(fl <= hi + 1e-13)
    assert np.all(fr >= lo - 1e-13) and np.all(fr <= hi + 1e-13)
    # the parabola through (fl, f, fr) is monotone in the cell: |C| <= |Delta|/6 after the tests
    D, C = fr - fl, f - 0.5 * (fl + fr)
    assert np.all(np.abs(D * C) <= D * D / 6.0 + 1e-13)


def test_ppa_star_limits_and_mirror():
    r = np.random.default_rng(7)
    f = np.cumsum(r.normal(size=64))
    f -= np.linspace(0, f[-1], 64)                      # roughly periodic
    fl, fr = ob.ppa_interfaces(f)
    assert np.array_equal(ob.ppa_star(f, 0.0), fr)      # zero displacement: interface value
    # |xi| -> 1 would sweep the whole upwind cell: mean = f (formula is exact for any x in [0,1])
    assert np.allclose(ob.ppa_star(f, 1.0), f, rtol=0, atol=1e-13)
    assert np.allclose(ob.ppa_star(f, -1.0), np.roll(f, -1), rtol=0, atol=1e-13)
    # mirror symmetry: reversing the ring and the sign of xi reverses the face values
    for xi in (0.31, -0.18):
        a = ob.ppa_star(f, xi)
        b = ob.ppa_star(f[::-1].copy(), -xi)
        # face i+1/2 of the original is face (n-2-i)+1/2 of the reversed ring
        assert np.allclose(a, np.roll(b[::-1], -1), rtol=0, atol=1e-13)


def test_ppa_star_brute_force_against_quadrature():
    """Brute force: build the limited parabola in each cell from (fl, f, fr) and integrate it over the
    swept interval numerically."""
    r = np.random.default_rng(11)
    f = np.cumsum(r.normal(size=40))
    fl, fr = ob.ppa_interfaces(f)
    n = len(f)
    for xi in (0.4, -0.27):
        fs = ob.ppa_star(f, xi)
        for i in range(n):
            u = i if xi >= 0 else (i + 1) % n
            D, f6 = fr[u] - fl[u], 6.0 * (f[u] - 0.5 * (fl[u] + fr[u]))
            # Colella & Woodward parabola a(s) = fl + s (D + f6 (1 - s)), s in [0,1] across the cell
            s = np.linspace(1.0 - xi, 1.0, 2001) if xi >= 0 else np.linspace(0.0, -xi, 2001)
            val = fl[u] + s * (D + f6 * (1.0 - s))
            mean = np.sum(0.5 * (val[1:] + val[:-1]) * np.diff(s)) / abs(xi)
            assert fs[i] == pytest.approx(mean, rel=1e-6, abs=1e-6)


# ------------------------------------------------------------------ boundary fills (reading G22)
def _bc_state(kind, normal_field):
    """1-D column along Y with 4 active cells carrying 1,2,3,4 (5 for the face above)."""
    bc = ((W.PERIODIC,) * 2, (kind, kind), (W.PERIODIC,) * 2)
    m = mesh(2, 4, 1, bc=bc)
    o = Oracle(m, W.CARTESIAN, W.ADIABATIC, W.Params())
    col = np.array([1.0, 2.0, 3.0, 4.0])[None, :, None] * np.ones((1, 4, 2))
    one = np.ones((1, 4, 2))
    o.set_fields(col, one, one, col, None)
    o.step_until("BC1")
    return o.array("rho")[0, :, 0], o.array("vy")[0, :, 0]


def test_bc_periodic_hand_example():
    rho, vy = _bc_state(W.PERIODIC, None)
    assert rho.tolist() == [2, 3, 4, 1, 2, 3, 4, 1, 2, 3]
    assert vy.tolist() == [2, 3, 4, 1, 2, 3, 4, 1, 2, 3]


def test_bc_outflow_hand_example():
    rho, vy = _bc_state(W.OUTFLOW, None)
    assert rho.tolist() == [1, 1, 1, 1, 2, 3, 4, 4, 4, 4]      # zero gradient
    assert vy.tolist() == [1, 1, 1, 1, 2, 3, 4, 4, 4, 4]


def test_bc_reflecting_hand_example():
    rho, vy = _bc_state(W.REFLECTING, None)
    assert rho.tolist() == [3, 2, 1, 1, 2, 3, 4, 4, 3, 2]      # mirror about the wall
    # normal velocity lives on faces: index 3 is the lower wall face, index 7 the upper wall face
    # -> zero on the walls, antisymmetric about them
    assert vy.tolist() == [-4, -3, -2, 0, 2, 3, 4, 0, -4, -3]
