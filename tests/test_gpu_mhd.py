"""GPU parity for the MHD substeps (sections 3.6.1-3.6.2; csrc/k_mhd.cu) against the CPU oracle
(oracle/mhd.cpp) on the same seeded inputs, through the C ABI (fargo_set_bfield / fargo_step / fargo_get_bfield):
fields and B within 1e-10 (fp64; bit-identical in practice), the clock bit-equal, the EMFs of the last update compared
edge by edge, div B at rounding level.  The oracle itself is pinned in tests/test_oracle_mhd.py (among others to the
field-loop energy the paper prints)."""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W

pytestmark = pytest.mark.gpu

P, O, R = W.PERIODIC, W.OUTFLOW, W.REFLECTING
TOL64, TOL32 = 1e-10, 1e-4


def _box(nx, ny, nz, bc):
    return W.Mesh(nx, ny, nz, 0.0, 1.0, W.uedges(0.0, 0.8, ny), W.uedges(-0.3, 0.4, nz), bc)


def _curl_a(shape, dx, dy, dz, seed, amp):
    r = np.random.default_rng(seed)
    ax, ay, az = (amp * r.standard_normal(shape) for _ in range(3))
    up = lambda a, axis: np.roll(a, -1, axis=axis)
    return ((up(az, 1) - az) / dy - (up(ay, 0) - ay) / dz, (up(ax, 0) - ax) / dz - (up(az, 2) - az) / dx,
            (up(ay, 2) - ay) / dx - (up(ax, 1) - ax) / dy)


def _case(name):
    r = np.random.default_rng(11)
    if name == "brio_wu":          # section 5.2.1 on a thin 3-D mesh, 200 cells along z
        n = 200
        m = W.Mesh(4, 4, n, 0.0, 16.0, W.uedges(0.0, 16.0, 4), W.uedges(0.0, 800.0, n), ((P, P), (P, P), (O, O)))
        shape = (n, 4, 4)
        left = (np.arange(n) < n // 2)[:, None, None] * np.ones(shape, dtype=bool)
        rho = np.where(left, 1.0, 0.1)
        e = np.where(left, 1.0, 0.1) / (2.0 - 1.0)
        z = np.zeros(shape)
        return dict(mesh=m, eos=W.ADIABATIC, prm=W.Params(gamma=2.0), f=(rho, e, z, z, z), b=(z, np.where(left, 1.0, -1.0), z + 0.75),
                    nsteps=60, eta=0.0, passive=False)
    if name in ("fargo", "sheet"):   # section 3.7: orbital advection of B; the sheet adds Eq. 29 and Tab. 2's X momentum
        nx, ny, nz = 66, 14, 9
        sheet = name == "sheet"
        bc = ((P, P), (R, R), (P, P)) if sheet else ((P, P), (P, P), (P, P))
        m = W.Mesh(nx, ny, nz, 0.0, 2.0, W.uedges(-0.5, 0.5, ny), W.uedges(-0.2, 0.2, nz), bc)
        shape = (nz, ny, nx)
        y = m.yc()[None, :, None] * np.ones(shape)
        bx, by, bz = _curl_a(shape, 2.0 / nx, 1.0 / ny, 0.4 / nz, 5, 0.01)
        bx += 0.05; by += 0.3; bz -= 0.1
        rho = 1.0 + 0.2 * r.uniform(-1, 1, shape)
        e = 0.9 * (1.0 + 0.2 * r.uniform(-1, 1, shape))
        shear = -24.0 * y if sheet else 15.0 * np.sin(2 * math.pi * y)          # arcs of up to two zones per update, both signs
        v = (shear + 0.2 * r.uniform(-1, 1, shape), 0.2 * r.uniform(-1, 1, shape), 0.2 * r.uniform(-1, 1, shape))
        prm = W.Params(gamma=1.4, fargo_on=1, omega_frame=1.0 if sheet else 0.0, oort_a=-0.75 if sheet else 0.0)
        return dict(mesh=m, eos=W.ADIABATIC, prm=prm, f=(rho, e) + v, b=(bx, by, bz), nsteps=6, eta=0.0, passive=False,
                    geometry=W.SHEARING_SHEET if sheet else W.CARTESIAN)
    if name in ("cyl", "cyl_fargo", "sph"):   # curvilinear meshes (reading G38): a magnetised Keplerian disk with noise
        sphc = name == "sph"
        nx, ny, nz = (192 if name == "cyl_fargo" else 48), 18, 10   # cyl_fargo: arcs of more than one zone at the inner edge
        zed = W.uedges(0.5 * math.pi - 0.25, 0.5 * math.pi + 0.25, nz) if sphc else W.uedges(-0.3, 0.3, nz)
        m = W.Mesh(nx, ny, nz, 0.0, 2.0 * math.pi, W.uedges(0.6, 1.8, ny), zed, ((P, P), (R, O), (O, R) if sphc else (P, P)))
        shape = (nz, ny, nx)
        rr = m.yc()[None, :, None] * np.ones(shape)
        om = 0.0 if name == "cyl_fargo" else 0.5                        # inertial frame: the planet also moves in the frame
        prm = W.Params(gamma=1.4, fargo_on=1 if name == "cyl_fargo" else 0, omega_frame=om, gm_star=1.0, planet_mass=1e-3, planet_r=1.1,
                       planet_phi0=0.3, planet_omega=0.5, planet_eps=0.05)
        rho = rr ** -1.0 * (1.0 + 0.1 * r.uniform(-1, 1, shape))
        e = rho * (0.1 ** 2 / rr) / 0.4 * (1.0 + 0.1 * r.uniform(-1, 1, shape))
        v = (rr ** -0.5 - rr * om + 0.03 * r.uniform(-1, 1, shape), 0.03 * r.uniform(-1, 1, shape), 0.03 * r.uniform(-1, 1, shape))
        b = tuple(0.05 * r.uniform(-1, 1, shape) + s0 for s0 in (0.02, 0.01, 0.05))
        return dict(mesh=m, eos=W.ADIABATIC, prm=prm, f=(rho, e) + v, b=b, nsteps=6, eta=0.0, passive=False,
                    geometry=W.SPHERICAL if sphc else W.CYLINDRICAL)
    bcs = {"periodic": ((P, P), (P, P), (P, P)), "mixed": ((O, R), (R, O), (O, O)), "resistive": ((P, P), (O, O), (P, P)),
           "passive": ((P, P), (P, P), (P, P)), "iso": ((P, P), (P, P), (R, R))}
    nx, ny, nz = (34, 13, 11) if name != "mixed" else (21, 12, 14)
    m = _box(nx, ny, nz, bcs[name])
    shape = (nz, ny, nx)
    bx, by, bz = _curl_a(shape, 1.0 / nx, 0.8 / ny, 0.7 / nz, 3, 0.02)
    bx += 0.4; by -= 0.3; bz += 0.2
    rho = 1.0 + 0.3 * r.uniform(-1, 1, shape)
    eos = W.ISOTHERMAL if name == "iso" else W.ADIABATIC
    e = 0.9 * (1.0 + 0.2 * r.uniform(-1, 1, shape)) if eos == W.ISOTHERMAL else 1.5 * (1.0 + 0.3 * r.uniform(-1, 1, shape))
    v = tuple(0.6 * r.uniform(-1, 1, shape) for _ in range(3))
    return dict(mesh=m, eos=eos, prm=W.Params(gamma=1.4), f=(rho, e) + v, b=(bx, by, bz), nsteps=6,
                eta=3e-3 if name == "resistive" else 0.0, passive=name == "passive")


def _pair(c, precision=64, use_graph=True):
    from paper_1602_02359_b200 import Fargo
    geo = c.get("geometry", W.CARTESIAN)
    g = Fargo(c["mesh"], geo, c["eos"], c["prm"], precision=precision, use_graph=use_graph, mhd=True)
    g.set_fields(*c["f"])
    g.set_bfield(*c["b"], eta=c["eta"], passive=c["passive"])
    o = Oracle(c["mesh"], geo, c["eos"], c["prm"])
    o.set_fields(*c["f"])
    o.set_bfield(*c["b"], eta=c["eta"], passive=c["passive"])
    return g, o


def _rel(a, b):
    s = float(np.max(np.abs(b)))
    d = float(np.max(np.abs(np.asarray(a, dtype=np.float64) - b)))
    return d / s if s > 0 else d


CASES = ["periodic", "mixed", "resistive", "passive", "iso", "brio_wu", "fargo", "sheet", "cyl", "cyl_fargo", "sph"]


@pytest.mark.parametrize("name", CASES)
@pytest.mark.parametrize("use_graph", [True, False], ids=["graph", "stream"])
def test_mhd_updates_match_the_oracle(name, use_graph):
    c = _case(name)
    g, o = _pair(c, use_graph=use_graph)
    g.step(c["nsteps"]); o.step(c["nsteps"])
    assert g.time() == o.time(), (g.time(), o.time())
    for nm, a, b in zip(("rho", "e", "vx", "vy", "vz"), g.get_fields(), o.get_fields()):
        assert np.isfinite(a).all() and _rel(a, b) <= TOL64, (name, nm, _rel(a, b))
    bg, bo = g.get_bfield(), o.get_bfield()
    for nm, a, b in zip(("bx", "by", "bz"), bg, bo):
        assert np.isfinite(a).all() and _rel(a, b) <= TOL64, (name, nm, _rel(a, b))
        assert not np.array_equal(b, np.broadcast_to(c["b"]["xyz".index(nm[1])], b.shape)) or name == "brio_wu" and nm != "by"
    # the electromotive forces of the last update, edge by edge, ghost zones included
    for nm in ("emfx", "emfy", "emfz"):
        a, b = g.array(nm), o.array(nm)
        assert _rel(a, b) <= TOL64, (name, nm, _rel(a, b))
    g.close(); o.close()


def test_div_b_stays_at_rounding_level_on_the_gpu():
    c = _case("periodic")
    g, _ = _pair(c)
    g.step(10)
    bx, by, bz = g.get_bfield()
    m = c["mesh"]
    div = (np.roll(bx, -1, 2) - bx) * m.nx + (np.roll(by, -1, 1) - by) * (m.ny / 0.8) + (np.roll(bz, -1, 0) - bz) * (m.nz / 0.7)
    scale = float(np.sqrt(np.mean(bx ** 2 + by ** 2 + bz ** 2))) * max(m.nx, m.ny / 0.8, m.nz / 0.7)
    assert float(np.max(np.abs(div))) <= 1e-13 * scale
    g.close()


def test_mhd_fp32_build_is_close_to_the_fp64_oracle():
    c = _case("periodic")
    g, o = _pair(c, precision=32)
    g.step(c["nsteps"]); o.step(c["nsteps"])
    assert abs(g.time()[0] - o.time()[0]) <= 1e-5 * o.time()[0]
    for a, b in zip(g.get_fields() + g.get_bfield(), o.get_fields() + o.get_bfield()):
        assert a.dtype == np.float32 and _rel(a, b) <= TOL32, _rel(a, b)
    g.close(); o.close()


def test_mhd_argument_errors_and_second_set_bfield():
    from paper_1602_02359_b200 import Fargo
    c = _case("periodic")
    g = Fargo(c["mesh"], W.CARTESIAN, c["eos"], c["prm"])          # created without mhd
    g.set_fields(*c["f"])
    with pytest.raises(RuntimeError):
        g.set_bfield(*c["b"])
    g.close()
    sp = _case("sph")
    with pytest.raises(RuntimeError):                                 # the resistive term: Cartesian metric only
        gs = Fargo(sp["mesh"], W.SPHERICAL, sp["eos"], sp["prm"], mhd=True)
        gs.set_fields(*sp["f"])
        gs.set_bfield(*sp["b"], eta=1e-3)
    with pytest.raises(ValueError):                                   # a 2-D mesh: thin 3-D meshes are the way
        Fargo(W.Mesh(16, 16, 1, 0.0, 1.0, W.uedges(0, 1, 16), np.array([0.0, 1.0])), W.CARTESIAN, c["eos"], c["prm"], mhd=True)
    g, o = _pair(c)
    g.step(2); o.step(2)
    for x in (g, o):                                                   # restart both from the same state with a new field
        x.set_fields(*c["f"])
        x.set_bfield(c["b"][0] * 0.5, c["b"][1], c["b"][2] * 2.0)
    g.step(3); o.step(3)
    assert g.time() == o.time()
    for a, b in zip(g.get_bfield(), o.get_bfield()):
        assert _rel(a, b) <= TOL64
    g.close(); o.close()
