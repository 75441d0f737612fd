"""Parity at BASELINE.json's FULL sizes (config 5 at 512^3, config 4 at 1536x512x128), in the launch
configuration bench.py times (one context, CUDA-graph replay, whole mesh resident in HBM).

The oracle needs ~60 s and ~25 GB per full-size update, so the comparison is made on what it can compute
piecewise, from the SAME seeded inputs and from nothing the CUDA path produced:

* the time step: Eq. 59 is a max over cells of a quantity that needs only the cell and its upper faces, so
  dt(full mesh) = min over slabs of dt(slab) EXACTLY.  Each slab is an oracle run on a slice of the generated
  input plus one cover layer that supplies the upper-face velocity of the slab's last layer and is itself
  made harmless (zero sound speed, zero vx, vy), so it can never hold the maximum rate;
* the fields: one full update of a cell depends on inputs within a few cells of it (source step 3 cells,
  each sweep 2) once dt is given.  Sub-boxes of the generated input are advanced by the oracle with
  dt_fixed = the oracle's own full-mesh dt and compared with the same cells of the full-size GPU run,
  leaving out a margin of MARGIN cells per update along every cut (rings are never cut: orbital advection
  needs them whole).  A sub-box that touches a real boundary keeps that boundary's kind;
* several updates: both sides run with the same dt_fixed and the margin grows with the update count;
* properties that hold at any size: total mass is conserved to rounding (periodic box; walls at rest).

Bar: the north_star's 1e-10 (fp64) on every compared cell, dt bit-equal.
"""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL64 = 1e-10
MARGIN = 8     # cells per update (domain of dependence of one update is <= 7 cells per direction)


def _gpu(w, params=None):
    from paper_1602_02359_b200 import Fargo
    g = Fargo(w.mesh, w.geometry, w.eos, params or w.params)
    g.set_fields(*w.fields())
    return g


def _copy_params(p, **kw):
    import dataclasses
    return dataclasses.replace(p, **kw)


# ---------------------------------------------------------------- dt by slabs --------------------------
def oracle_dt_by_slabs(w, nslab_layers):
    """min over Z slabs of the oracle's CFL time step; equals the full-mesh dt exactly (see module docstring)."""
    m = w.mesh
    nz = m.nz
    per_z = m.bc[2][0] == W.PERIODIC
    best = math.inf
    for z0 in range(0, nz, nslab_layers):
        z1 = min(nz, z0 + nslab_layers)
        last = z1 == nz
        cover = not (last and not per_z)          # a real wall on top needs no cover layer
        zs = list(range(z0, z1)) + ([z1 % nz] if cover else [])
        zedges = m.zedges[z0:z1 + 1]
        if cover:   # the cover layer's own width is irrelevant: give it the width of the layer below it
            zedges = np.concatenate([zedges, [zedges[-1] + (zedges[-1] - zedges[-2])]])
        lo = m.bc[2][0] if (z0 == 0 and not per_z) else W.OUTFLOW
        hi = m.bc[2][1] if (last and not per_z) else W.OUTFLOW
        sm = W.Mesh(m.nx, m.ny, len(zs), m.xmin, m.xmax, m.yedges, zedges, (m.bc[0], m.bc[1], (lo, hi)))
        f = [None if a is None else np.ascontiguousarray(a[zs]) for a in w.fields()]
        if cover:
            f[0][-1] = 1.0
            f[1][-1] = 1e-30      # no sound speed (e or c_s): the cover layer cannot bind
            f[2][-1] = 0.0
            if f[3] is not None:
                f[3][-1] = 0.0
            # f[4][-1] stays: it is the velocity on the upper face of the slab's last real layer
        o = Oracle(sm, w.geometry, w.eos, w.params)
        o.set_fields(*f)
        o.step_until("DT")
        best = min(best, o.time()[1])
        o.close()
    return best


# ---------------------------------------------------------------- sub-boxes -----------------------------
def _axis_cut(n, lo, size, periodic):
    """Indices of a window [lo, lo+size) along an axis of n cells; (indices, touches_low, touches_high)."""
    if size >= n:
        return np.arange(n), True, True
    if periodic:
        return (lo + np.arange(size)) % n, False, False
    lo = max(0, min(lo, n - size))
    return np.arange(lo, lo + size), lo == 0, lo + size == n


def sub_workload(w, lo, size):
    """The window lo=(i,j,k), size=(sx,sy,sz) of workload w as a workload of its own (cuts become OUTFLOW).
    Returns (sub workload, index arrays, per-axis flags (whole, low is real, high is real))."""
    m = w.mesh
    n = (m.nx, m.ny, m.nz)
    idx, flags, bc = [], [], []
    for ax in range(3):
        per = m.bc[ax][0] == W.PERIODIC
        ii, tl, th = _axis_cut(n[ax], lo[ax], size[ax], per)
        whole = len(ii) == n[ax]
        idx.append(ii)
        flags.append((whole, tl, th))
        bc.append(m.bc[ax] if whole else (m.bc[ax][0] if (tl and not per) else W.OUTFLOW,
                                          m.bc[ax][1] if (th and not per) else W.OUTFLOW))
    ix, iy, iz = idx
    dx = m.dx

    def edges(full, ii, whole):
        if whole:
            return full
        if ii[-1] > ii[0]:                      # contiguous window: the true edges (curvilinear meshes need them)
            return full[ii[0]:ii[-1] + 2]
        d = full[1] - full[0]                   # wrapped window (periodic Cartesian axis): same uniform spacing
        return full[0] + d * np.arange(len(ii) + 1)
    if flags[0][0]:
        xmin, xmax = m.xmin, m.xmax
    else:
        x0 = int(ix[0]) if ix[-1] > ix[0] else 0
        xmin, xmax = m.xmin + x0 * dx, m.xmin + (x0 + len(ix)) * dx
    sm = W.Mesh(len(ix), len(iy), len(iz), xmin, xmax, edges(m.yedges, iy, flags[1][0]),
                edges(m.zedges, iz, flags[2][0]), tuple(bc))
    f = [None if a is None else np.ascontiguousarray(a[np.ix_(iz, iy, ix)]) for a in w.fields()]
    sw = W.Workload(w.name + "_sub", sm, w.geometry, w.eos, w.params, f[0], f[1], f[2], f[3], f[4], 1)
    return sw, idx, flags


def compare_boxes(w, gpu_fields, boxes, nsteps, dt_fixed, margin=MARGIN):
    """Advance each sub-box with the oracle (dt_fixed) and compare its interior with the GPU's full-size result."""
    worst = {}
    for lo, size in boxes:
        sw, idx, flags = sub_workload(w, lo, size)
        prm = _copy_params(w.params, dt_fixed=dt_fixed)
        o = Oracle(sw.mesh, sw.geometry, sw.eos, prm)
        o.set_fields(*sw.fields())
        o.step(nsteps)
        fo = o.get_fields()
        o.close()
        mg = margin * nsteps
        sl, gi = [], []
        for ax in (2, 1, 0):   # array axes are (z, y, x)
            whole, tl, th = flags[ax]
            n = len(idx[ax])
            a = 0 if (whole or tl) else mg
            b = n if (whole or th) else n - mg
            assert b - a >= 4, "sub-box too small for its margin"
            sl.append(slice(a, b))
            gi.append(idx[ax][a:b])
        for name, fg, fo_ in zip(("rho", "e", "vx", "vy", "vz"), gpu_fields, fo):
            if fg is None:
                continue
            a = fg[np.ix_(*gi)]
            b = fo_[tuple(sl)]
            assert np.isfinite(a).all(), name
            rel = float(np.max(np.abs(a - b))) / float(np.max(np.abs(b)))
            worst[name] = max(worst.get(name, 0.0), rel)
            assert rel <= TOL64, "box %r %s: rel %.3e over %d cells" % ((lo, size), name, rel, a.size)
    return worst


def _mass(w, rho):
    """Sum of rho * V over active cells with the closed-form cell volumes (Tab. 5)."""
    m = w.mesh
    ye, ze = np.asarray(m.yedges), np.asarray(m.zedges)
    if w.geometry in (W.CARTESIAN, W.SHEARING_SHEET):
        vj, vk = np.diff(ye), np.diff(ze)
    elif w.geometry == W.CYLINDRICAL:
        vj, vk = 0.5 * np.diff(ye ** 2), np.diff(ze)
    else:
        vj, vk = np.diff(ye ** 3) / 3.0, -np.diff(np.cos(ze))
    vol = m.dx * vk[:, None, None] * vj[None, :, None]
    return float(np.sum(rho * vol, dtype=np.longdouble))


# ---------------------------------------------------------------- config 5 at 512^3 ----------------------
@pytest.fixture(scope="module")
def noise512():
    return W.noise_box(512)


def test_noise512_one_update_cfl_dt(noise512):
    """One update from the seeded state with the CFL time step: dt bit-equal to the oracle's (by slabs), fields
    within 1e-10 on three sub-boxes, one of them wrapped across all three periodic seams."""
    w = noise512
    dt_o = oracle_dt_by_slabs(w, 32)
    g = _gpu(w)
    g.step(1)
    t, dt_g, ns = g.time()
    assert ns == 1 and dt_g == dt_o and t == dt_o, "dt: gpu %.17g oracle %.17g" % (dt_g, dt_o)
    fg = g.get_fields()
    g.close()
    boxes = [((500, 500, 500), (40, 40, 40)), ((200, 300, 100), (40, 40, 40)), ((0, 0, 0), (72, 24, 24))]
    worst = compare_boxes(w, fg, boxes, 1, dt_o)
    print("noise512 one update, worst rel per field:", {k: "%.2e" % v for k, v in worst.items()})


def test_noise512_three_updates_fixed_dt(noise512):
    """Three updates (graph replay, as bench.py runs them) with a fixed dt on both sides; mass conserved."""
    w = noise512
    dt = 5e-4
    g = _gpu(w, _copy_params(w.params, dt_fixed=dt))
    g.step(3)
    assert g.time()[2] == 3
    fg = g.get_fields()
    g.close()
    m0, m1 = _mass(w, w.rho), _mass(w, fg[0])
    assert abs(m1 - m0) <= 1e-12 * abs(m0), (m0, m1)
    boxes = [((480, 490, 500), (64, 64, 64)), ((100, 200, 300), (64, 64, 64))]
    worst = compare_boxes(w, fg, boxes, 3, dt)
    print("noise512 three updates, worst rel per field:", {k: "%.2e" % v for k, v in worst.items()})


# ---------------------------------------------------------------- config 4 at 1536x512x128 ---------------
@pytest.fixture(scope="module")
def disk3d():
    return W.disk3d()


def test_disk3d_one_update_cfl_dt(disk3d):
    """Config 4 at full size: dt (cell limit and shear limit, Eq. 73) bit-equal, fields within 1e-10 on whole-ring
    sub-boxes at the inner/lower walls, around the planet and at the outer/upper walls."""
    w = disk3d
    dt_o = oracle_dt_by_slabs(w, 8)
    g = _gpu(w)
    g.step(1)
    t, dt_g, ns = g.time()
    assert ns == 1 and dt_g == dt_o, "dt: gpu %.17g oracle %.17g" % (dt_g, dt_o)
    fg = g.get_fields()
    g.close()
    nx = w.mesh.nx
    boxes = [((0, 0, 0), (nx, 40, 40)), ((0, 126, 44), (nx, 40, 40)), ((0, 472, 88), (nx, 40, 40))]
    worst = compare_boxes(w, fg, boxes, 1, dt_o)
    print("disk3d one update, worst rel per field:", {k: "%.2e" % v for k, v in worst.items()})


def test_disk3d_three_updates_fixed_dt(disk3d):
    """Three updates with a fixed dt (rings shift by several cells at the inner edge); mass conserved (walls at rest)."""
    w = disk3d
    dt = 4e-3
    g = _gpu(w, _copy_params(w.params, dt_fixed=dt))
    g.step(3)
    fg = g.get_fields()
    g.close()
    m0, m1 = _mass(w, w.rho), _mass(w, fg[0])
    assert abs(m1 - m0) <= 1e-12 * abs(m0), (m0, m1)
    nx = w.mesh.nx
    boxes = [((0, 0, 0), (nx, 56, 56)), ((0, 118, 36), (nx, 56, 56))]
    worst = compare_boxes(w, fg, boxes, 3, dt)
    print("disk3d three updates, worst rel per field:", {k: "%.2e" % v for k, v in worst.items()})


# ---------------------------------------------------------------- NEXT-1 workloads at the sizes bench.py times -----
@pytest.fixture(scope="module")
def sheet3d():
    return W.sheet3d()


def test_sheet3d_one_update_cfl_dt_and_three_with_fixed_dt(sheet3d):
    """Shearing sheet 1024x512x128 (bench workload sheet3d): dt bit-equal by slabs; fields on whole-row sub-boxes at
    both walls and in the middle (rows are never cut: orbital advection); mass conserved between the walls."""
    w = sheet3d
    dt_o = oracle_dt_by_slabs(w, 8)
    g = _gpu(w)
    g.step(1)
    t, dt_g, ns = g.time()
    assert ns == 1 and dt_g == dt_o, "dt: gpu %.17g oracle %.17g" % (dt_g, dt_o)
    fg = g.get_fields()
    g.close()
    nx = w.mesh.nx
    boxes = [((0, 0, 0), (nx, 40, 40)), ((0, 236, 100), (nx, 40, 40)), ((0, 472, 50), (nx, 40, 40))]
    worst = compare_boxes(w, fg, boxes, 1, dt_o)
    print("sheet3d one update, worst rel per field:", {k: "%.2e" % v for k, v in worst.items()})
    dt = 2e-3
    g = _gpu(w, _copy_params(w.params, dt_fixed=dt))
    g.step(3)
    fg = g.get_fields()
    g.close()
    m0, m1 = _mass(w, w.rho), _mass(w, fg[0])
    assert abs(m1 - m0) <= 1e-12 * abs(m0), (m0, m1)
    worst = compare_boxes(w, fg, [((0, 0, 90), (nx, 56, 56)), ((0, 300, 10), (nx, 56, 56))], 3, dt)
    print("sheet3d three updates, worst rel per field:", {k: "%.2e" % v for k, v in worst.items()})


def test_disk3d_viscous_one_update_cfl_dt(disk3d):
    """Config 4 with nu = 1e-5 (bench workload disk3dvisc: fused source pass with the extra ghost layer, then 7d in
    one pass): dt bit-equal (the viscous limit of Eq. 59 is per cell), fields on whole-ring sub-boxes; the viscous
    stencil adds two cells to the domain of dependence, hence the wider margin."""
    import dataclasses
    w = dataclasses.replace(disk3d, params=_copy_params(disk3d.params, nu=1e-5))
    dt_o = oracle_dt_by_slabs(w, 8)
    g = _gpu(w)
    g.step(1)
    t, dt_g, ns = g.time()
    assert ns == 1 and dt_g == dt_o, "dt: gpu %.17g oracle %.17g" % (dt_g, dt_o)
    fg = g.get_fields()
    g.close()
    nx = w.mesh.nx
    boxes = [((0, 0, 0), (nx, 44, 44)), ((0, 126, 42), (nx, 44, 44)), ((0, 468, 84), (nx, 44, 44))]
    worst = compare_boxes(w, fg, boxes, 1, dt_o, margin=10)
    print("disk3dvisc one update, worst rel per field:", {k: "%.2e" % v for k, v in worst.items()})
