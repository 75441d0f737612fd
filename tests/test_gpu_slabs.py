"""Slab decomposition in Y (section 4.1) on ONE GPU: N contexts, each a slab of rows
with FARGO_EXTERNAL cut faces, advanced through fargo_update_phase with their halos passed buffer to buffer, against
the undivided mesh.  The paper's "indiscernibility" criterion (3 ghost layers make the cut invisible) is here
exact: every field and the clock must agree BIT for bit with the single-context run (which the other tests hold to
the oracle).  The NCCL transport of slabs.py shares everything but the message routing, which tests/test_slabs_host.py
covers with gloo on CPU."""
import dataclasses

import numpy as np
import pytest

import gpu_cases as G
from paper_1602_02359_b200 import workloads as W

pytestmark = pytest.mark.gpu

CASES = [(G.cart_adi_periodic_even, 2), (G.cart_adi_periodic_even, 3), (G.sph3d_iso_fargo, 2), (G.sph3d_iso_fargo, 3),
         (G.cyl3d_visc_fargo, 2), (G.cart_adi_mixed_bc, 3), (G.cyl2d_iso_fargo_visc, 4), (G.sheet3d_adi_fargo, 3),
         (G.nonuniform_cyl2d, 2),
         # cuts in Y and Z (py, pz): edges and corners travel with the Z planes
         (G.cart_adi_periodic_even, (2, 2)), (G.sph3d_iso_fargo, (2, 2)), (G.cart_adi_mixed_bc, (1, 3)), (G.cyl3d_visc_fargo, (2, 2)),
         (G.sph3d_adi_nofargo, (2, 3))]


def _single(w, params=None):
    from paper_1602_02359_b200 import Fargo
    g = Fargo(w.mesh, w.geometry, w.eos, params or w.params)
    g.set_fields(*w.fields())
    return g


@pytest.mark.parametrize("make,nslabs", CASES, ids=["%s-%s" % (m.__name__, n) for m, n in CASES])
def test_slabs_equal_the_undivided_mesh(make, nslabs):
    from paper_1602_02359_b200.slabs import SlabRun
    w = make()
    g = _single(w)
    g.step(w.nsteps)
    s = SlabRun(w.mesh, w.geometry, w.eos, w.params, nslabs=nslabs)
    s.set_fields(*w.fields())
    s.step(w.nsteps)
    s.synchronize()
    assert s.time() == g.time()
    for name, a, b in zip(("rho", "e", "vx", "vy", "vz"), s.get_fields(), g.get_fields()):
        assert (a is None) == (b is None)
        if a is not None:
            assert np.array_equal(a, b), "%s: %d cells differ, max %.3e" % (name, int((a != b).sum()), float(np.max(np.abs(a - b))))
    s.close()


def _sheet_periodic_y():
    """Orbital advection with a PERIODIC Y axis: v0 jumps across the seam, so the ring pair (ny-1, 0) would bind the
    shear limit of Eq. 73 if a sub-domain took it; the undivided mesh does not (rings ny-1 and 0 are no pair there)."""
    w = G.sheet3d_adi_fargo()
    P = W.PERIODIC
    m = w.mesh
    mesh = W.Mesh(m.nx, m.ny, m.nz, m.xmin, m.xmax, m.yedges, m.zedges, ((P, P), (P, P), (P, P)))
    return W.Workload("sheet3d_periodic_y", mesh, w.geometry, w.eos, w.params, w.rho, w.e, w.vx, w.vy, w.vz, w.nsteps)


@pytest.mark.parametrize("nslabs", [2, 3, (2, 2)])
def test_orbital_advection_with_a_periodic_y_axis(nslabs):
    from paper_1602_02359_b200.slabs import SlabRun
    w = _sheet_periodic_y()
    g = _single(w)
    g.step(w.nsteps)
    s = SlabRun(w.mesh, w.geometry, w.eos, w.params, nslabs=nslabs)
    s.set_fields(*w.fields())
    s.step(w.nsteps)
    s.synchronize()
    assert s.time() == g.time()
    for a, b in zip(s.get_fields(), g.get_fields()):
        assert np.array_equal(a, b)
    s.close()


ORACLE_CASES = [(G.sph3d_iso_fargo, (2, 2)), (G.cart_adi_mixed_bc, 3), (G.cyl3d_visc_fargo, 2), (_sheet_periodic_y, 3)]


@pytest.mark.parametrize("make,nslabs", ORACLE_CASES, ids=["%s-%s" % (m.__name__, n) for m, n in ORACLE_CASES])
def test_slabs_against_the_oracle(make, nslabs):
    """The decomposed run DIRECTLY against the CPU oracle of the undivided mesh (not through the single-context CUDA
    run): fields within 1e-10, the clock bit-equal."""
    from oracle.binding import Oracle
    from paper_1602_02359_b200.slabs import SlabRun
    w = make()
    o = Oracle(w.mesh, w.geometry, w.eos, w.params)
    o.set_fields(*w.fields())
    o.step(w.nsteps)
    s = SlabRun(w.mesh, w.geometry, w.eos, w.params, nslabs=nslabs)
    s.set_fields(*w.fields())
    s.step(w.nsteps)
    s.synchronize()
    assert s.time() == o.time(), (s.time(), o.time())
    for name, a, b in zip(("rho", "e", "vx", "vy", "vz"), s.get_fields(), o.get_fields()):
        if a is None:
            continue
        rel = float(np.max(np.abs(a - b))) / float(np.max(np.abs(b)))
        assert rel <= 1e-10, "%s: rel %.3e" % (name, rel)
    s.close(); o.close()


def test_t_stop_is_reached_together():
    """Each slab clips its own dt; the minimum decides and the flag is retaken after the all-reduce."""
    from paper_1602_02359_b200.slabs import SlabRun
    w = G.cart_adi_periodic_even(nx=66, ny=12, nz=10)
    g0 = _single(w)
    g0.step(3)
    prm = dataclasses.replace(w.params, t_stop=0.93 * g0.time()[0])          # lands inside the third update
    g = _single(w, prm)
    g.step(6)
    s = SlabRun(w.mesh, w.geometry, w.eos, prm, nslabs=3)
    s.set_fields(*w.fields())
    s.step(6)
    s.synchronize()
    assert s.time() == g.time() and g.time()[0] == prm.t_stop and g.time()[2] == 3
    for a, b in zip(s.get_fields(), g.get_fields()):
        assert np.array_equal(a, b)


def test_a_slab_refuses_fargo_step_and_out_of_order_phases():
    from paper_1602_02359_b200.slabs import SlabRun
    w = G.cart_adi_periodic_even(nx=66, ny=12, nz=10)
    s = SlabRun(w.mesh, w.geometry, w.eos, w.params, nslabs=2)
    s.set_fields(*w.fields())
    with pytest.raises(RuntimeError):
        s.ctx[0].step(1)
    with pytest.raises(RuntimeError):
        s.ctx[0].update_phase(1)
    s.step(1)
    s.synchronize()


def test_fp32_sub_domains_equal_the_undivided_fp32_mesh():
    from paper_1602_02359_b200 import Fargo
    from paper_1602_02359_b200.slabs import SlabRun
    w = G.sph3d_iso_fargo()
    g = Fargo(w.mesh, w.geometry, w.eos, w.params, precision=32)
    g.set_fields(*w.fields())
    g.step(w.nsteps)
    s = SlabRun(w.mesh, w.geometry, w.eos, w.params, nslabs=(3, 2), precision=32)
    s.set_fields(*w.fields())
    s.step(w.nsteps)
    s.synchronize()
    assert s.time() == g.time()
    for a, b in zip(s.get_fields(), g.get_fields()):
        assert a.dtype == np.float32 and np.array_equal(a, b)
