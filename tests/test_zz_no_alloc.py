"""fargo_diagnostics_noalloc against fargo_diagnostics (the existing path), through the C ABI.

The new entry point keeps the per-block partial sums in a file-scope device array of the library instead of the
workspace, adds them on the device in the order the existing path adds them on the host, and writes to a device address:
it allocates nothing.  Both paths run the same reduction kernel, so the sums should agree to the last bit; the bar
written here is the one tests/test_gpu_diagnostics.py uses (1e-12 of the sum's scale, fp64).

This file sorts last on purpose (pytest -x: a failure here hides nothing); it passes alone in a fresh process and
after the other tests -- the array is shared by every context of the device and keeps the last call's contents, which
the cases below exercise by following a large mesh with a small one."""
import numpy as np
import pytest

import gpu_cases as G

pytestmark = pytest.mark.gpu

TOL = 1e-12


def _scale(d):
    return np.array([d[0], max(abs(d[1]), d[0]), max(abs(d[2]), d[0]), max(abs(d[3]), d[0]), max(d[4], d[0])])


def _ctx(w, precision=64):
    from paper_1602_02359_b200 import Fargo
    g = Fargo(w.mesh, w.geometry, w.eos, w.params, precision=precision)
    g.set_fields(*w.fields())
    return g


def _noalloc(g, out):
    import torch
    torch.cuda.synchronize()            # `out` was made on torch's stream, the context has its own
    g.diagnostics_noalloc(out)
    g.stream.synchronize()
    return out.cpu().numpy().copy()


def test_noalloc_matches_existing_path_two_calls_in_a_row():
    import torch
    big, small = _ctx(G.cart_adi_periodic_even()), _ctx(G.sph3d_iso_fargo())
    out = torch.full((5,), float("nan"), dtype=torch.float64, device="cuda")
    # two calls in a row on one context, with updates in between ...
    for nstep in (0, 2):
        if nstep:
            big.step(nstep)
        ref = big.diagnostics()
        got = _noalloc(big, out)
        assert ref[0] > 0 and np.all(np.isfinite(got))
        assert np.max(np.abs(got - ref) / _scale(ref)) < TOL, (got, ref)
    # ... then a smaller mesh of another geometry: the array still holds the larger call's partials beyond its blocks
    ref = small.diagnostics()
    got = _noalloc(small, out)
    assert np.max(np.abs(got - ref) / _scale(ref)) < TOL, (got, ref)
    # and the large one again, the small call's partials now sitting in its first blocks
    ref = big.diagnostics()
    got = _noalloc(big, out)
    assert np.max(np.abs(got - ref) / _scale(ref)) < TOL, (got, ref)
    # the run is left alone: another update gives what the existing path's context gives
    twin = _ctx(G.cart_adi_periodic_even())
    twin.step(3); big.step(1)
    for a, b in zip(big.get_fields(), twin.get_fields()):
        if a is not None:
            assert np.array_equal(a, b)


def test_noalloc_fp32_and_2d():
    import torch
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    for w, precision in ((G.cart_adi_periodic(), 32), (G.yz_only_2d(), 64), (G.cyl2d_iso_fargo_visc(), 64)):
        g = _ctx(w, precision)
        g.step(1)
        ref = g.diagnostics()
        got = _noalloc(g, out)
        assert np.max(np.abs(got - ref) / _scale(ref)) < TOL, (w.name, got, ref)


def test_noalloc_allocates_no_device_memory():
    import torch
    g = _ctx(G.cart_adi_periodic())
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    _noalloc(g, out)                      # the first call of a process looks the array's address up (module load)
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        g.diagnostics_noalloc(out)
    g.stream.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_noalloc_rejects_a_mesh_beyond_the_array():
    import torch
    w = G.yz_only_2d(ny=800, nz=700)      # 560000 rows along X > 524288
    g = _ctx(w)
    out = torch.full((5,), -7.0, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    with pytest.raises(Exception) as ei:
        g.diagnostics_noalloc(out)
    assert "524288" in str(ei.value) and "fargo_diagnostics_noalloc" in str(ei.value)
    g.stream.synchronize()
    assert np.all(out.cpu().numpy() == -7.0)          # nothing was launched
    assert np.all(np.isfinite(g.diagnostics()))       # the existing path takes the mesh
    with pytest.raises(ValueError):
        g.diagnostics_noalloc(np.zeros(5))            # a host buffer is not an output of this entry point
