"""GPU parity of fargo_diagnostics (the sum reductions of P:787: mass, Tab. 2 momenta, internal energy) against the
oracle on every small parity case, before and after a few updates.  The kernel adds lanes, warps and blocks in a
fixed tree, the oracle adds cell after cell: they differ by rounding only; the bar is 1e-12 of the sum's scale
(mass x the largest momentum per unit mass), fp64."""
import numpy as np
import pytest

import gpu_cases as G
from oracle.binding import Oracle

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("make", G.ALL, ids=[f.__name__ for f in G.ALL])
def test_diagnostics_match_the_oracle(make):
    from paper_1602_02359_b200 import Fargo
    w = make()
    g = Fargo(w.mesh, w.geometry, w.eos, w.params)
    o = Oracle(w.mesh, w.geometry, w.eos, w.params)
    for c in (g, o):
        c.set_fields(*w.fields())
    for nstep in (0, 2):
        if nstep:
            g.step(nstep); o.step(nstep)
        dg, do = g.diagnostics(), o.diagnostics()
        assert do[0] > 0
        scale = np.array([do[0], max(abs(do[1]), do[0]), max(abs(do[2]), do[0]), max(abs(do[3]), do[0]), max(do[4], do[0])])
        assert np.max(np.abs(dg - do) / scale) < 1e-12, (dg, do)
    # reproducible from call to call, and it leaves the run alone
    assert np.array_equal(g.diagnostics(), dg)
    g.step(1); o.step(1)
    for a, b in zip(g.get_fields(), o.get_fields()):
        if a is not None and np.max(np.abs(b)) > 0:
            assert np.max(np.abs(a - b)) <= 1e-10 * np.max(np.abs(b))
