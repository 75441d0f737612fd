"""The OpenMP build of the oracle (oracle/liboracle_omp.so: the SAME sources, `#pragma omp parallel for` on the outer
loop of each triple loop) must be bit-identical to the one-thread build that every parity test refers to
(SURVEY.md 8(d.4)): loop bodies are cell- or line-independent and the only reductions are exact max/min.  It exists
to produce full-length references at 512^3 and config 4, where one thread would take hours.  CPU only."""
import os

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W
import gpu_cases as GC


def _run(w, n, omp, threads=None):
    if threads:
        os.environ["OMP_NUM_THREADS"] = str(threads)
    o = Oracle(w.mesh, w.geometry, w.eos, w.params, omp=omp)
    o.set_fields(*w.fields())
    if w.planets:
        o.set_planets(**w.planets)
    o.step(n)
    out = o.get_fields(), o.time()
    o.close()
    return out


def _same(a, b):
    (fa, ta), (fb, tb) = a, b
    assert ta == tb
    for x, y in zip(fa, fb):
        assert np.array_equal(x, y)


def test_openmp_build_is_bit_identical_on_128_cubed():
    """Config 5 at 128^3, 3 updates (every loop of an adiabatic periodic update), all host cores."""
    w = W.noise_box(128)
    _same(_run(w, 3, False), _run(w, 3, True))


@pytest.mark.parametrize("case", ["sph3d_iso_fargo", "cyl2d_iso_fargo_visc", "cart_adi_mixed_bc", "sod_small",
                                  "cyl3d_adi_fargo", "cart3d_visc_mixed_bc", "sph3d_visc_fargo", "sheet3d_adi_fargo",
                                  "x_only_1d", "yz_only_2d"])
def test_openmp_build_is_bit_identical_on_the_small_cases(case):
    """Orbital advection, walls, ghosted X, t_stop, 2-D and 3-D viscosity, the shearing sheet: the loops 128^3 misses."""
    w = getattr(GC, case)()
    _same(_run(w, w.nsteps, False), _run(w, w.nsteps, True))


def test_openmp_thread_count_does_not_matter():
    w = GC.sph3d_iso_fargo()
    ref = _run(w, 3, True, threads=1)
    for t in (2, 3, 7):
        _same(ref, _run(w, 3, True, threads=t))
    os.environ.pop("OMP_NUM_THREADS", None)
