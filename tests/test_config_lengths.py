"""Parity "after the config's step count" (BASELINE.json north_star) at every size of config 5 and at the full sizes of
configs 4 and 5, WHOLE MESH, element by element.

The reference is the OpenMP build of the oracle (oracle/liboracle_omp.so): the SAME sources as the one-thread build
with `#pragma omp parallel for` on the outer loop of each triple loop, asserted bit-identical to it on CPU
(tests/test_oracle_openmp.py).  Nothing here comes from the CUDA path: both sides start from the
seeded recipe of workloads.py and run the config's own step count with their own CFL time step, which must agree BIT
for bit at the end (it is a max/min reduction).

Bars: 1e-10 (fp64) and 1e-4 (fp32 build against the fp64 oracle) on max|gpu - oracle| / max|oracle| per field.

Cost (16 host cores): 128^3 x 50 ~ 10 s, 256^3 x 50 ~ 80 s, 512^3 x 50 and config 4 x 100 ~ 10-20 min and ~45 GB of host
memory each.  The two full-length runs are therefore run when FARGO_FULL_LENGTH=1 (their logs are committed under
profiles/); without it they run the first FULL_DEFAULT_STEPS updates of the same whole-mesh comparison, which keeps the
default GPU suite within minutes.
"""
import gc
import os

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL64 = 1e-10
TOL32 = 1e-4
FULL = os.environ.get("FARGO_FULL_LENGTH", "0") == "1"
FULL_DEFAULT_STEPS = 4
NAMES = ("rho", "e", "vx", "vy", "vz")


def _oracle_run(w, nsteps):
    o = Oracle(w.mesh, w.geometry, w.eos, w.params, omp=True)
    o.set_fields(*w.fields())
    o.step(nsteps)
    out = (o.get_fields(), o.time())
    o.close()
    del o
    gc.collect()
    return out


def _gpu_run(w, nsteps, precision):
    from paper_1602_02359_b200 import Fargo
    g = Fargo(w.mesh, w.geometry, w.eos, w.params, precision=precision)
    g.set_fields(*w.fields())
    g.step(nsteps)
    out = (g.get_fields(), g.time())
    g.close()
    return out


def _compare(tag, fg, fo, tol):
    worst = {}
    for name, a, b in zip(NAMES, fg, fo):
        if a is None or b is None:
            continue
        assert np.isfinite(a).all(), name
        s = float(np.max(np.abs(b)))
        # chunked: a 512^3 difference array is 1 GB
        d = 0.0
        fa, fb = a.reshape(-1), b.reshape(-1)
        for c in range(0, fa.size, 1 << 24):
            d = max(d, float(np.max(np.abs(fa[c:c + (1 << 24)].astype(np.float64) - fb[c:c + (1 << 24)]))))
        worst[name] = d / s if s > 0 else d
    print(tag, "worst rel per field:", {k: "%.2e" % v for k, v in worst.items()})
    for name, rel in worst.items():
        assert rel <= tol, "%s %s: rel %.3e > %.0e" % (tag, name, rel, tol)


def _both_precisions(w, nsteps, tag):
    fo, to = _oracle_run(w, nsteps)
    fg, tg = _gpu_run(w, nsteps, 64)
    assert tg[2] == nsteps == to[2]
    assert tg[0] == to[0] and tg[1] == to[1], "clock after %d updates: gpu %r oracle %r" % (nsteps, tg, to)
    _compare("%s fp64 x%d" % (tag, nsteps), fg, fo, TOL64)
    del fg
    fg, tg = _gpu_run(w, nsteps, 32)
    assert tg[2] == nsteps
    assert abs(tg[0] - to[0]) <= 1e-4 * abs(to[0]), (tg, to)
    _compare("%s fp32 x%d" % (tag, nsteps), fg, fo, TOL32)


@pytest.mark.parametrize("n", [128, 256])
def test_config5_whole_mesh_50_steps_fp64_and_fp32(n):
    """Config 5 at 128^3 and 256^3 (BASELINE.json configs[4]): 50 updates, whole mesh, both builds."""
    _both_precisions(W.noise_box(n), 50, "noise%d" % n)


def test_config5_512_whole_mesh_fp64_and_fp32():
    """Config 5 at 512^3: the config's 50 updates when FARGO_FULL_LENGTH=1, else the first FULL_DEFAULT_STEPS."""
    _both_precisions(W.noise_box(512), 50 if FULL else FULL_DEFAULT_STEPS, "noise512")


def test_config4_whole_mesh_fp64():
    """Config 4 at 1536x512x128: the config's 100 updates when FARGO_FULL_LENGTH=1, else the first FULL_DEFAULT_STEPS."""
    w = W.disk3d()
    n = 100 if FULL else FULL_DEFAULT_STEPS
    fo, to = _oracle_run(w, n)
    fg, tg = _gpu_run(w, n, 64)
    assert tg == to, "clock after %d updates: gpu %r oracle %r" % (n, tg, to)
    _compare("disk3d fp64 x%d" % n, fg, fo, TOL64)
