"""Shared test helpers (no method arithmetic beyond what a test needs to state its expectation)."""
import numpy as np

from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W


def mesh(nx, ny, nz, x=(0.0, 1.0), y=(0.0, 1.0), z=(0.0, 1.0), bc=None):
    bc = bc or ((W.PERIODIC,) * 2,) * 3
    return W.Mesh(nx, ny, nz, x[0], x[1], W.uedges(y[0], y[1], ny), W.uedges(z[0], z[1], nz), bc)


def oracle_for(w, nghost=3):
    o = Oracle(w.mesh, w.geometry, w.eos, w.params, nghost=nghost)
    o.set_fields(*w.fields())
    return o


def rng_fields(shape, seed=1, vamp=0.1):
    r = np.random.default_rng(seed)
    rho = 1.0 + 0.2 * r.uniform(-1, 1, shape)
    e = 1.5 + 0.3 * r.uniform(-1, 1, shape)
    vx, vy, vz = (vamp * r.uniform(-1, 1, shape) for _ in range(3))
    return rho, e, vx, vy, vz


def relerr(a, b):
    d = float(np.max(np.abs(a - b)))
    s = float(np.max(np.abs(b)))
    return d / s if s > 0 else d
