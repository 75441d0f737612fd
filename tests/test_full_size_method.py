"""CPU check of the piecewise method test_full_size.py uses at sizes the whole-mesh oracle cannot reach:
at a small size, (i) the min over Z slabs of the oracle's time step equals the whole-mesh oracle's bit for
bit, and (ii) a sub-box advanced with that dt reproduces the whole-mesh oracle inside the margin."""
import numpy as np

import test_full_size as T
from oracle.binding import Oracle
from paper_1602_02359_b200 import workloads as W


def _whole(w, n, dt_fixed=0.0):
    import dataclasses
    o = Oracle(w.mesh, w.geometry, w.eos, dataclasses.replace(w.params, dt_fixed=dt_fixed))
    o.set_fields(*w.fields())
    o.step(n)
    out = o.time()[1], [f if src is not None else None for f, src in zip(o.get_fields(), w.fields())]
    o.close()
    return out


def test_slab_dt_and_sub_boxes_periodic_box():
    w = W.noise_box(shape3=(48, 40, 36))
    dt, f = _whole(w, 1)
    assert T.oracle_dt_by_slabs(w, 8) == dt
    worst = T.compare_boxes(w, f, [((40, 30, 30), (30, 30, 30)), ((5, 5, 5), (30, 30, 30))], 1, dt)
    assert max(worst.values()) <= 1e-13


def test_slab_dt_and_sub_boxes_disk():
    w = W.disk3d(96, 48, 24)
    dt, f = _whole(w, 1)
    assert T.oracle_dt_by_slabs(w, 5) == dt
    worst = T.compare_boxes(w, f, [((0, 0, 0), (96, 30, 24)), ((0, 18, 0), (96, 30, 24))], 1, dt)
    assert max(worst.values()) <= 1e-13


def test_sub_boxes_two_updates_fixed_dt():
    w = W.noise_box(shape3=(56, 56, 56))
    dt = 3e-3
    _, f = _whole(w, 2, dt_fixed=dt)
    worst = T.compare_boxes(w, f, [((30, 30, 30), (48, 48, 48))], 2, dt)
    assert max(worst.values()) <= 1e-13
