"""Host logic of the slab decomposition (paper_1602_02359_b200/slabs.py): row ranges,
neighbour tables, and the message routing over torch.distributed with the gloo backend, world size 2 and 3, on CPU
(the same route_halos / all_reduce(MIN) calls the NCCL transport makes).  No CUDA, no method arithmetic."""
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_1602_02359_b200 import workloads as W
from paper_1602_02359_b200.slabs import exchange_plan, neighbours, slab_mesh, slab_ranges

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_ranges_cover_the_rows_once():
    for ny, n in ((512, 8), (13, 4), (9, 3), (7, 2)):
        r = slab_ranges(ny, n)
        assert r[0][0] == 0 and r[-1][1] == ny and all(a[1] == b[0] for a, b in zip(r, r[1:]))
        assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1 and min(b - a for a, b in r) >= 3
    with pytest.raises(ValueError):
        slab_ranges(8, 3)


def test_neighbours_and_faces():
    assert neighbours(0, 1, True) == (None, None)
    assert neighbours(0, 3, False) == (None, 1) and neighbours(2, 3, False) == (1, None)
    assert neighbours(0, 3, True) == (2, 1) and neighbours(2, 3, True) == (1, 0)
    m = W.Mesh(8, 12, 4, 0.0, 1.0, W.uedges(0.5, 2.0, 12), W.uedges(0.0, 1.0, 4),
               ((W.PERIODIC,) * 2, (W.REFLECTING, W.OUTFLOW), (W.PERIODIC,) * 2))
    subs = [slab_mesh(m, r, 3) for r in range(3)]
    assert [s.bc[1] for s, _ in subs] == [(W.REFLECTING, 3), (3, 3), (3, W.OUTFLOW)]
    assert np.array_equal(np.concatenate([s.yedges[:-1] for s, _ in subs] + [m.yedges[-1:]]), m.yedges)
    # the edges beyond a cut are the neighbour's; at a real wall there are none
    assert subs[0][0].yedges_ext[0] is None and np.array_equal(subs[0][0].yedges_ext[1], m.yedges[5:8])
    assert np.array_equal(subs[1][0].yedges_ext[0], m.yedges[1:4]) and subs[2][0].yedges_ext[1] is None
    # a 2 x 2 grid: Y fastest; Z periodic, so every Z face is cut and the seam's edges continue the mesh
    m2 = W.Mesh(8, 12, 8, 0.0, 1.0, W.uedges(0.5, 2.0, 12), W.uedges(0.0, 1.0, 8),
                ((W.PERIODIC,) * 2, (W.REFLECTING, W.OUTFLOW), (W.PERIODIC,) * 2))
    g = [slab_mesh(m2, r, (2, 2)) for r in range(4)]
    assert [x[1] for x in g] == [((0, 6), (0, 4)), ((6, 12), (0, 4)), ((0, 6), (4, 8)), ((6, 12), (4, 8))]
    assert all(x[0].bc[2] == (3, 3) for x in g)
    assert np.allclose(g[0][0].zedges_ext[0], [-0.375, -0.25, -0.125]) and np.array_equal(g[0][0].zedges_ext[1], m2.zedges[5:8])
    assert np.array_equal(g[2][0].zedges_ext[0], m2.zedges[1:4]) and np.allclose(g[2][0].zedges_ext[1], [1.125, 1.25, 1.375])


def test_every_send_has_its_receive():
    for n, per in ((2, True), (3, True), (4, False), (2, False)):
        sends = {(r, peer, side) for r in range(n) for peer, side, _ in exchange_plan(r, n, per)}
        recvs = {(peer, r, 1 - side) for r in range(n) for peer, _, side in exchange_plan(r, n, per)}
        assert sends == recvs     # (sender, receiver, sender's side): what is unpacked on side s was packed on side 1 - s


_WORKER = """
import os, sys
sys.path.insert(0, {root!r})
import torch, torch.distributed as dist
from paper_1602_02359_b200.slabs import exchange_plan, route_halos
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
per = {per}
plan = exchange_plan(rank, world, per)
send = [torch.full((5,), 10.0 * rank + side) for side in (0, 1)]      # what I packed next to my lower / upper face
recv = [torch.full((5,), -1.0) for _ in (0, 1)]
route_halos(dist, None, plan, send, recv)
got = [float(recv[0][0]), float(recv[1][0])]
dt = torch.tensor([0.5 + 0.1 * ((rank + 1) % world)], dtype=torch.float64)
dist.all_reduce(dt, op=dist.ReduceOp.MIN)
sys.stdout.write("RESULT %d %g %g %g\\n" % (rank, got[0], got[1], float(dt[0]))); sys.stdout.flush()
dist.destroy_process_group()
"""


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world,per", [(2, True), (2, False), (3, True)])
def test_halo_routing_and_dt_min_over_gloo(tmp_path, world, per):
    import re
    script = tmp_path / "worker.py"
    script.write_text(_WORKER.format(root=ROOT, per=per))
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
                        "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), str(script)],
                       capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    res = {int(a): (float(b), float(c), float(d)) for a, b, c, d in
           re.findall(r"RESULT (\d+) (-?[0-9.]+) (-?[0-9.]+) ([0-9.]+)", r.stdout)}
    assert len(res) == world
    for rank, (lo_ghost, hi_ghost, dt) in res.items():
        lo = rank - 1 if rank > 0 else (world - 1 if per else None)
        hi = rank + 1 if rank + 1 < world else (0 if per else None)
        assert lo_ghost == (-1.0 if lo is None else 10.0 * lo + 1)      # the UPPER rows of the slab below
        assert hi_ghost == (-1.0 if hi is None else 10.0 * hi + 0)      # the LOWER rows of the slab above
        assert dt == 0.5
