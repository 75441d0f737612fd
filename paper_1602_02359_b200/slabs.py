"""Domain decomposition in Y and Z over several contexts (section 4.1).

The paper splits the mesh in Y (and Z), never in X, exchanges 3 ghost layers at cells 2 and 9 of Fig. 2 and takes the
minimum of the time step over the sub-domains.  Here a sub-domain is an ordinary context (C ABI,
include/fargo.h) whose cut Y / Z faces have the kind FARGO_EXTERNAL; this module only does the plumbing the ABI leaves to the caller:
who is whose neighbour, the halo messages, the all-reduce of dt.  No arithmetic of the method lives here.

Two transports:
  * `SlabRun(..., nslabs=N)`            every slab in this process on the current device, all on ONE stream; a halo
                                        packed by one slab is unpacked by its neighbour directly.  This is how the
                                        decomposition is verified bit for bit on a single GPU (tests/test_gpu_slabs.py).
  * `SlabRun(..., group=process_group)` one slab per rank of torch.distributed (NCCL over NVLink): halos by
                                        batch_isend_irecv, dt by all_reduce(MIN) in place on the device.
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Tuple

import numpy as np

from . import workloads as W
from .binding import PLAN_SEAM_ABOVE

EXTERNAL = 3   # FARGO_EXTERNAL of include/fargo.h


def slab_ranges(ny: int, nslabs: int) -> List[Tuple[int, int]]:
    """Rows [j0, j1) of each slab: as even as possible, the first ny % nslabs slabs one row longer; >= 3 rows each
    (a halo message is the 3 active rows next to the cut)."""
    if nslabs < 1 or ny < 3 * nslabs:
        raise ValueError("every slab needs at least 3 rows")
    base, extra = divmod(ny, nslabs)
    out, j = [], 0
    for r in range(nslabs):
        n = base + (1 if r < extra else 0)
        out.append((j, j + n))
        j += n
    return out


def neighbours(rank: int, nslabs: int, periodic_y: bool) -> Tuple[Optional[int], Optional[int]]:
    """(slab below, slab above) of `rank`; None at a real boundary.  With one slab there is no cut at all."""
    if nslabs == 1:
        return None, None
    lo = rank - 1 if rank > 0 else (nslabs - 1 if periodic_y else None)
    hi = rank + 1 if rank + 1 < nslabs else (0 if periodic_y else None)
    return lo, hi


def _edges_beyond(edges, n, j0, j1, lo, hi, ng=3):
    """The ng edges beyond a cut face = those of the undivided mesh, ghost continuation included (at a periodic seam
    the library continues the mesh by the width of the adjacent cell: the same rule, the same fp64 operations, here)."""
    e = np.asarray(edges, dtype=np.float64)
    full = np.empty(n + 1 + 2 * ng)
    full[ng:ng + n + 1] = e
    wlo, whi = e[1] - e[0], e[n] - e[n - 1]
    for g in range(1, ng + 1):
        full[ng - g] = e[0] - float(g) * wlo
        full[ng + n + g] = e[n] + float(g) * whi
    return (None if lo is None else full[j0:j0 + ng].copy(), None if hi is None else full[ng + j1 + 1:ng + j1 + 1 + ng].copy())


def grid_coords(rank: int, grid: Tuple[int, int]) -> Tuple[int, int]:
    """(position along Y, position along Z) of `rank` in a py x pz grid of sub-domains (Y fastest)."""
    return rank % grid[0], rank // grid[0]


def slab_mesh(mesh: W.Mesh, rank: int, nslabs):
    """The sub-mesh of sub-domain `rank` (true edges: curvilinear meshes need them) and its (row range, plane range).
    nslabs: an int (slabs in Y only) or (py, pz)."""
    grid = (nslabs, 1) if isinstance(nslabs, int) else tuple(nslabs)
    ry, rz = grid_coords(rank, grid)
    j0, j1 = slab_ranges(mesh.ny, grid[0])[ry]
    k0, k1 = slab_ranges(mesh.nz, grid[1])[rz] if grid[1] > 1 else (0, mesh.nz)
    ylo, yhi = neighbours(ry, grid[0], mesh.bc[1][0] == W.PERIODIC)
    zlo, zhi = neighbours(rz, grid[1], mesh.bc[2][0] == W.PERIODIC)
    bcy = (mesh.bc[1][0] if ylo is None else EXTERNAL, mesh.bc[1][1] if yhi is None else EXTERNAL)
    bcz = (mesh.bc[2][0] if zlo is None else EXTERNAL, mesh.bc[2][1] if zhi is None else EXTERNAL)
    yext = _edges_beyond(mesh.yedges, mesh.ny, j0, j1, ylo, yhi) if (ylo is not None or yhi is not None) else None
    zext = _edges_beyond(mesh.zedges, mesh.nz, k0, k1, zlo, zhi) if (zlo is not None or zhi is not None) else None
    sub = W.Mesh(mesh.nx, j1 - j0, k1 - k0, mesh.xmin, mesh.xmax, np.ascontiguousarray(np.asarray(mesh.yedges)[j0:j1 + 1]),
                 np.ascontiguousarray(np.asarray(mesh.zedges)[k0:k1 + 1]), (mesh.bc[0], bcy, bcz), zedges_ext=zext, yedges_ext=yext)
    return sub, ((j0, j1), (k0, k1))


def exchange_plan(rank: int, nslabs: int, periodic_y: bool):
    """What sub-domain number `rank` of a line of `nslabs` sends and receives in one halo exchange along that line: a
    list of (peer, side_packed_here, side_unpacked_here).  The layers packed next to my LOWER face fill the UPPER
    ghosts of the sub-domain below me, and vice versa."""
    lo, hi = neighbours(rank, nslabs, periodic_y)
    plan = []
    if lo is not None:
        plan.append((lo, 0, 0))   # send my lower rows to `lo`; receive its upper rows into my lower ghosts
    if hi is not None:
        plan.append((hi, 1, 1))
    return plan


def route_halos(dist, group, plan, send, recv):
    """The messages of one exchange for this rank: send[side] goes to the neighbour on that side, recv[side] is filled
    by it.  Sends are posted lower side first, receives upper side first: when both neighbours are the SAME rank
    (two slabs, periodic Y) its first message (its lower rows) is the one that belongs beyond my upper face."""
    ops = [dist.P2POp(dist.isend, send[side], peer, group) for peer, side, _ in plan]
    ops += [dist.P2POp(dist.irecv, recv[side], peer, group) for peer, _, side in reversed(plan)]
    for w in (dist.batch_isend_irecv(ops) if ops else []):
        w.wait()


class SlabRun:
    """One mesh advanced as a grid of sub-domains: `nslabs` = N (Y slabs) or (py, pz), all on this device (local
    transport), or one sub-domain per rank of `group` (NCCL transport; `grid` = (py, pz), default (world size, 1))."""

    def __init__(self, mesh, geometry, eos, params, nslabs=None, group=None, precision: int = 64, grid=None):
        import torch
        from .binding import Fargo
        self._torch = torch
        self.mesh, self.group = mesh, group
        self.periodic = (None, mesh.bc[1][0] == W.PERIODIC, mesh.bc[2][0] == W.PERIODIC)
        if group is not None:
            import torch.distributed as dist
            self._dist = dist
            world = dist.get_world_size(group)
            self.grid = tuple(grid) if grid else (world, 1)
            assert self.grid[0] * self.grid[1] == world
            self.ranks = [dist.get_rank(group)]
        else:
            self.grid = (int(nslabs), 1) if isinstance(nslabs, int) else tuple(nslabs)
            self.ranks = list(range(self.grid[0] * self.grid[1]))
        self.nslabs = self.grid[0] * self.grid[1]
        self.stream = torch.cuda.Stream()
        self.ctx, self.rows, self.planes = {}, {}, {}
        prm = dataclasses.replace(params)
        with torch.cuda.stream(self.stream):          # every context picks up this (non-default) stream
            for r in self.ranks:
                sub, (rows, planes) = slab_mesh(mesh, r, self.grid)
                # the last sub-domain of a periodic Y axis: its upper cut is the seam, no ring pair of Eq. 73 across it
                seam = self.periodic[1] and self.grid[0] > 1 and grid_coords(r, self.grid)[0] == self.grid[0] - 1
                self.ctx[r] = Fargo(sub, geometry, eos, prm, precision=precision, use_graph=True,   # one graph per phase
                                    kernel_plan=PLAN_SEAM_ABOVE if seam else 0)
                self.rows[r], self.planes[r] = rows, planes
        self._buf = {}

    # ---- fields --------------------------------------------------------------------------------------
    def set_fields(self, rho, e, vx, vy=None, vz=None):
        for r in self.ranks:
            (j0, j1), (k0, k1) = self.rows[r], self.planes[r]
            self.ctx[r].set_fields(*[None if a is None else np.ascontiguousarray(np.asarray(a)[k0:k1, j0:j1, :])
                                     for a in (rho, e, vx, vy, vz)])

    def get_fields(self):
        """Local transport: the whole mesh; NCCL transport: this rank's block (see self.rows, self.planes)."""
        parts = {r: self.ctx[r].get_fields() for r in self.ranks}
        if self.group is not None:
            return parts[self.ranks[0]]
        py, pz = self.grid
        out = []
        for f in range(5):
            if parts[0][f] is None:
                out.append(None)
                continue
            out.append(np.concatenate([np.concatenate([parts[ry + py * rz][f] for ry in range(py)], axis=1)
                                       for rz in range(pz)], axis=0))
        return tuple(out)

    def time(self):
        return self.ctx[self.ranks[0]].time()

    # ---- one update ----------------------------------------------------------------------------------
    def _buffers(self, r, which, direction):
        key = (r, which, direction)
        if key not in self._buf:
            n = self.ctx[r].halo_bytes(which, direction)
            mk = lambda: self._torch.empty(n, dtype=self._torch.uint8, device=self.ctx[r].device)
            self._buf[key] = {"send": [mk(), mk()], "recv": [mk(), mk()]}
        return self._buf[key]

    def _plan(self, r, direction):
        """exchange_plan along Y (direction 1) or Z (2), with the peers as ranks of the grid."""
        py, pz = self.grid
        ry, rz = grid_coords(r, self.grid)
        if direction == 1:
            return [(p + py * rz, a, b) for p, a, b in exchange_plan(ry, py, self.periodic[1])]
        return [(ry + py * p, a, b) for p, a, b in exchange_plan(rz, pz, self.periodic[2])]

    def _exchange(self, which, direction):
        plans = {r: self._plan(r, direction) for r in self.ranks}
        if not any(plans.values()):
            return
        for r in self.ranks:                               # pack the active layers next to every cut
            for _, side, _ in plans[r]:
                self.ctx[r].halo(which, direction, side, True, self._buffers(r, which, direction)["send"][side])
        if self.group is None:                             # local: my neighbour's send buffer is my message
            for r in self.ranks:
                for peer, _, side in plans[r]:
                    self.ctx[r].halo(which, direction, side, False, self._buffers(peer, which, direction)["send"][1 - side])
            return
        r = self.ranks[0]
        b = self._buffers(r, which, direction)
        route_halos(self._dist, self.group, plans[r], b["send"], b["recv"])
        for _, _, side in plans[r]:
            self.ctx[r].halo(which, direction, side, False, b["recv"][side])

    def _reduce_dt(self):
        if self.group is None:   # one device, one stream: pairwise min into the first sub-domain, then back out (our own kernel)
            first = self.ctx[self.ranks[0]]
            for r in self.ranks[1:]:
                first.dt_min_with(self.ctx[r])
            for r in self.ranks[1:]:
                self.ctx[r].dt_min_with(first)
        else:
            self._dist.all_reduce(self.ctx[self.ranks[0]].dt_tensor(), op=self._dist.ReduceOp.MIN, group=self.group)

    def _phase(self, p):
        for r in self.ranks:
            self.ctx[r].update_phase(p)

    def step(self, n: int = 1):
        with self._torch.cuda.stream(self.stream):
            for _ in range(n):
                self._exchange(0, 1)                       # cell 2: Y halos of the state ...
                self._phase(0)                             # ... ghost fill of the faces that are not cut ...
                self._exchange(0, 2)                       # ... Z halos (the planes carry the Y ghosts: edges, corners)
                self._phase(1)                             # cells 3-6
                self._reduce_dt()                          # minimum over the sub-domains
                self._phase(2)                             # cell 7
                self._exchange(1, 1)                       # cell 9, the same way for (e, v)
                self._phase(3)
                self._exchange(1, 2)
                self._phase(4)                             # cell 12

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        for c in self.ctx.values():
            c.close()
