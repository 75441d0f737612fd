"""Slab decomposition in Y over several contexts (section 4.1).

The paper splits the mesh in Y (and Z), never in X, exchanges 3 ghost layers at cells 2 and 9 of Fig. 2 and takes the
minimum of the time step over the sub-domains.  Here a slab is an ordinary context (C ABI, include/fargo.h)
whose cut Y faces have the kind FARGO_EXTERNAL; this module only does the plumbing the ABI leaves to the caller:
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


def slab_mesh(mesh: W.Mesh, rank: int, nslabs: int) -> Tuple[W.Mesh, Tuple[int, int]]:
    """The sub-mesh of slab `rank` (true Y edges: curvilinear meshes need them) and its row range."""
    j0, j1 = slab_ranges(mesh.ny, nslabs)[rank]
    per = mesh.bc[1][0] == W.PERIODIC
    lo, hi = neighbours(rank, nslabs, per)
    bcy = (mesh.bc[1][0] if lo is None else EXTERNAL, mesh.bc[1][1] if hi is None else EXTERNAL)
    # the edges beyond a cut face are those of the undivided mesh, ghost continuation included (at a periodic seam the
    # library continues the mesh by the width of the adjacent cell: the same rule, the same fp64 operations, here)
    ye = np.asarray(mesh.yedges, dtype=np.float64)
    ng, n = 3, mesh.ny
    full = np.empty(n + 1 + 2 * ng)
    full[ng:ng + n + 1] = ye
    wlo, whi = ye[1] - ye[0], ye[n] - ye[n - 1]
    for g in range(1, ng + 1):
        full[ng - g] = ye[0] - float(g) * wlo
        full[ng + n + g] = ye[n] + float(g) * whi
    ext = (None if lo is None else full[j0:j0 + ng].copy(), None if hi is None else full[ng + j1 + 1:ng + j1 + 1 + ng].copy())
    sub = W.Mesh(mesh.nx, j1 - j0, mesh.nz, mesh.xmin, mesh.xmax, np.ascontiguousarray(ye[j0:j1 + 1]),
                 mesh.zedges, (mesh.bc[0], bcy, mesh.bc[2]), yedges_ext=ext)
    return sub, (j0, j1)


def exchange_plan(rank: int, nslabs: int, periodic_y: bool):
    """What slab `rank` sends and receives in one halo exchange: a list of (peer, side_packed_here, side_unpacked_here).
    The rows packed next to my LOWER face fill the UPPER ghosts of the slab below me, and vice versa."""
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
    """One mesh advanced as `nslabs` slabs (local transport) or as one slab per rank of `group` (NCCL transport)."""

    def __init__(self, mesh, geometry, eos, params, nslabs: Optional[int] = None, group=None, precision: int = 64):
        import torch
        from .binding import Fargo
        self._torch = torch
        self.mesh, self.group = mesh, group
        self.periodic_y = mesh.bc[1][0] == W.PERIODIC
        if group is not None:
            import torch.distributed as dist
            self._dist = dist
            self.nslabs, self.ranks = dist.get_world_size(group), [dist.get_rank(group)]
        else:
            self.nslabs, self.ranks = int(nslabs), list(range(int(nslabs)))
        self.stream = torch.cuda.Stream()
        self.ctx, self.rows = {}, {}
        prm = dataclasses.replace(params)
        with torch.cuda.stream(self.stream):          # every context picks up this (non-default) stream
            for r in self.ranks:
                sub, rows = slab_mesh(mesh, r, self.nslabs)
                self.ctx[r] = Fargo(sub, geometry, eos, prm, precision=precision, use_graph=False)
                self.rows[r] = rows
        self._buf = {}

    # ---- fields --------------------------------------------------------------------------------------
    def set_fields(self, rho, e, vx, vy=None, vz=None):
        for r in self.ranks:
            j0, j1 = self.rows[r]
            self.ctx[r].set_fields(*[None if a is None else np.ascontiguousarray(np.asarray(a)[:, j0:j1, :])
                                     for a in (rho, e, vx, vy, vz)])

    def get_fields(self):
        """Local transport: the whole mesh; NCCL transport: this rank's rows (see self.rows)."""
        parts = [self.ctx[r].get_fields() for r in self.ranks]
        return tuple(None if parts[0][f] is None else np.concatenate([p[f] for p in parts], axis=1) for f in range(5))

    def time(self):
        return self.ctx[self.ranks[0]].time()

    # ---- one update ----------------------------------------------------------------------------------
    def _buffers(self, r, which):
        key = (r, which)
        if key not in self._buf:
            n = self.ctx[r].halo_bytes(which)
            mk = lambda: self._torch.empty(n, dtype=self._torch.uint8, device=self.ctx[r].device)
            self._buf[key] = {"send": [mk(), mk()], "recv": [mk(), mk()]}
        return self._buf[key]

    def _exchange(self, which):
        plans = {r: exchange_plan(r, self.nslabs, self.periodic_y) for r in self.ranks}
        for r in self.ranks:                               # pack the active rows next to every cut
            for _, side, _ in plans[r]:
                self.ctx[r].halo(which, side, True, self._buffers(r, which)["send"][side])
        if self.group is None:                             # local: my neighbour's send buffer is my message
            for r in self.ranks:
                for peer, _, side in plans[r]:
                    self.ctx[r].halo(which, side, False, self._buffers(peer, which)["send"][1 - side])
            return
        r = self.ranks[0]
        b = self._buffers(r, which)
        route_halos(self._dist, self.group, plans[r], b["send"], b["recv"])
        for _, _, side in plans[r]:
            self.ctx[r].halo(which, side, False, b["recv"][side])

    def _reduce_dt(self):
        views = [self.ctx[r].dt_tensor() for r in self.ranks]
        if self.group is None:
            m = self._torch.stack(views).min(dim=0).values
            for v in views:
                v.copy_(m)
        else:
            self._dist.all_reduce(views[0], op=self._dist.ReduceOp.MIN, group=self.group)

    def step(self, n: int = 1):
        with self._torch.cuda.stream(self.stream):
            for _ in range(n):
                self._exchange(0)                          # cell 2: halos of the state
                for r in self.ranks:
                    self.ctx[r].update_phase(0)
                self._reduce_dt()                          # cell 6: minimum over the sub-domains
                for r in self.ranks:
                    self.ctx[r].update_phase(1)
                self._exchange(1)                          # cell 9: halos of (e, v) after the source step
                for r in self.ranks:
                    self.ctx[r].update_phase(2)

    def synchronize(self):
        self.stream.synchronize()

    def close(self):
        for c in self.ctx.values():
            c.close()
