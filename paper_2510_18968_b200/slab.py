"""Slab decomposition of one block along z with a halo exchange per stage (the paper's
"boxes" on MPI ranks with ghost-zone synchronisation).

Each slab is an ordinary handle of the C-ABI whose z direction is ``RGRMHD_BC_EXTERNAL``: the library fills the x and y
ghosts of every plane it owns, the three ghost planes below and above belong to this module.  Per right-hand side one
exchange of 3 planes x 17 fields (14 stage primitives + 3 conduction-current components) per shared face, at the two
exchange points of the split step (``rgrmhd_step_begin`` / ``rgrmhd_step_continue``); recovery, sources and the stage
algebra are point-wise and need nothing.  The planes travel over their FULL padded x-y extent, i.e. with the x / y ghost
columns the sender has just filled, which makes the result identical (bit for bit) to the single-block ghost fill
"x, then y, then z".  At a global boundary: periodic = the exchange partner is the slab at the other end; outflow = the
three ghost planes are copies of the boundary plane.  The CFL reduction is a max over slabs.

Argument marshalling and plumbing only -- every kernel is the library's:

* ``LocalSlabs``: all slabs in ONE process on one GPU, stepped part by part in turn (no kernel ever waits for another):
  the correctness harness (tests compare it bit for bit with the undivided block);
* ``DistSlab``: one slab per ``torch.distributed`` rank (NCCL send/recv of CUDA buffers on the GPU box; the exchange
  plan is covered on CPU with gloo).  This build's GPU box has ONE GPU, so the multi-rank path is unmeasured.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np

from . import workloads as wl

NFIELDS = 17


def slab_ranges(nz: int, nslabs: int) -> List[Tuple[int, int]]:
    """Balanced z ranges [lo, hi) of ``nslabs`` slabs; every slab needs >= 3 planes (a halo is 3 deep)."""
    if nslabs < 1 or nz < 3 * nslabs:
        raise ValueError("need at least 3 planes per slab")
    base, rem = divmod(nz, nslabs)
    out, lo = [], 0
    for r in range(nslabs):
        hi = lo + base + (1 if r < rem else 0)
        out.append((lo, hi))
        lo = hi
    return out


def neighbours(rank: int, world: int, bc_z: int) -> Tuple[Optional[int], Optional[int]]:
    """(lower, upper) exchange partner of a slab; None = a global outflow boundary."""
    lower = rank - 1 if rank > 0 else (world - 1 if bc_z == wl.BC_PERIODIC else None)
    upper = rank + 1 if rank < world - 1 else (0 if bc_z == wl.BC_PERIODIC else None)
    return lower, upper


def outflow_ghost(own_send, side: int):
    """Ghost planes of a global outflow boundary from the slab's own packed interior layers (layer order = increasing
    z): three copies of the plane next to the boundary ("copied from the nearest interior point")."""
    v = own_send.view(NFIELDS, 3, -1)
    near = v[:, 0:1] if side == 0 else v[:, 2:3]
    return near.expand(NFIELDS, 3, v.shape[2]).contiguous().view(-1)


class _SlabBase:
    def _make(self, binding, w, rank, world, device, fields, rhs_variant):
        import torch
        self.w, self.rank, self.world = w, rank, world
        self.lo, self.hi = slab_ranges(w.n[2], world)[rank]
        self.n = (w.n[0], w.n[1], self.hi - self.lo)
        self.external = world > 1
        bc = (w.bc[0], w.bc[1], wl.BC_EXTERNAL if self.external else w.bc[2])
        f = fields if fields is not None else w.fields((0, 0, self.lo), self.n)
        self.g = binding.from_workload(w, fields=f, n=self.n, bc=bc, device=device)
        self.g.set_rhs_variant(rhs_variant)
        self.lower, self.upper = neighbours(rank, world, w.bc[2])
        if self.external:
            m = self.g.halo_doubles(2)
            dev = torch.device("cuda", device)
            self.send = [torch.empty(m, dtype=torch.float64, device=dev) for _ in range(2)]
            self.recv = [torch.empty(m, dtype=torch.float64, device=dev) for _ in range(2)]

    def pack(self):
        self.g.halo_pack(2, 0, self.send[0])
        self.g.halo_pack(2, 1, self.send[1])

    def interior_prims(self) -> np.ndarray:
        P = self.g.get_prims()
        return P[:, 3:-3, 3:-3, 3:-3]

    def interior_cons(self) -> np.ndarray:
        U = self.g.get_cons()
        return U[:, 3:-3, 3:-3, 3:-3]


class LocalSlabs:
    """``nslabs`` slabs of workload ``w`` in one process on one GPU (see the module docstring)."""

    def __init__(self, binding, w, nslabs: int, device: int = 0, rhs_variant: int = 0):
        self.w = w
        self.slabs = []
        for r in range(nslabs):
            s = _SlabBase()
            s._make(binding, w, r, nslabs, device, None, rhs_variant)
            self.slabs.append(s)

    def _exchange(self):
        if len(self.slabs) == 1:
            return
        for s in self.slabs:
            s.pack()
        for s in self.slabs:
            for side, nb in ((0, s.lower), (1, s.upper)):
                if nb is None:
                    buf = outflow_ghost(s.send[side], side)
                else:
                    buf = self.slabs[nb].send[1 - side]      # lower ghost <- the partner's UPPER interior layers
                s.g.halo_unpack(2, side, buf)

    def max_speed(self) -> float:
        return max(s.g.max_speed() for s in self.slabs)

    def step(self, dt: float, scheme: int):
        if len(self.slabs) == 1:
            self.slabs[0].g.step(dt, scheme)
            return
        for s in self.slabs:
            s.g.step_begin(dt, scheme)
        self._exchange()
        for s in self.slabs:
            assert s.g.step_continue()
        self._exchange()
        for s in self.slabs:
            assert not s.g.step_continue()

    def gather_prims(self) -> np.ndarray:
        return np.concatenate([s.interior_prims() for s in self.slabs], axis=1)

    def gather_cons(self) -> np.ndarray:
        return np.concatenate([s.interior_cons() for s in self.slabs], axis=1)


def exchange_plan(rank: int, world: int, bc_z: int):
    """The point-to-point operations of one halo exchange of ``rank``: a list of (op, peer, side) with op 'send' /
    'recv'; side = which of the rank's own buffers (0 = lower, 1 = upper).  A slab sends its lower interior layers to its
    lower partner and receives that partner's upper layers into its lower ghosts, and vice versa.  With two slabs and
    periodic boundaries both partners are the same rank: the tags below keep the two messages apart."""
    lower, upper = neighbours(rank, world, bc_z)
    plan = []
    for side, nb in ((0, lower), (1, upper)):
        if nb is not None:
            plan.append(("send", nb, side))
            plan.append(("recv", nb, side))
    return plan


def dist_exchange(dist, send, recv, rank: int, world: int, bc_z: int):
    """Run the plan with ``torch.distributed`` point-to-point operations.  ``send`` / ``recv``: the two packed buffers
    (index = side).  Returns the sides that were received (the others are global outflow boundaries)."""
    ops, got = [], []
    for op, peer, side in exchange_plan(rank, world, bc_z):
        # tag = the side as the RECEIVER numbers it: data sent from my side s arrives in the peer's side 1 - s
        if op == "send":
            ops.append(dist.P2POp(dist.isend, send[side], peer, tag=1 - side))
        else:
            ops.append(dist.P2POp(dist.irecv, recv[side], peer, tag=side))
            got.append(side)
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    return got


class DistSlab(_SlabBase):
    """One slab per ``torch.distributed`` rank (process group already initialised; NCCL for CUDA buffers)."""

    def __init__(self, binding, w, device: int = 0, rhs_variant: int = 0):
        import torch.distributed as dist
        self.dist = dist
        self._make(binding, w, dist.get_rank(), dist.get_world_size(), device, None, rhs_variant)

    def _exchange(self):
        if not self.external:
            return
        import torch
        self.pack()
        # the packs run on the handle's stream; the transport uses the current stream
        torch.cuda.current_stream().synchronize()
        got = dist_exchange(self.dist, self.send, self.recv, self.rank, self.world, self.w.bc[2])
        for side in (0, 1):
            buf = self.recv[side] if side in got else outflow_ghost(self.send[side], side)
            self.g.halo_unpack(2, side, buf)

    def max_speed(self) -> float:
        import torch
        t = torch.tensor([self.g.max_speed()], dtype=torch.float64, device=self.send[0].device if self.external else "cuda")
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def step(self, dt: float, scheme: int):
        if not self.external:
            self.g.step(dt, scheme)
            return
        self.g.step_begin(dt, scheme)
        self._exchange()
        assert self.g.step_continue()
        self._exchange()
        assert not self.g.step_continue()
