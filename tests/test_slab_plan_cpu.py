"""Host logic of the slab decomposition (paper_2510_18968_b200/slab.py) on CPU: the z ranges,
the exchange partners, and the halo exchange itself over ``torch.distributed`` with the gloo backend (world sizes 2 and
3), on a stand-in handle whose pack / unpack follow the C-ABI's definition (rgrmhd_halo_pack / rgrmhd_halo_unpack) on
NumPy arrays.  Expected ghost planes come from np.pad of the undivided array (wrap = periodic, edge = outflow)."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2510_18968_b200 import slab, workloads as wl  # noqa: E402


def test_slab_ranges_and_neighbours():
    assert slab.slab_ranges(10, 3) == [(0, 4), (4, 7), (7, 10)]
    assert slab.slab_ranges(512, 8) == [(64 * r, 64 * (r + 1)) for r in range(8)]
    with pytest.raises(ValueError):
        slab.slab_ranges(8, 3)                                       # a halo is 3 planes deep
    assert slab.neighbours(0, 4, wl.BC_OUTFLOW) == (None, 1) and slab.neighbours(3, 4, wl.BC_OUTFLOW) == (2, None)
    assert slab.neighbours(0, 4, wl.BC_PERIODIC) == (3, 1) and slab.neighbours(3, 4, wl.BC_PERIODIC) == (2, 0)
    assert slab.neighbours(0, 2, wl.BC_PERIODIC) == (1, 1)           # two slabs: both partners are the other one
    # every send has its matching receive with the same tag on the other side
    for world in (2, 3, 5):
        for bc in (wl.BC_PERIODIC, wl.BC_OUTFLOW):
            msgs = {}
            for r in range(world):
                for op, peer, side in slab.exchange_plan(r, world, bc):
                    key = (r, peer, 1 - side) if op == "send" else (peer, r, side)      # (from, to, tag)
                    msgs.setdefault(key, []).append(op)
            assert all(sorted(v) == ["recv", "send"] for v in msgs.values()), (world, bc, msgs)


class FakeHandle:
    """pack / unpack of the C-ABI on a NumPy array f[field, z, y, x] with 3 ghost planes below and above."""

    def __init__(self, arr):
        self.f = arr

    def halo_pack(self, direction, side, buf):
        assert direction == 2
        nz = self.f.shape[1] - 6
        sl = slice(3, 6) if side == 0 else slice(3 + nz - 3, 3 + nz)
        buf.copy_(torch.from_numpy(np.ascontiguousarray(self.f[:, sl]).reshape(-1)))

    def halo_unpack(self, direction, side, buf):
        nz = self.f.shape[1] - 6
        sl = slice(0, 3) if side == 0 else slice(3 + nz, 6 + nz)
        self.f[:, sl] = buf.numpy().reshape(self.f[:, sl].shape)


def _global_field(nz, ny=5, nx=4):
    rng = np.random.default_rng(99)
    return rng.standard_normal((slab.NFIELDS, nz, ny, nx))


def _worker(rank, world, port, bc, nz, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch.distributed as dist
    dist.init_process_group("gloo")
    G = _global_field(nz)
    lo, hi = slab.slab_ranges(nz, world)[rank]
    local = np.full((slab.NFIELDS, hi - lo + 6) + G.shape[2:], np.nan)
    local[:, 3:-3] = G[:, lo:hi]
    h = FakeHandle(local)
    m = slab.NFIELDS * 3 * G.shape[2] * G.shape[3]
    send = [torch.empty(m, dtype=torch.float64) for _ in range(2)]
    recv = [torch.empty(m, dtype=torch.float64) for _ in range(2)]
    h.halo_pack(2, 0, send[0]); h.halo_pack(2, 1, send[1])
    got = slab.dist_exchange(dist, send, recv, rank, world, bc)
    for side in (0, 1):
        h.halo_unpack(2, side, recv[side] if side in got else slab.outflow_ghost(send[side], side))
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, lo, hi, local))


@pytest.mark.parametrize("world,bc", [(2, wl.BC_PERIODIC), (2, wl.BC_OUTFLOW), (3, wl.BC_PERIODIC), (3, wl.BC_OUTFLOW)])
def test_halo_exchange_gloo(world, bc):
    nz = 11
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() * 7 + world * 3 + bc) % 2000
    ps = [ctx.Process(target=_worker, args=(r, world, port, bc, nz, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = [q.get(timeout=180) for _ in ps]
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    G = _global_field(nz)
    padded = np.pad(G, [(0, 0), (3, 3), (0, 0), (0, 0)], mode="wrap" if bc == wl.BC_PERIODIC else "edge")
    for rank, lo, hi, local in out:
        assert np.array_equal(local, padded[:, lo:hi + 6]), rank       # interior + both halos, bit for bit
