"""Host logic of the multi-GPU halo exchange (paper_2607_08743_b200/halo.py) on CPU: gloo, world sizes
2 and 4. A periodic global grid is cut into blocks, one per rank; after exchange_halos every rank's patch -- ghosts,
edges and corners included -- must equal, bit for bit, its block of the globally ghost-filled state (numpy.pad wrap).
pack / unpack are stand-ins written here from the buffer layout sacra.h states (this container has no GPU; the CUDA
kernels are checked against the same layout in tests/test_gpu_halo.py)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_08743_b200 import halo
from paper_2607_08743_b200 import workloads as wl

NF, NG = wl.NF, wl.NG


class NumpyOps:
    """the buffer layout of sacra_pack_face / sacra_unpack_face (include/sacra.h), as numpy slicing"""

    def __init__(self, w):
        self.w = w

    def new_buffer(self, patch, axis, like):
        s = [patch.nx + 2 * NG, patch.ny + 2 * NG, patch.nz + 2 * NG]
        return torch.zeros(NF * NG * s[0] * s[1] * s[2] // s[axis], dtype=torch.float64)

    def _layers(self, patch, u, f, axis, lo):
        v = self.w.field_view(u.numpy(), 0, f)[:, :, :patch.nx + 2 * NG]        # (z, y, x) storage, pitch padding cut
        sl = [slice(None)] * 3
        sl[2 - axis] = slice(lo, lo + NG)
        return np.moveaxis(v[tuple(sl)], 2 - axis, 0)                            # layer first, then slower, faster

    def pack(self, patch, u, axis, side, buf):
        n = [patch.nx, patch.ny, patch.nz][axis]
        b = buf.numpy().reshape(NF, -1)
        for f in range(NF):
            b[f] = self._layers(patch, u, f, axis, NG if side == 0 else n).reshape(-1)

    def unpack(self, patch, u, axis, side, buf):
        n = [patch.nx, patch.ny, patch.nz][axis]
        b = buf.numpy().reshape(NF, -1)
        for f in range(NF):
            dst = self._layers(patch, u, f, axis, 0 if side == 0 else n + NG)
            dst[...] = b[f].reshape(dst.shape)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


LOCAL = (7, 6, 8)      # active cells per rank (x, y, z)


def _global_filled(dims, seed=11):
    rng = np.random.default_rng(seed)
    g = rng.normal(size=(NF, LOCAL[2] * dims[2], LOCAL[1] * dims[1], LOCAL[0] * dims[0]))
    return np.pad(g, ((0, 0), (NG, NG), (NG, NG), (NG, NG)), mode="wrap")


def _worker(rank, world, port, dims, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        topo = halo.CartTopology(dims)
        c = topo.coords(rank)
        gf = _global_filled(dims)
        ps, total = wl.make_layout([LOCAL], [0.1], [0.02], [(0, 0, 0)])
        w = wl.Workload("block", ps, dict(wl.DEFAULT_PARAMS), np.full(total, np.nan))
        o = [c[a] * LOCAL[a] for a in range(3)]
        blk = gf[:, o[2]:o[2] + LOCAL[2] + 2 * NG, o[1]:o[1] + LOCAL[1] + 2 * NG, o[0]:o[0] + LOCAL[0] + 2 * NG]
        for f in range(NF):
            w.active_view(w.state, 0, f)[...] = blk[f, NG:-NG, NG:-NG, NG:-NG]
        u = torch.from_numpy(w.state)
        bufs = {}
        sent = 0
        for _ in range(2):                                       # twice: the buffers are reused
            sent = halo.exchange_halos(ps[0], u, topo, rank, ops=NumpyOps(w), buffers=bufs)
        ok = all(np.array_equal(w.field_view(u.numpy(), 0, f)[:, :, :LOCAL[0] + 2 * NG], blk[f]) for f in range(NF))
        out[rank] = (ok, sent)
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("dims", [(1, 1, 2), (2, 1, 1), (2, 1, 2), (1, 3, 1)])
def test_exchange_fills_every_ghost_like_the_global_periodic_fill(dims):
    world, port = dims[0] * dims[1] * dims[2], _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, dims, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == set(range(world))
    nmsg = 2 * sum(1 for d in dims if d > 1)
    for r in range(world):
        assert res[r] == (True, nmsg), (r, res[r])


def test_topology_neighbours():
    t = halo.CartTopology((2, 3, 4))
    assert t.size == 24
    for r in range(24):
        assert t.rank_of(t.coords(r)) == r
        for a in range(3):
            assert t.neighbour(t.neighbour(r, a, 0), a, 1) == r
    assert t.neighbour(0, 0, 0) == 1 and t.neighbour(0, 1, 0) == 4 and t.neighbour(0, 2, 0) == 18 and t.neighbour(23, 2, 1) == 5
