"""Halo exchange of a 3-D block decomposition over several GPUs ("the ghost layers
are packed into buffers and exchanged with non-blocking GPU-aware point-to-point calls before each Runge-Kutta
substage"; PAPER.md:378 lists overlapping the exchange with the computation as future work).

One process per GPU. Every rank owns one patch of the same size; the ranks form a px x py x pz Cartesian grid over a
periodic global domain. Only the host logic lives here -- who talks to whom, in which order, with which buffers; the
data movement is the library's: sacra_pack_face / sacra_unpack_face (CUDA kernels) fill and drain the buffers and
torch.distributed moves them (NCCL send/recv between GPUs, over NVLink when the ranks share a node).

    x, then y, then z. A face buffer carries the whole storage extent of the two other axes, ghosts included, so the
    ghosts received along x travel on along y and z: edges and corners need no messages of their own (6 instead of 26).

Per axis: pack low and high active layers; post the receives and sends of both directions as ONE batch (grouped: NCCL
needs matching send/recv pairs issued together to avoid a deadlock); wait; unpack. An axis with a single rank is its own
neighbour: the two packed buffers are unpacked locally, without a message.

`ops` supplies pack / unpack / new_buffer: the default (`CudaOps`) calls the library; tests drive the same exchange
logic on the CPU (gloo) with a stand-in that slices numpy views, since this container has no GPU.
"""
from __future__ import annotations

from dataclasses import dataclass


@dataclass(frozen=True)
class CartTopology:
    """px x py x pz ranks, x fastest: rank = cx + px (cy + py cz). The global domain is periodic."""
    dims: tuple

    @property
    def size(self) -> int:
        return self.dims[0] * self.dims[1] * self.dims[2]

    def coords(self, rank: int):
        px, py, _ = self.dims
        return (rank % px, (rank // px) % py, rank // (px * py))

    def rank_of(self, c) -> int:
        px, py, pz = self.dims
        return (c[0] % px) + px * ((c[1] % py) + py * (c[2] % pz))

    def neighbour(self, rank: int, axis: int, side: int) -> int:
        """rank of the neighbour behind the low (side 0) or high (side 1) face along the axis"""
        c = list(self.coords(rank))
        c[axis] += 1 if side else -1
        return self.rank_of(c)


class CudaOps:
    """the library's kernels on torch CUDA tensors"""

    def __init__(self, stream=None):
        self.stream = stream

    def new_buffer(self, patch, axis, like):
        import torch
        from . import sacra
        return torch.empty(sacra.face_doubles(patch, axis), dtype=torch.float64, device=like.device)

    def pack(self, patch, u, axis, side, buf):
        from . import sacra
        sacra.pack_face(patch, u, axis, side, buf, stream=self.stream)

    def unpack(self, patch, u, axis, side, buf):
        from . import sacra
        sacra.unpack_face(patch, u, axis, side, buf, stream=self.stream)


def exchange_halos(patch, u, topo: CartTopology, rank: int, ops=None, group=None, buffers=None):
    """Fill every ghost cell of this rank's patch from its neighbours (periodic global domain). `u`: the rank's state.
    `buffers`: optional dict reused between calls (send / receive buffers per axis). Returns the number of messages sent."""
    import torch.distributed as dist
    ops = ops or CudaOps()
    buffers = buffers if buffers is not None else {}
    sent = 0
    for axis in range(3):
        key = ("face", axis)
        if key not in buffers:
            buffers[key] = [ops.new_buffer(patch, axis, u) for _ in range(4)]     # send low, send high, recv low, recv high
        s_lo, s_hi, r_lo, r_hi = buffers[key]
        ops.pack(patch, u, axis, 0, s_lo)
        ops.pack(patch, u, axis, 1, s_hi)
        lo, hi = topo.neighbour(rank, axis, 0), topo.neighbour(rank, axis, 1)
        if topo.dims[axis] == 1:
            # my own neighbour on both sides: the high layers are my low ghosts and vice versa
            ops.unpack(patch, u, axis, 0, s_hi)
            ops.unpack(patch, u, axis, 1, s_lo)
            continue
        # my low layers go to the low neighbour (its high ghosts); its high layers come back as my low ghosts
        reqs = dist.batch_isend_irecv([
            dist.P2POp(dist.irecv, r_lo, lo, group=group, tag=2 * axis + 1),
            dist.P2POp(dist.irecv, r_hi, hi, group=group, tag=2 * axis),
            # (with two ranks on the axis both messages go to the same peer: NCCL pairs them in issue order, so the
            #  high layers -- the peer's first receive, its low ghosts -- are sent first; gloo goes by the tags)
            dist.P2POp(dist.isend, s_hi, hi, group=group, tag=2 * axis + 1),
            dist.P2POp(dist.isend, s_lo, lo, group=group, tag=2 * axis),
        ])
        for r in reqs:
            r.wait()
        sent += 2
        ops.unpack(patch, u, axis, 0, r_lo)
        ops.unpack(patch, u, axis, 1, r_hi)
    return sent


def rk4_step_distributed(patch, params, u, work, topo: CartTopology, rank: int, ops=None, group=None, buffers=None,
                         overlap=False):
    """One RK4 step of this rank's block: the halo exchange stands where sacra_rk4_step has its periodic fill
    (exchange, substage, four times; exchange of the result). work: 3 states like sacra_rk4_step.

    overlap=True (PAPER.md:378 lists it as future work): per substage the cells that need no exchanged ghost
    (sacra_rk4_substep_part, PART_INTERIOR) are computed on the caller's stream WHILE the stage input's halos are packed,
    sent and unpacked on a second stream; the boundary shell (PART_SHELL) follows when both are done. Same bits."""
    from . import sacra
    n = u.numel()
    w0, w1, acc = work[:n], work[n:2 * n], work[2 * n:]
    buffers = buffers if buffers is not None else {}
    seq = [(u, w0), (w0, w1), (w1, w0), (w0, u)]
    if not overlap:
        for stage, (src, dst) in enumerate(seq, start=1):
            exchange_halos(patch, src, topo, rank, ops, group, buffers)
            sacra.rk4_substep([patch], params, stage, u, src, dst, acc)
        exchange_halos(patch, u, topo, rank, ops, group, buffers)
        return
    import torch
    main = torch.cuda.current_stream()
    if "comm_stream" not in buffers:
        buffers["comm_stream"] = torch.cuda.Stream()
    comm = buffers["comm_stream"]
    faces = [1] * 6                      # every face of a block of a periodic decomposition is an exchange face
    # the overlapped exchanges pack / unpack on the second stream through an ops object of their own: the caller's
    # `ops` (and whatever stream it carries) is left as it was and serves the final exchange below
    comm_ops = CudaOps(comm) if ops is None or isinstance(ops, CudaOps) else ops
    for stage, (src, dst) in enumerate(seq, start=1):
        comm.wait_stream(main)           # the stage input is complete
        with torch.cuda.stream(comm):
            exchange_halos(patch, src, topo, rank, comm_ops, group, buffers)
        sacra.rk4_substep_part([patch], params, stage, sacra.PART_INTERIOR, faces, u, src, dst, acc)
        main.wait_stream(comm)           # ghosts of the stage input are in place
        sacra.rk4_substep_part([patch], params, stage, sacra.PART_SHELL, faces, u, src, dst, acc)
    exchange_halos(patch, u, topo, rank, ops, group, buffers)
