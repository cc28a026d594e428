"""N > 1 path of bench.py ("replicas only") on CPU: world_size 2, gloo."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_08743_b200 import replicas


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = [10.0, 12.5][rank]                      # rank 1 is the slower replica
        pts = [1000, 1000][rank]
        value, mx = replicas.whole_job_throughput(pts, 4, ms)
        out[rank] = (value, mx, replicas.max_over_ranks(float(rank)), replicas.sum_over_ranks(1.0))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_whole_job_throughput_is_sum_of_points_over_max_time():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    for rank in (0, 1):
        value, mx, mr, sr = res[rank]
        assert mx == 12.5 and mr == 1.0 and sr == 2.0
        assert value == pytest.approx(2000 * 4 / 12.5e-3 / 1e6)


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    v, ms = replicas.whole_job_throughput(1 << 20, 10, 50.0)
    assert ms == 50.0 and v == pytest.approx((1 << 20) * 10 / 50e-3 / 1e6)
