"""N > 1 host logic ("replicas only") with world_size-2 gloo on CPU: barrier +
max-over-ranks timing and the whole-job aggregate bench.py prints."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_10445_b200 import replicas


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    ms = replicas.max_over_ranks(1.0 + rank, dist)            # rank 1 is the slow one
    dist.barrier()
    out[rank] = ms
    dist.destroy_process_group()


def test_max_over_ranks_world2_gloo():
    world = 2
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
        assert out[0] == out[1] == 2.0
    assert replicas.whole_job_us_per_layer(2.0, 8, 2) == 125.0


def test_single_process_is_identity():
    assert replicas.max_over_ranks(3.5) == 3.5
    assert replicas.whole_job_us_per_layer(0.8, 8, 1) == 100.0
