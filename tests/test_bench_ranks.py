"""The N>1 path of bench.py is "replicas only": ranks own independent worlds, the only
communication is a barrier and a MAX over the ranks' times.  Covered here with world_size-2 gloo
on CPU: seeds differ per rank, the aggregate counts every rank's beads once, time = max."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_02954_b200 import worlds


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank(rank, world_size, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world_size)
    w = worlds.make_world("4a", seed=rank)          # replicas: same recipe, seed = rank
    n = int(w["offsets"][-1])
    ms = torch.tensor([10.0 + 5.0 * rank], dtype=torch.float64)  # stand-in for this rank's device time
    dist.barrier()
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    chk = torch.tensor([float(np.asarray(w["xy"], dtype=np.float64).sum())], dtype=torch.float64)
    gathered = [torch.zeros_like(chk) for _ in range(world_size)]
    dist.all_gather(gathered, chk)
    steps = 7
    value = world_size * n * steps / (float(ms.item()) * 1e-3)
    if rank == 0:
        out.put((value, float(ms.item()), [float(g.item()) for g in gathered], n))
    dist.destroy_process_group()


def test_replicas_aggregate_two_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_rank, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    value, ms, sums, n = q.get()
    assert ms == 15.0                                # max over ranks, not mean
    assert sums[0] != sums[1]                        # the two ranks own different worlds
    assert abs(value - 2 * n * 7 / 15e-3) < 1e-6 * value
