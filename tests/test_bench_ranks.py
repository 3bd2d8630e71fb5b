"""The N>1 path of bench.py is "replicas only": ranks own independent worlds, the only
communication is a barrier and a MAX over the ranks' times.  Covered here with world_size-2 gloo
on CPU: seeds differ per rank, the aggregate counts every rank's beads once, time = max."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench  # the repo-root bench.py: its aggregate() is what the N>1 run reports
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
    value = bench.aggregate(n, steps, world_size, float(ms.item()))  # bench.py's own formula
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
    assert abs(value - 2 * n * 7 / 15e-3) < 1e-6 * value   # both ranks' beads over the slower rank's time


def test_byte_models_and_stale_traffic_guard(tmp_path, monkeypatch):
    # the four step models differ by exactly the G round trip (16 B/node) and the gather reads (16 B/node)
    nc, nb = 1000, 10
    assert bench.step_bytes(nc, nb, model="raw") == 112 * nc + 64 * nb
    assert bench.step_bytes(nc, nb, model="raw") - bench.step_bytes(nc, nb, model="reduced") == 16 * nc
    assert bench.step_bytes(nc, nb, model="raw_with_gathers") - bench.step_bytes(nc, nb, model="raw") == 16 * nc
    assert bench.step_bytes(nc, nb, model="reduced_with_gathers") == bench.step_bytes(nc, nb, model="raw")
    # per-kernel models: the node bytes add up to the reduced step model; the bead bytes exceed the
    # step's 64 B/bead by the three extra reads of X (the step model counts X once, four kernels read it)
    assert sum(bench.kernel_bytes(nc, 0).values()) == bench.step_bytes(nc, 0, model="reduced")
    assert sum(bench.kernel_bytes(0, nb).values()) == bench.step_bytes(0, nb, model="reduced") + 3 * 8 * nb
    # an ncu capture of another build must be refused
    import json
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    (tmp_path / "profiles").mkdir()
    (tmp_path / "paper_2607_02954_b200" / "csrc").mkdir(parents=True)
    (tmp_path / "paper_2607_02954_b200" / "csrc" / "a.cu").write_text("x")
    sha = bench.csrc_sha()
    (tmp_path / "profiles" / "r2_traffic.json").write_text(json.dumps(
        {"csrc_sha": "deadbeef", "world": "4d", "dram_bytes_per_launch": {"k_lbm_spread_tile": 5.0}}))
    v, note = bench.ncu_traffic("K3b_lbm", "4d")
    assert v is None and "stale" in note
    (tmp_path / "profiles" / "r2_traffic.json").write_text(json.dumps(
        {"csrc_sha": sha, "world": "4d", "command": "c", "dram_bytes_per_launch": {"k_lbm_spread_tile": 5.0}}))
    v, note = bench.ncu_traffic("K3b_lbm", "4d")
    assert v == 5.0
