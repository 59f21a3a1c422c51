"""The N > 1 path on CPU (gloo, world size 2): the hot path shards by request with NO exchange step
(DESIGN.md section 9).  Each rank takes a contiguous slice of the batch, computes the step on its
shard alone (here with the oracle, the only CPU implementation), and the gathered shards must equal the
unsharded result exactly; the timing reduction bench.py uses (max over ranks) is exercised too."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from oracle.workload_io import oracle_step


def shard_requests(batch, rank, world):
    per = (batch + world - 1) // world
    return range(min(rank * per, batch), min((rank + 1) * per, batch))


def _worker(rank, world, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2606_06453_b200.workloads import make_workload, subproblem
        w = make_workload("C5-small", device="cpu")
        mine = shard_requests(w.spec.batch, rank, world)
        ref = oracle_step(subproblem(w, mine))
        out = torch.from_numpy(ref["out"]).contiguous()
        sel = torch.from_numpy(ref["sel_logical"]).contiguous()
        outs = [torch.empty_like(out) for _ in range(world)]
        sels = [torch.empty_like(sel) for _ in range(world)]
        dist.all_gather(outs, out)            # test plumbing only: the data path itself has no collective
        dist.all_gather(sels, sel)
        t = torch.tensor([1.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        if rank == 0:
            ret["out"] = torch.cat(outs).numpy()
            ret["sel"] = torch.cat(sels).numpy()
            ret["tmax"] = float(t)
    finally:
        dist.destroy_process_group()


def test_request_shards_concatenate_to_the_unsharded_step():
    world = 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ret = mp.Manager().dict()
    mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
    from paper_2606_06453_b200.workloads import make_workload
    w = make_workload("C5-small", device="cpu")
    assert w.spec.batch % world == 0
    full = oracle_step(w)
    assert ret["tmax"] == float(world)
    assert np.array_equal(ret["sel"], full["sel_logical"])
    assert np.array_equal(ret["out"], full["out"])


def test_shards_partition_the_batch():
    for batch in (1, 2, 7, 32, 128):
        for world in (1, 2, 4, 8):
            got = [r for k in range(world) for r in shard_requests(batch, k, world)]
            assert got == list(range(batch))
