"""N > 1 path of bench.py (replicas only) on CPU: world_size 2, gloo backend."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1812_07993_b200 import inputs as I
from paper_1812_07993_b200 import replicas as R


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    assert R.dist_env() == (rank, rank, world)
    units, secs = 1000.0 * (rank + 1), 0.5 + 0.25 * rank          # rank 1 is slower and did more work
    value, t = R.job_throughput(units, secs)
    seed = R.replica_seed(I.BASE_SEED + 2, rank)
    gathered = [None] * world
    dist.all_gather_object(gathered, seed)
    dist.barrier()
    if rank == 0:
        out.put((value, t, gathered))
    dist.destroy_process_group()


def test_two_rank_aggregate_is_sum_of_units_over_slowest_rank():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    value, t, seeds = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert t == 0.75 and abs(value - 3000.0 / 0.75) < 1e-9
    assert len(set(seeds)) == 2 and seeds[0] == I.BASE_SEED + 2


def test_replicas_are_distinct_and_single_rank_is_identity():
    a = I.cylinder_config(512, R.replica_seed(11, 0), "a", box=22.0, length=4)
    b = I.cylinder_config(512, R.replica_seed(11, 1), "b", box=22.0, length=4)
    assert a["pos"].shape == b["pos"].shape and not np.array_equal(a["pos"], b["pos"])
    assert np.array_equal(a["wall"], b["wall"])                   # same pore, different gas
    assert R.job_throughput(10.0, 2.0) == (5.0, 2.0)              # no process group: identity
