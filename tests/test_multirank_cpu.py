"""The N>1 path of bench.py (replicas only) on CPU: world_size-2 gloo processes check
the max-over-ranks timing rule, the whole-job aggregate and that replicas differ only in the seed."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench
import gkinputs


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)            # rank 1 is the slow one
        cfg = bench.replica_config(1, rank)
        f = gkinputs.initial_f(cfg, np.complex64)
        out[rank] = (ms, cfg["seed"], float(abs(f).sum()), bench.aggregate_value(4608, 3, world, ms))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_replicas_and_max_over_ranks_gloo_world2():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 15.0                              # max over ranks on both
    assert res[1][1] == res[0][1] + 1 and res[0][2] != res[1][2]       # seeds (and data) differ
    np.testing.assert_allclose(res[0][3], 2 * 4608 * 4 * 3 / 15e-3)    # whole-job aggregate


def test_single_rank_needs_no_process_group():
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.replica_config(3, 0)["name"].startswith("cfg3")
    assert bench.replica_config(5, 0, storage=1)["opts"]["storage"] == 1
