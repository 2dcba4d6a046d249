"""N > 1 path of bench.py ("replicas only") on CPU: world_size-2 gloo processes,
the timing reduction is the max over ranks and the throughput the whole-job aggregate."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    from paper_2603_07038_b200.replicas import aggregate_throughput, max_over_ranks
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = 2.0 + 3.0 * rank                      # rank 1 is the slow replica: 5 ms
        ms = max_over_ranks(mine, dist)
        value = aggregate_throughput(1000.0, ms * 1e-3, world)
        dist.barrier()
        torch.save({"ms": ms, "value": value}, os.path.join(out, "r%d.pt" % rank))
    finally:
        dist.destroy_process_group()


def test_replicas_world2_gloo(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    for r in range(world):
        res = torch.load(os.path.join(str(tmp_path), "r%d.pt" % r))
        assert res["ms"] == 5.0                                   # max over ranks on every rank
        assert res["value"] == pytest.approx(2 * 1000.0 / 5e-3)   # units of ALL ranks / max time


def test_single_process_is_identity():
    from paper_2603_07038_b200.replicas import aggregate_throughput, max_over_ranks
    assert max_over_ranks(1.25, None) == 1.25
    assert aggregate_throughput(10.0, 2.0, 1) == 5.0
    with pytest.raises(ValueError):
        aggregate_throughput(10.0, 0.0, 1)
