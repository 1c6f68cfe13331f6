"""N > 1 launch logic of bench.py on CPU: 2 ranks, gloo backend (the path is "replicas only",
DESIGN.md S6: no data-path collective; only the timing is reduced with MAX over ranks)."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    ms = bench.max_over_ranks(local_ms, dist, torch.device("cpu"))
    value = bench.whole_job_value(world, 4, 10, ms)
    dist.barrier()
    out[rank] = (ms, value)
    dist.destroy_process_group()


def test_two_rank_replica_aggregation():
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    world = 2
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0] == res[1]                                    # every rank sees the max
    ms, value = res[0]
    assert ms == 15.0
    assert value == pytest.approx(2 * 4 * 10 / 15e-3)         # all ranks' samples / slowest rank


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, None) == 3.5
    assert bench.whole_job_value(1, 4, 20, 20.0) == pytest.approx(4000.0)
    w = bench.layer_work(4, 90, 180, 768, 8, 90 * 91)
    assert w["bytes"] == 5 * 4 * 90 * 180 * 768 * 2 + 3 * 2 * (8 * 96 * 96 * 2 + 768 * 2) * 4
    assert w["flops_model"] == 6 * 2 * 192 * 192 * 8 * 8190 * 4
