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


# ---- sharding logic (paper_2208_05419_b200/sharding.py) on 2 gloo ranks --------------------------
# The compute here is the ORACLE (test infrastructure): what is tested is the host logic of the product's sharding
# module (sample / block ranges, the flat gradient bucket and its single all-reduce) against the unsharded result.

def _small_problem():
    import numpy as np
    rng = np.random.default_rng(7)
    B, H, W, C, nb = 3, 6, 10, 16, 4     # B = 3 over 2 ranks: an uneven split
    bs = C // nb
    x = rng.standard_normal((B, H, W, C))
    dy = rng.standard_normal((B, H, W, C))
    w1, b1, w2, b2 = [0.2 * rng.standard_normal(s) for s in [(nb, bs, bs, 2), (nb, bs, 2), (nb, bs, bs, 2), (nb, bs, 2)]]
    return (B, H, W, C, nb), x, dy, (w1, b1, w2, b2)


def _shard_worker(rank, world, port, out):
    import numpy as np
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from oracle import afno_oracle
    from paper_2208_05419_b200 import sharding
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    (B, H, W, C, nb), x, dy, params = _small_problem()
    bs = C // nb
    # --- data parallel: local samples, gradients into the flat bucket, ONE all-reduce(SUM) ---
    b0, n = sharding.shard_batch(B, rank, world)
    cfg = afno_oracle.Config(n, H, W, C, nb, lam=0.05, kept_fraction=1.0)
    g = afno_oracle.backward(cfg, x[b0:b0 + n], dy[b0:b0 + n], *params)
    bucket = sharding.GradBucket.allocate(nb, bs, 1, device="cpu")
    for v, k in zip(bucket.views, ("dw1", "db1", "dw2", "db2")):
        v.copy_(torch.from_numpy(np.asarray(g[k], dtype=np.float32)))
    views = bucket.all_reduce(dist)
    dp = {k: v.numpy().copy() for v, k in zip(views, ("dw1", "db1", "dw2", "db2"))}
    dp["dx"] = np.asarray(g["dx"]), (b0, n)
    # --- block (feature) parallel: own blocks only, no collective ---
    j0, nj, c0, nc = sharding.shard_blocks(nb, C, rank, world)
    cfg_b = afno_oracle.Config(B, H, W, nc, nj, lam=0.05, kept_fraction=1.0)
    pl = sharding.slice_params_for_blocks(params, j0, nj)
    y_l = afno_oracle.forward(cfg_b, np.ascontiguousarray(x[..., c0:c0 + nc]), *pl)
    g_l = afno_oracle.backward(cfg_b, np.ascontiguousarray(x[..., c0:c0 + nc]), np.ascontiguousarray(dy[..., c0:c0 + nc]), *pl)
    dist.barrier()
    out[rank] = dict(dp=dp, blocks=dict(j0=j0, nj=nj, c0=c0, nc=nc, y=np.asarray(y_l),
                                        g={k: np.asarray(g_l[k]) for k in ("dx", "dw1", "db1", "dw2", "db2")}))
    dist.destroy_process_group()


def test_two_rank_sharding_matches_unsharded_oracle(oracle):
    import numpy as np
    torch = pytest.importorskip("torch")
    import torch.multiprocessing as mp
    world = 2
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_shard_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    (B, H, W, C, nb), x, dy, params = _small_problem()
    cfg = oracle.Config(B, H, W, C, nb, lam=0.05, kept_fraction=1.0)
    full = oracle.backward(cfg, x, dy, *params)
    y_full = oracle.forward(cfg, x, *params)
    for r in range(world):
        # data parallel: every rank holds the batch-summed gradients after the all-reduce (fp32 bucket)
        for k in ("dw1", "db1", "dw2", "db2"):
            ref = np.asarray(full[k])
            assert np.allclose(res[r]["dp"][k], ref, rtol=0, atol=2e-6 * np.abs(ref).max()), (r, k)
        dx, (b0, n) = res[r]["dp"]["dx"]
        assert np.allclose(dx, np.asarray(full["dx"])[b0:b0 + n], rtol=0, atol=1e-12)
        # block parallel: the rank's channel slice of y and dx and its blocks' gradients, no communication
        blk = res[r]["blocks"]
        c0, nc, j0, nj = blk["c0"], blk["nc"], blk["j0"], blk["nj"]
        assert np.allclose(blk["y"], np.asarray(y_full)[..., c0:c0 + nc], rtol=0, atol=1e-12)
        assert np.allclose(blk["g"]["dx"], np.asarray(full["dx"])[..., c0:c0 + nc], rtol=0, atol=1e-12)
        for k in ("dw1", "db1", "dw2", "db2"):
            assert np.allclose(blk["g"][k], np.asarray(full[k])[j0:j0 + nj], rtol=0, atol=1e-12), (r, k)
    # the two ranks' shards tile the batch and the blocks exactly
    assert sorted(res[r]["dp"]["dx"][1] for r in range(world)) == [(0, 2), (2, 1)]
    assert sorted((res[r]["blocks"]["j0"], res[r]["blocks"]["nj"]) for r in range(world)) == [(0, 2), (2, 2)]


def test_split_range_and_bucket_layout():
    sys.path.insert(0, ROOT)
    from paper_2208_05419_b200 import sharding
    for n in (1, 4, 7, 32):
        for world in (1, 2, 3, 8):
            parts = [sharding.split_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and sum(c for _, c in parts) == n
            assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(world - 1))
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
    with pytest.raises(ValueError):
        sharding.split_range(4, 2, 2)
    assert sharding.shard_blocks(8, 768, 3, 8) == (3, 1, 288, 96)
    offs, total = sharding.GradBucket.offsets(sharding.param_shapes(8, 96))
    assert all(o % 4 == 0 for o, _ in offs)                      # 16-byte aligned views (C ABI)
    assert total * 4 == 2 * (8 * 96 * 96 * 2 + 8 * 96 * 2) * 4   # 1.19 MB per step at 768 channels
