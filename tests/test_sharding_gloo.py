"""N>1 host logic on CPU: world_size-2 (and 3) `gloo` process groups exercise the pose
sharding, the result all-gather and the max-over-ranks timing used by bench.py.  The
per-slice evaluator here is the oracle (tests may call it); on the GPU box it is Scene.eval."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_04310_b200 import sharding, workloads as W


def test_shard_range_partitions():
    for n in (0, 1, 2, 7, 50, 204800, 65536):
        for world in (1, 2, 3, 8):
            r = [sharding.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [e - b for b, e in r]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        sharding.shard_range(5, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_poses, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import psdf_oracle as O
        w = W.make_config(2)
        poses = np.resize(w.poses, (n_poses, 3)).astype(np.float32)
        poses[:, 2] += np.arange(n_poses, dtype=np.float32) * 0.01

        def evaluate(p):
            if p.shape[0] == 0:
                return torch.empty(0, dtype=torch.float64), torch.empty((0, 3), dtype=torch.float64)
            r = O.evaluate(w.footprint, w.A, w.B, w.S, p.numpy())
            return torch.from_numpy(r.value), torch.from_numpy(r.grad)

        v, g = sharding.eval_sharded(evaluate, torch.from_numpy(poses))
        vl, gl, (b, e) = sharding.eval_sharded(evaluate, torch.from_numpy(poses), gather=False)
        tmax = sharding.max_over_ranks([1.0 + rank, 5.0 - rank])
        q.put((rank, v.numpy(), g.numpy(), vl.numpy(), (b, e), tmax))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,n_poses", [(2, 37), (2, 1), (3, 50)])
def test_sharded_eval_matches_unsharded(world, n_poses):
    from oracle import psdf_oracle as O
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_poses, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = W.make_config(2)
    poses = np.resize(w.poses, (n_poses, 3)).astype(np.float32)
    poses[:, 2] += np.arange(n_poses, dtype=np.float32) * 0.01
    ref = O.evaluate(w.footprint, w.A, w.B, w.S, poses)
    for rank, v, g, vl, (b, e), tmax in got:
        assert np.array_equal(v, ref.value) and np.array_equal(g, ref.grad)      # every rank has everything
        assert (b, e) == sharding.shard_range(n_poses, rank, world)
        assert np.array_equal(vl, ref.value[b:e])
        assert tmax == [float(world), 5.0]                                       # max over ranks


def test_max_over_ranks_single_process():
    assert sharding.max_over_ranks(0.25) == [0.25]
