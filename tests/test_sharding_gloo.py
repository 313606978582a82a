"""N > 1 host logic on CPU: world_size-2 gloo run of the point-range sharding and the timing reductions
that bench.py uses under torchrun (no data-path collective exists)."""
import os
import socket

import numpy as np
import pytest


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, q):
    import torch.distributed as dist

    from paper_2510_05282_b200 import dist as shd
    from paper_2510_05282_b200 import inputs

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert shd.env_world() == (rank, rank, world)
        b, e = inputs.shard_range(n, rank, world)
        pts = inputs.config1_cube()[:n]
        local = pts[b:e]
        # every rank works on its own slice only; the reductions below are bookkeeping, not data path
        total_pts = shd.sum_over_ranks(len(local))
        checksum = shd.sum_over_ranks(float(local.sum()))
        slowest = shd.max_over_ranks(10.0 + rank)
        dist.barrier()
        q.put((rank, b, e, total_pts, checksum, slowest, float(pts.sum())))
    finally:
        dist.destroy_process_group()


def test_shard_range_partitions():
    from paper_2510_05282_b200 import inputs

    for n in (0, 1, 7, 10008, 2**21 + 3):
        for world in (1, 2, 3, 8):
            r = [inputs.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [e - b for b, e in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        inputs.shard_range(10, 2, 2)


def test_two_rank_gloo_sharding():
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port, n, world = _free_port(), 10007, 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, b0, e0, tot0, cs0, slow0, full), (_, b1, e1, tot1, cs1, slow1, _) = res
    assert (b0, e1) == (0, n) and e0 == b1 and abs((e0 - b0) - (e1 - b1)) <= 1
    assert tot0 == tot1 == n
    assert np.isclose(cs0, full) and np.isclose(cs1, full)
    assert slow0 == slow1 == 11.0
