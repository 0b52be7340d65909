"""bench.py's multi-process plumbing on CPU: world_size-2 gloo (replicas only; the only
collectives are the two all-reduces that aggregate units and time)."""
import os
import socket
import sys

import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import bench
    r, w, lr = bench.dist_init(world, backend="gloo")
    assert (r, w, lr) == (rank, world, rank)
    bench.barrier()
    units, ms = bench.aggregate(1000.0 * (rank + 1), 5.0 + 2.0 * rank, device="cpu")
    q.put((rank, units, ms, bench.shard_range(4096, rank, world)))
    import torch.distributed as dist
    dist.destroy_process_group()


def test_aggregate_world2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, units, ms, _ in res:
        assert units == 3000.0 and ms == 7.0          # sum of units, max of time, identical on every rank
    assert res[0][3] == (0, 2048) and res[1][3] == (2048, 4096)


def test_shard_range_covers_everything():
    sys.path.insert(0, ROOT)
    import bench
    for n in (0, 1, 7, 4096, 4099):
        for world in (1, 2, 3, 8):
            parts = [bench.shard_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1


def test_replica_seeds_differ():
    sys.path.insert(0, ROOT)
    import numpy as np
    import bench
    a = bench.make_workload("C2-f64", 0)
    b = bench.make_workload("C2-f64", 1)
    assert a.tnfw.shape == b.tnfw.shape and not np.array_equal(a.tnfw, b.tnfw)
