"""world_size-2 gloo test of the N > 1 path of bench.py: replicas only, barrier + max-over-ranks timing."""
import os
import socket

import pytest


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2510_09812_b200 import replicas
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    replicas.barrier(dist)
    local_ms = 1000.0 if rank == 0 else 2500.0          # the slow rank sets the job time
    w, max_ms, value = replicas.aggregate(5, local_ms, dist)
    replicas.barrier(dist)
    q.put((rank, w, max_ms, value, replicas.world_info()))
    dist.destroy_process_group()


def test_replica_aggregate_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, w, max_ms, value, info in out:
        assert w == 2 and max_ms == 2500.0
        assert value == pytest.approx(2 * 5 / 2.5)
        assert info == (2, rank, rank)


def test_replica_aggregate_single():
    from paper_2510_09812_b200 import replicas
    assert replicas.aggregate(4, 2000.0) == (1, 2000.0, 2.0)
