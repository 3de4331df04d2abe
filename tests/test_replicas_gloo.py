"""World-size-2 gloo test of the N>1 plumbing bench.py uses (replicas only: a barrier, a max and a
sum over ranks; no data-path collective)."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2210_13641_b200 import replicas
    r, lr, w = replicas.init_from_env(backend="gloo")
    assert (r, lr, w) == (rank, rank, world)
    replicas.barrier()
    # rank 0 processed 1000 units in 2 s, rank 1 3000 units in 4 s -> 4000 / 4 s
    value, total, t = replicas.aggregate_throughput(1000.0 * (1 + 2 * rank), 2.0 * (1 + rank))
    q.put((rank, value, total, t, replicas.max_over_ranks(rank), replicas.sum_over_ranks(rank + 1)))
    replicas.barrier()
    replicas.shutdown()


def test_replica_aggregation_world_size_2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, value, total, t, mx, sm in out:
        assert (value, total, t, mx, sm) == (1000.0, 4000.0, 4.0, 1.0, 3.0)


def test_single_process_is_identity():
    from paper_2210_13641_b200 import replicas
    assert replicas.aggregate_throughput(500.0, 2.0) == (250.0, 500.0, 2.0)
    replicas.barrier()
