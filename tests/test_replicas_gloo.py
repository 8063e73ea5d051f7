"""World-size-2 gloo test (CPU) of the N > 1 host logic: replicas only, timing = max over
ranks, work = sum over ranks, no data-path collective."""
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
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2404_19163_b200 import replicas
    r, lr, w = replicas.init("gloo")
    replicas.barrier()
    t, u = replicas.aggregate(10.0 + 5.0 * rank, 3.0)        # rank 1 is slower
    replicas.barrier()
    replicas.shutdown()
    q.put((r, w, t, u))


def test_two_replicas_aggregate_max_time_and_sum_units():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = [q.get(timeout=120) for _ in ps]
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for r, w, t, u in out:
        assert w == 2 and t == 15.0 and u == 6.0


def test_single_process_is_identity():
    from paper_2404_19163_b200 import replicas
    assert replicas.aggregate(7.0, 2.0) == (7.0, 2.0)
