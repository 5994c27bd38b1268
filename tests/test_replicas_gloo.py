"""The N > 1 path is N independent replicas; its only cross-rank logic (barrier, sum of units, max of
times) is covered here with world_size 2 over gloo on the CPU."""
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
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1907_02290_b200 import replicas
    r, w, _ = replicas.init_from_env("gloo")
    replicas.barrier(w)
    units, ms = replicas.reduce_timing(100.0 * (rank + 1), 10.0 + 5.0 * rank, w)
    q.put((r, w, units, ms))
    import torch.distributed as dist
    dist.destroy_process_group()


def test_two_replicas_reduce_sum_and_max():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[0] for g in got] == [0, 1]
    for _, w, units, ms in got:
        assert w == 2 and units == 300.0 and ms == 15.0


def test_single_process_is_identity():
    from paper_1907_02290_b200 import replicas
    assert replicas.reduce_timing(7.0, 3.0, 1) == (7.0, 3.0)
