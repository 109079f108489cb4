"""N > 1 path of bench.py on CPU: two gloo ranks, the max-over-ranks timing reduction and the whole-job
throughput (replicas only, no data-path collective)."""
import os
import socket

import pytest


def _worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_2510_02639_b200 import replicas
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, e2e = replicas.max_over_ranks([100.0 + 50.0 * rank, 2.0 - rank])     # rank 1 is slower on the first entry
    dist.barrier()
    q.put((rank, ms, e2e, replicas.aggregate_throughput(1000, world, ms)))
    dist.destroy_process_group()


def test_two_replicas_max_over_ranks():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, e2e, value in out:
        assert ms == 150.0 and e2e == 2.0                    # both ranks see the slowest rank's time
        assert value == pytest.approx(2 * 1000 / 0.150)      # whole-job aggregate of two replicas


def test_single_process_is_identity():
    from paper_2510_02639_b200 import replicas
    assert replicas.max_over_ranks([3.0, 4.5]) == [3.0, 4.5]
    assert replicas.aggregate_throughput(10, 1, 1000.0) == 10.0
