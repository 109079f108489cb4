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


def _run_bench(argv, env_extra=None, timeout=300):
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    env.update(env_extra or {})
    return subprocess.run([sys.executable, os.path.join(root, "bench.py")] + argv, env=env, capture_output=True, text=True,
                          timeout=timeout)


def test_bench_gpus_flag_spawns_the_ranks_and_takes_the_max():
    """`python bench.py --gpus 2` outside a launcher starts two ranks itself (torch.distributed.run, 127.0.0.1) and the
    line carries n_gpus = 2, the SLOWEST rank's step time and the whole-job aggregate. --stub swaps the CUDA step for a
    sleep (rank r sleeps (r + 1) x 20 ms per step) so that the plumbing runs on CPU ranks over gloo."""
    import json
    p = _run_bench(["--gpus", "2", "--steps", "3", "--stub"])
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [ln for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                   # rank 0 alone prints
    out = json.loads(lines[0])
    assert out["stub"] is True and out["n_gpus"] == 2 and out["steps"] == 3
    assert out["ms_per_step"] >= 39.0 and out["ms_per_step_rank0"] < 35.0      # max over ranks, not rank 0's own time
    assert out["value"] == pytest.approx(2 * 1000 / (out["ms_per_step"] * 1e-3))


def test_bench_refuses_a_replica_count_that_is_not_the_world_size():
    p = _run_bench(["--gpus", "2", "--steps", "1", "--stub"], {"WORLD_SIZE": "1", "RANK": "0", "LOCAL_RANK": "0"})
    assert p.returncode != 0 and "WORLD_SIZE=1" in p.stderr
