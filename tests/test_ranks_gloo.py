"""The N > 1 path of bench.py on CPU: world_size 2, gloo backend (max-over-ranks time, summed units)."""
import os
import socket

import torch.multiprocessing as mp


def _worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_2509_07175_b200 import ranks
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r processed 1000 units in (10 + 5 r) ms: whole job = 2000 units / 15 ms
    rate, ms = ranks.whole_job_rate(1000.0, 10.0 + 5.0 * rank)
    out.put((rank, rate, ms, len(ranks.shard_of_replicas(7, rank, world))))
    dist.barrier()
    dist.destroy_process_group()


def test_whole_job_rate_two_ranks_gloo():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, rate, ms, n in res:
        assert abs(ms - 15.0) < 1e-12
        assert abs(rate - 2000.0 / 15e-3) < 1e-6
        assert n == 7


def test_whole_job_rate_single_process():
    from paper_2509_07175_b200 import ranks
    rate, ms = ranks.whole_job_rate(500.0, 20.0)
    assert ms == 20.0 and abs(rate - 25000.0) < 1e-9
