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
    out.put((rank, rate, ms, 7))
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


def _shard_worker(rank, world, port, out):
    """Each rank runs the ORACLE on its block of simplices (the CUDA path needs a GPU; the exchange step does
    not), then the ranks combine partial cells exactly as bench.py --gpus N does."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from oracle import oracle
    from paper_2509_07175_b200 import inputs, ranks
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = inputs.config(2, "small")
    b, e = ranks.simplex_block(w.m, rank, world)
    part = oracle.compute(w.sites, w.verts, w.simplices[b:e], w.kind)
    # what vd_partial_moments / vd_finish_centroids do on the device, written out for the oracle's partial cells
    packed = torch.from_numpy(np.concatenate([part.measure[:, None], part.measure[:, None] * part.centroid], axis=1))
    ranks.all_reduce_sums(packed)
    s = packed.numpy()
    m = s[:, 0].copy()
    c = np.where(m[:, None] > 0, s[:, 1:] / np.where(m > 0, m, 1.0)[:, None], w.sites)
    out.put((rank, b, e, m, c))
    dist.barrier()
    dist.destroy_process_group()


def test_simplex_blocks_cover_and_balance():
    from paper_2509_07175_b200 import ranks
    for m, world in [(48000, 8), (7, 3), (2, 4), (1, 1)]:
        blocks = [ranks.simplex_block(m, r, world) for r in range(world)]
        assert blocks[0][0] == 0 and blocks[-1][1] == m
        assert all(blocks[k][1] == blocks[k + 1][0] for k in range(world - 1))
        sizes = [e - b for b, e in blocks]
        assert max(sizes) - min(sizes) <= 1


def test_sharded_cells_combine_to_the_whole_two_ranks_gloo():
    import numpy as np
    from oracle import oracle
    from paper_2509_07175_b200 import inputs
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=300) for _ in range(2)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = inputs.config(2, "small")
    whole = oracle.compute(w.sites, w.verts, w.simplices, w.kind)
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == w.m
    for _, _, _, m, c in res:      # every rank ends with the whole diagram's measures and centroids
        assert np.abs(m - whole.measure).max() <= 1e-12 * whole.measure.max()
        assert np.abs(c - whole.centroid).max() <= 1e-9
        assert abs(m.sum() - w.measure) <= 1e-12 * w.measure


def test_balanced_blocks_follow_the_pairs():
    """Work-balanced blocks on the clustered replica: contiguous, covering, and closer to equal PAIRS
    (counted by the oracle: pieces per simplex) than equal-count blocks are."""
    import numpy as np
    from oracle import oracle
    from paper_2509_07175_b200 import inputs, ranks
    w = inputs.config(3, "small")
    world = 4
    blocks = ranks.simplex_blocks_balanced(w.sites, w.verts, w.simplices, world)
    assert blocks[0][0] == 0 and blocks[-1][1] == w.m and all(blocks[k][1] == blocks[k + 1][0] for k in range(world - 1))
    assert blocks == ranks.simplex_blocks_balanced(w.sites, w.verts, w.simplices, world)      # deterministic
    o = oracle.compute(w.sites, w.verts, w.simplices, w.kind)
    per_simplex = np.bincount(o.piece_simplex, minlength=w.m)
    bal = [per_simplex[b:e].sum() for b, e in blocks]
    eq = [per_simplex[slice(*ranks.simplex_block(w.m, r, world))].sum() for r in range(world)]
    assert sum(bal) == sum(eq) == len(o.piece_simplex)
    assert max(bal) < max(eq), (bal, eq)
    assert max(bal) <= 1.5 * sum(bal) / world, bal
