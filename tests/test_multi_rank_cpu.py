"""World-size-2 gloo test of the N > 1 host path: word-column
shards + count gather + max-over-ranks timing.  The compute stand-in on CPU is
the oracle with a word subset (tests may use it; the product path cannot run
without a GPU) - what is under test is the sharding / gathering logic, which is
the same code bench.py and a multi-GPU user call."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp

import workloads as wl


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, W, q):
    import torch.distributed as dist

    import oracle
    from paper_1301_6082_b200 import shard

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w0, w1 = shard.shard_words(W, world, rank)
    o = oracle.Oracle(256, 64 * W, 0.3, 0.12, 17, wl.PCPD, Ts=128, D=32, A=4, words=list(range(w0, w1)))
    o.init(wl.INIT_BERNOULLI)
    o.run(3)
    allc = shard.gather_counts(o.counts(), W)
    tmax = shard.max_over_ranks(10.0 + rank)
    dist.barrier()
    if rank == 0:
        q.put((allc, tmax))
    dist.destroy_process_group()


def test_two_rank_shards_equal_single_run():
    import oracle

    W, world = 5, 2  # ragged: 3 + 2 columns
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, W, q)) for r in range(world)]
    for p in procs:
        p.start()
    allc, tmax = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ref = oracle.Oracle(256, 64 * W, 0.3, 0.12, 17, wl.PCPD, Ts=128, D=32, A=4)
    ref.init(wl.INIT_BERNOULLI)
    ref.run(3)
    assert np.array_equal(allc, ref.counts())
    assert tmax == 11.0


def test_shard_words_partition():
    from paper_1301_6082_b200 import shard

    for W in (1, 5, 32, 33):
        for world in (1, 2, 3, 8):
            cols = []
            for r in range(world):
                a, b = shard.shard_words(W, world, r)
                cols += list(range(a, b))
            assert cols == list(range(W))
