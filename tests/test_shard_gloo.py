"""N > 1 host logic on CPU: two gloo ranks take disjoint windows of the request stream and agree on the MAX of their
times / SUM of their request counts (what bench.py reports at --gpus N).  No GPU, no oracle."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1412_5989_b200 import shard, workloads as W


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard.rank_window(rank, world, n)
    cfg = W.make_config(0)                       # tiny: all-pairs stream, windows wrap around it like bench.py
    allreq = cfg.requests()
    idx = np.arange(lo, hi) % len(allreq)
    mine = allreq[idx]
    t = shard.max_over_ranks(1.0 + rank)          # pretend rank r took (1 + r) ms
    total = shard.sum_over_ranks(float(len(mine)))
    q.put((rank, lo, hi, t, total, int(mine[:, 0].sum())))
    dist.destroy_process_group()


def test_two_rank_windows_and_reductions():
    world, n = 2, 5000
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, t0, tot0, _), (r1, lo1, hi1, t1, tot1, _) = res
    assert (lo0, hi0, lo1, hi1) == (0, n, n, 2 * n)            # disjoint, consecutive windows
    assert t0 == t1 == 2.0                                      # MAX over ranks, same on every rank
    assert tot0 == tot1 == 2.0 * n                              # whole-job request count


def test_single_process_is_identity():
    assert shard.max_over_ranks(3.5) == 3.5 and shard.sum_over_ranks(2.0) == 2.0
    assert shard.rank_window(3, 8, 100) == (300, 400)
    with pytest.raises(ValueError):
        shard.rank_window(2, 2, 10)
