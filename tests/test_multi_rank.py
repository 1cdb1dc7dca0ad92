"""N > 1 is "replicas only": channel ranges per rank, no data-path collective.
World-size-2 gloo test on CPU of the host-side logic bench.py uses (barrier, max over ranks, channel split)."""
import os
import socket

import numpy as np
import pytest

import oracle
import workloads as wl
from paper_1503_06189_b200 import replicas

torch = pytest.importorskip("torch")


def test_channel_ranges_partition():
    for f in (1, 7, 64, 1024):
        for w in (1, 2, 3, 8):
            r = replicas.channel_ranges(f, w)
            assert r[0][0] == 0 and r[-1][1] == f and all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [e - b for b, e in r]
            assert max(sizes) - min(sizes) <= 1
    assert replicas.whole_job_rate(10.0, 4, 2.0) == 20.0
    assert replicas.max_over_ranks(3.5) == 3.5


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        fr = wl.uniform_frame(16, 6, 64, seed=3)            # every rank generates the same seeded frame
        b, e = replicas.channel_ranges(6, world)[rank]
        mine = oracle.planar(np.ascontiguousarray(fr[:, b:e, :]))  # a replica works on its own channels only
        dist.barrier()
        t = replicas.max_over_ranks(1.0 + rank, dist)        # slowest rank's time
        q.put((rank, b, e, mine, t))
    finally:
        dist.destroy_process_group()


def test_two_replicas_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in procs], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    full = oracle.planar(wl.uniform_frame(16, 6, 64, seed=3))
    cat = np.concatenate([r[3] for r in res], axis=0)        # results concatenate along f, no exchange needed
    assert np.array_equal(cat, full)
    assert all(r[4] == 2.0 for r in res)                     # max over ranks of (1.0, 2.0)
    assert replicas.whole_job_rate(3.0, 2, res[0][4]) == 3.0
