"""world_size-2 gloo test of the multi-GPU plumbing (CPU): band shards are disjoint and cover the
block, the step time is the max over ranks, and per-rank inputs are distinct but reproducible."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import torch.distributed as dist
    import synth
    from paper_2507_08578_b200 import sharding
    sharding.init("gloo")
    assert sharding.active()
    sharding.barrier()
    mx = sharding.max_over_ranks(10.0 + rank)
    b0, b1 = sharding.band_shard(1025, rank, world)
    got = [None] * world
    dist.all_gather_object(got, (b0, b1))
    # strong-scaling style check: a rank's shard of a seeded block equals the same bands of the full block
    cfg = synth.make_config("c0", with_vloc=False)
    kin = [np.linspace(0.0, 8.0, 50)]
    full = synth.gen_psi(cfg, kin, nband=8)
    s0, s1 = sharding.band_shard(8, rank, world)
    mine = synth.gen_psi(cfg, kin, bands=range(s0, s1))
    ok = bool(np.array_equal(mine, full[:, s0:s1]))
    q.put((rank, mx, got, ok))
    sharding.shutdown()


def test_two_ranks_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, mx, got, ok in res:
        assert mx == 11.0 and ok
        assert got == [(0, 513), (513, 1025)]


def test_band_shard_properties():
    sys.path.insert(0, ROOT)
    from paper_2507_08578_b200 import sharding
    for n in (0, 1, 7, 1024, 1025):
        for w in (1, 2, 3, 8):
            parts = [sharding.band_shard(n, r, w) for r in range(w)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[i][1] == parts[i + 1][0] for i in range(w - 1))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1
