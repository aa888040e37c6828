"""N>1 path on CPU: event sharding + whole-job reduction with torch.distributed (gloo, world_size 2)."""
import os
import sys

import numpy as np
import pytest

from paper_2402_14670_b200 import datagen as dg
from paper_2402_14670_b200 import sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_event_ranges_cover_and_balance():
    b = dg.generate_config(1, n_events=300)
    for world in (1, 2, 3, 8):
        r = sharding.event_ranges(b.seed_offsets, world)
        assert r[0][0] == 0 and r[-1][1] == b.n_events
        assert all(r[i][1] == r[i + 1][0] for i in range(world - 1))
        seeds = [int(b.seed_offsets[e1]) - int(b.seed_offsets[e0]) for e0, e1 in r]
        assert sum(seeds) == b.n_seeds
        assert max(seeds) - min(seeds) <= 2 * 260   # within about one event of seeds
    # degenerate: more ranks than events, and an empty batch
    assert sharding.event_ranges(np.array([0, 5, 9], np.uint32), 4)[-1][1] == 2
    assert sharding.event_ranges(np.array([0], np.uint32), 2) == [(0, 0), (0, 0)]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    sys.path.insert(0, ROOT)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import lf_oracle  # CPU stand-in for the per-rank compute in this *test* only
    b = dg.generate_config(1, n_events=40)
    e0, e1 = sharding.event_ranges(b.seed_offsets, world)[rank]
    sub = b.slice_events(e0, e1)
    r = lf_oracle.run(dg.toy_geometry(), dg.default_params(), sub)
    ms, counts = sharding.reduce_job(10.0 * (rank + 1), [sub.n_events, sub.n_seeds, r.n_tracks])
    assert sharding.dist_env() == (rank, rank, world)
    q.put((rank, ms, counts, r.n_tracks))
    dist.barrier()
    dist.destroy_process_group()


def test_gloo_world2_sharded_job_equals_single_process():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    from oracle import lf_oracle
    b = dg.generate_config(1, n_events=40)
    full = lf_oracle.run(dg.toy_geometry(), dg.default_params(), b)
    for rank, ms, counts, _ in res:
        assert ms == 20.0                                  # max over ranks of the device time
        assert counts == [float(b.n_events), float(b.n_seeds), float(full.n_tracks)]   # sums over ranks
    assert res[0][3] + res[1][3] == full.n_tracks          # shards are independent: no exchange step
