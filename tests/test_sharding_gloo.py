"""N>1 host logic of bench.py on CPU: world_size 2 over gloo ("replicas only").

Events are independent units, so ranks shard by event seed with no data-path
collective.  Checked here: the per-rank seed sets are disjoint and cover 1..world*n; the
max-over-ranks timing reduction; and that a rank's events, processed alone by the oracle, are
exactly what a single process gets for the same seeds (the "subset" metamorphic check of
SURVEY.md section 8(c) at event granularity).
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

N_PER_RANK = 3
N_FEDS = 4


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_summary(rank: int, world: int):
    """What one rank computes for its shard: (seed, n_clusters, sum of charges) per event."""
    import bench
    from oracle import sst_oracle
    from paper_2101_11489_b200 import synth
    sst_oracle.build()
    cfg = synth.CONFIGS[3]
    calib = synth.make_calibration(N_FEDS, cfg.bad_frac)
    seeds = bench.event_seeds_for_rank(rank, world, N_PER_RANK)
    events = bench.generate_events(3, N_FEDS, seeds, calib, workers=1)
    rows = []
    for seed, (raw, fo, _meta) in zip(seeds, events):
        r = sst_oracle.run(raw, fo, N_FEDS, calib.gain, calib.noise, calib.bad, calib.chan_module,
                           (2.0, 3.0, 5.0))
        rows.append((seed, int(r.n_clusters), int(np.asarray(r.cl_charge, np.int64).sum())))
    return rows


def _worker(rank: int, world: int, port: int, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        rows = _rank_summary(rank, world)
        # timing reduction used by bench.py: max over ranks
        t = bench.max_over_ranks(10.0 + rank)
        gathered = [None] * world
        dist.all_gather_object(gathered, rows)
        dist.barrier()
        if rank == 0:
            q.put((t, gathered))
    finally:
        dist.destroy_process_group()


def test_seed_shards_are_disjoint_and_cover():
    import bench
    for world in (1, 2, 4, 8):
        seen = []
        for r in range(world):
            seen += bench.event_seeds_for_rank(r, world, 64)
        assert sorted(seen) == list(range(1, 64 * world + 1))


@pytest.mark.timeout(300)
def test_two_ranks_gloo_match_single_process():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    t, gathered = q.get(timeout=240)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert t == 11.0  # max over ranks of 10 + rank
    got = [row for rows in gathered for row in rows]
    assert [g[0] for g in got] == list(range(1, world * N_PER_RANK + 1))
    # single process, same seeds, world = 1
    want = []
    for r in range(world):
        want += _rank_summary(r, world)
    assert got == want
    assert all(n > 0 for _, n, _ in got)
