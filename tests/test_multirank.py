"""N > 1 path of bench.py on CPU: two gloo ranks, barrier + max-over-ranks timing, rank 0 reports the aggregate
(replicas only: no collective touches the data path)."""
import os
import socket
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = bench.max_over_ranks(10.0 * (rank + 1), world, device="cpu")      # rank r measured 10*(r+1) ms
    val = bench.aggregate_value(events_per_rank=16, steps=5, ms=ms, world=world)
    # replicas only: every rank generates and tracks its OWN batch (here: generates it, and runs its first event
    # through the CPU oracle in place of the tracker -- no GPU on this box -- to show the per-rank work is real)
    seeds = bench.event_seeds("pp", 4, rank)
    evs = bench.make_events("pp", 4, rank)
    import numpy as np
    import oracle
    from paper_1712_09416_b200 import gen
    g = oracle.Geometry(evs[0].n_sectors, gen.row_x().astype(np.float32), gen.TAN_HALF_ANGLE, evs[0].sigma, evs[0].sigma, evs[0].bz)
    n_trk = oracle.track_event(g, evs[0].sector_offset, evs[0].y, evs[0].z, evs[0].row, precision="float").n_tracks
    dist.barrier()
    q.put((rank, ms, val, seeds, [ev.n_clusters for ev in evs], n_trk))
    dist.destroy_process_group()


def test_two_ranks_gloo_max_time_and_aggregate():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val, seeds, ncl, n_trk in res:
        assert ms == pytest.approx(20.0)                      # the slower rank decides
        assert val == pytest.approx(2 * 16 * 5 / 0.020)       # whole-job events/s
        assert len(seeds) == 4 and n_trk > 50
    s0, s1 = set(res[0][3]), set(res[1][3])
    assert not (s0 & s1) and min(s0) == 2000                  # disjoint batches; rank 0 has the single-GPU batch
    assert res[0][4] != res[1][4]                             # different events indeed


def test_single_rank_is_identity():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.max_over_ranks(7.5, 1, device="cpu") == 7.5
    assert bench.aggregate_value(16, 10, 1000.0, 1) == pytest.approx(160.0)
