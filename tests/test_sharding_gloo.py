"""N > 1 host logic on CPU: world_size 2, gloo.  The data path has no collective (slices are independent units,
PAPER.md:23); what is exercised is the slice assignment and the timing protocol bench.py uses (max over ranks of
the step time, sum of the hits)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1411_3968_b200 import sharding
from paper_1411_3968_b200 import workload as W


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # every rank generates ITS slice (different seed), as bench.py does
        w = W.make_config(1, time_scale=0.01, seed_offset=sharding.workload_seed_offset(rank, 0, world))
        ms, units = sharding.reduce_timing(1.0 + rank, w.n)
        mine = sharding.my_slices(7, rank, world)
        gathered = [None] * world
        dist.all_gather_object(gathered, (w.n, int(w.hits["t_ps"][:64].sum()), mine))
        if rank == 0:
            out.put((ms, units, gathered))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    ms, units, gathered = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == 2.0  # max over ranks
    assert units == gathered[0][0] + gathered[1][0]  # whole-job hits
    assert gathered[0][1] != gathered[1][1]  # the ranks worked on different slices
    assert sorted(gathered[0][2] + gathered[1][2]) == list(range(7))  # every slice has exactly one owner
    assert gathered[0][2] == [0, 2, 4, 6] and gathered[1][2] == [1, 3, 5]


def _gather_worker(rank: int, world: int, port: int, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r contributes 3 r + 1 records (rank 2 none at all) whose words name their origin
        m = 0 if rank == 2 else 3 * rank + 1
        rec = torch.stack([torch.arange(m, dtype=torch.int64) + 1000 * rank, torch.full((m,), rank, dtype=torch.int64)], dim=1)
        cat, offs = sharding.all_gather_records(rec.reshape(m, 2))
        out.put((rank, cat.tolist(), offs))
    finally:
        dist.destroy_process_group()


def test_all_gather_records_gloo():
    """The one exchange of the by-tower path (NEXT-4): variable-length record lists, concatenated in rank order with
    their offsets, identical on every rank -- world size 3, one rank empty."""
    world = 3
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gather_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    got = [out.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want = [[0, 0]] + [[1000 + k, 1] for k in range(4)]
    for rank, cat, offs in got:
        assert offs == [0, 1, 5, 5] and cat == want, rank


def test_tower_ranges_and_split():
    import numpy as np

    assert sharding.tower_ranges(100, 3) == [(0, 34), (34, 67), (67, 100)]
    assert sharding.tower_ranges(2, 4) == [(0, 1), (1, 2), (2, 2), (2, 2)]
    ro = np.arange(0, 10 * 6 + 1, 10, dtype=np.uint32)  # 3 towers x 2 PMTs, 10 hits per run
    parts = sharding.split_runs_by_tower(ro, 2, 3, 2)
    assert [(a, b) for a, b, _ in parts] == [(0, 40), (40, 60)]
    assert parts[0][2].tolist() == [0, 10, 20, 30, 40] and parts[1][2].tolist() == [0, 10, 20]


def test_single_process_is_identity():
    assert sharding.reduce_timing(3.5, 10) == (3.5, 10)
    assert sharding.my_slices(3, 0, 1) == [0, 1, 2]
