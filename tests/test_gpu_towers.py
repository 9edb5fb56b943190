"""NEXT-4: the trigger of a multi-tower detector sharded BY TOWER with one exchange
of L1 hits.  The ranks are emulated one after the other on the one GPU of the test box (no kernel waits on another
rank); the exchange itself (all_gather_records) is covered on CPU with gloo in test_sharding_gloo.py.  What every rank
ends up with must be, hit for hit, what the oracle computes on the WHOLE detector."""
import numpy as np
import pytest
import torch

from paper_1411_3968_b200 import sharding
from paper_1411_3968_b200 import workload as W
from util import oracle_chain

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1411_3968_b200 import binding

    binding.load()
    return binding


def _run_sharded(B, w, world, prm, geo):
    g = w.geometry
    parts = sharding.split_runs_by_tower(w.run_offsets, g.pmts_per_tower, g.n_tower, world)
    states = [sharding.tower_local(B, r, np.ascontiguousarray(w.hits[a:b]), ro, prm) for r, (a, b, ro) in enumerate(parts)]
    gathered = torch.cat([s["l1"] for s in states], dim=0)  # what all_gather_records returns on every rank
    offs = [0]
    for s in states:
        offs.append(offs[-1] + int(s["l1"].shape[0]))
    return [sharding.tower_global(B, s, gathered, offs, geo, prm) for s in states]


@pytest.mark.parametrize("world", [1, 2, 3, 7])
@pytest.mark.parametrize("mode", [0, 1])
def test_by_tower_equals_whole_detector(world, mode, B, oracle_lib):
    w = W.make_config(4, time_scale=0.002)  # 100 towers, 0.4 ms: ~185 k hits, tracks crossing several towers
    p, g = w.params, w.geometry
    p.l2_mode = mode
    o = oracle_chain(w.hits, w.seg_offsets, g, p)
    assert len(o["seeds"]) > 0 and len(o["events"]) > 0
    geo = B.Geometry(g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks)
    prm = B.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps)
    res = _run_sharded(B, w, world, prm, geo)
    tower = o["sorted"]["pmt_id"].astype(np.int64) // g.pmts_per_tower
    cross = 0
    for r, (lo, hi) in enumerate(sharding.tower_ranges(g.n_tower, world)):
        mine = (tower >= lo) & (tower < hi)  # the rank's hits, in the global sorted order = its own sorted order
        rr = res[r]
        assert rr["status"] == 0
        assert rr["sorted"].tobytes() == o["sorted"][mine].tobytes(), f"rank {r}: sorted records"
        bad = np.nonzero(rr["flags"] != o["flags"][mine])[0]
        assert len(bad) == 0, (r, len(bad), bad[:8], rr["flags"][bad[:8]], o["flags"][mine][bad[:8]])
        assert (rr["seeds"] == np.nonzero(o["flags"][mine] & 16)[0]).all(), f"rank {r}: seeds"
        assert rr["n_global_seeds"] == len(o["seeds"])
        assert len(rr["events"]) == len(o["events"])
        for f in ("t_start", "t_end", "seed_begin", "n_seeds"):
            assert (rr["events"][f] == o["events"][f]).all(), (r, f)
        cross += int(((o["flags"][mine] & 16) != 0).sum())
    assert cross == len(o["seeds"])  # every global seed belongs to exactly one rank
    geo.close()


def test_eight_towers_one_gpu_per_tower(B, oracle_lib):
    """The paper's own layout (Fig. 4): 8 towers, one TGPU each -- 8 ranks of one tower (emulated)."""
    w = W.make_config(5, time_scale=0.05)  # 8 towers, 10 ms: ~370 k hits
    p, g = w.params, w.geometry
    assert g.n_tower == 8
    o = oracle_chain(w.hits, w.seg_offsets, g, p)
    assert len(o["seeds"]) > 0
    geo = B.Geometry(g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks)
    prm = B.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps)
    res = _run_sharded(B, w, 8, prm, geo)
    tower = o["sorted"]["pmt_id"].astype(np.int64) // g.pmts_per_tower
    for r in range(8):
        mine = tower == r
        assert res[r]["status"] == 0 and (res[r]["flags"] == o["flags"][mine]).all(), r
        assert (res[r]["seeds"] == np.nonzero(o["flags"][mine] & 16)[0]).all(), r
        assert (res[r]["events"]["t_start"] == o["events"]["t_start"]).all() and (res[r]["events"]["t_end"] == o["events"]["t_end"]).all()
    geo.close()


def test_by_tower_needs_the_exchange(B, oracle_lib):
    """The exchange is not decoration: a track that crosses towers meets the multiplicity only with the L1 hits of the
    neighbouring towers -- without them (every rank alone) seeds are lost."""
    w = W.make_config(4, time_scale=0.002)
    p, g = w.params, w.geometry
    o = oracle_chain(w.hits, w.seg_offsets, g, p)
    parts = sharding.split_runs_by_tower(w.run_offsets, g.pmts_per_tower, g.n_tower, 4)
    alone = 0
    for a, b, ro in parts:
        h = np.ascontiguousarray(w.hits[a:b])
        oo = oracle_chain(h, np.array([0, len(h)], dtype=np.uint32), g, p)
        alone += len(oo["seeds"])
    assert alone < len(o["seeds"])


def test_l1_export_overflow_and_empty(B, oracle_lib):
    w = W.make_config(1, time_scale=0.02)
    p = w.params
    prm = B.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps)
    st = sharding.tower_local(B, 5, w.hits, w.run_offsets, prm)
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, p)
    l1 = st["l1"].cpu().numpy().reshape(-1).view(B.L1HIT_DTYPE)
    want = np.nonzero(o["flags"] & 4)[0]
    assert (l1["idx"] == want).all() and (l1["src"] == 5).all()
    assert (l1["t_ps"] == o["sorted"]["t_ps"][want]).all() and (l1["pmt_id"] == o["sorted"]["pmt_id"][want]).all()
    # capacity too small: true count, prefix valid, status bit
    d_l1 = torch.zeros((3, 2), dtype=torch.int64, device="cuda")
    d_m = torch.zeros(1, dtype=torch.int32, device="cuda")
    d_st = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.tt_l1_export(st["d_sorted"], st["d_flags"], 5, d_l1, d_m, d_st)
    torch.cuda.synchronize()
    assert int(d_m.item()) == len(want) and int(d_st.item()) == B.TT_S_L1_OVERFLOW
    assert (d_l1.cpu().numpy().reshape(-1).view(B.L1HIT_DTYPE)["idx"] == want[:3]).all()


def _tower_worker(rank: int, world: int, port: int, out):
    import os

    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)  # NCCL refuses two ranks on one GPU; the exchange is the same code
    try:
        from paper_1411_3968_b200 import binding as Bn

        torch.cuda.set_device(0)
        Bn.load()
        w = W.make_config(4, time_scale=0.002)  # every rank sees the same slice and takes its towers
        p, g = w.params, w.geometry
        geo = Bn.Geometry(g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks)
        prm = Bn.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps)
        a, b, ro = sharding.split_runs_by_tower(w.run_offsets, g.pmts_per_tower, g.n_tower, world)[rank]
        st = sharding.tower_local(Bn, rank, np.ascontiguousarray(w.hits[a:b]), ro, prm)
        gathered, offs = sharding.all_gather_records(st["l1"])
        res = sharding.tower_global(Bn, st, gathered, offs, geo, prm)
        out.put((rank, res["flags"].tobytes(), res["seeds"].tobytes(), res["events"].tobytes(), res["n_global_seeds"], res["status"]))
    finally:
        dist.destroy_process_group()


def test_by_tower_two_processes(B, oracle_lib):
    """The real multi-process flow: two ranks (processes), each computing on the GPU, exchanging their L1 records through
    torch.distributed (gloo here: both share the box's one GPU), against the oracle on the whole detector."""
    import socket

    import torch.multiprocessing as mp

    world = 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_tower_worker, args=(r, world, port, out)) for r in range(world)]
    for pr in procs:
        pr.start()
    got = {}
    for _ in range(world):
        r = out.get(timeout=600)
        got[r[0]] = r
    for pr in procs:
        pr.join(timeout=120)
        assert pr.exitcode == 0
    w = W.make_config(4, time_scale=0.002)
    g = w.geometry
    o = oracle_chain(w.hits, w.seg_offsets, g, w.params)
    tower = o["sorted"]["pmt_id"].astype(np.int64) // g.pmts_per_tower
    for r, (lo, hi) in enumerate(sharding.tower_ranges(g.n_tower, world)):
        mine = (tower >= lo) & (tower < hi)
        _, fl, sd, ev, ngs, st = got[r]
        assert st == 0 and ngs == len(o["seeds"])
        assert fl == o["flags"][mine].tobytes(), f"rank {r}: flags"
        assert sd == np.nonzero(o["flags"][mine] & 16)[0].astype(np.uint32).tobytes(), f"rank {r}: seeds"
        evs = np.frombuffer(ev, dtype=B.EVENT_DTYPE)
        assert len(evs) == len(o["events"]) and (evs["t_start"] == o["events"]["t_start"]).all() and (evs["t_end"] == o["events"]["t_end"]).all()
