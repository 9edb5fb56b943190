"""GPU parity: the CUDA path (through the C ABI) against the oracle, bit-exact (integer work).
Element-by-element: sorted records, permutation, flags, seeds, events."""
import numpy as np
import pytest
import torch

import oracle
from cases import case_arrays, directed_cases
from paper_1411_3968_b200 import workload as W
from util import oracle_chain, single_tower_geo

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1411_3968_b200 import binding

    binding.load()
    return binding


def _geo(B, g):
    return B.Geometry(g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks)


def _prm(B, p):
    return B.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps)


def _compare(r, o):
    assert r.sorted.tobytes() == o["sorted"].tobytes()
    assert (r.perm == o["perm"]).all()
    bad = np.nonzero(r.flags != o["flags"])[0]
    assert len(bad) == 0, (bad[:10], r.flags[bad[:10]], o["flags"][bad[:10]])
    assert r.n_seeds == len(o["seeds"]) and (r.seeds == o["seeds"]).all()
    assert r.n_events == len(o["events"])
    assert r.events.tobytes() == o["events"].tobytes()
    assert (r.status & 8) == (o["status"] & 8)


CASES = directed_cases()


@pytest.mark.parametrize("c", CASES, ids=[c["name"] for c in CASES])
def test_directed_cases(c, B, oracle_lib):
    h, seg = case_arrays(c)
    g = single_tower_geo(c["table"])
    p = W.Params(**c["params"])
    o = oracle_chain(h, seg, g, p)
    geo = _geo(B, g)
    for runs in (None, np.arange(len(h) + 1, dtype=np.uint32)):  # radix path; every hit its own run
        r = B.process_slice(h, seg, runs, geo, _prm(B, p))
        _compare(r, o)
        e = c["expect"]
        if "flags" in e:
            assert r.flags.tolist() == e["flags"]
        if "seeds" in e:
            assert r.seeds.tolist() == e["seeds"]
        if "events" in e:
            assert [tuple(int(x) for x in ev) for ev in r.events] == e["events"]
        assert r.status == 0


@pytest.mark.parametrize("cfg,ts,ss", [(0, 0.25, 1), (1, 0.1, 1), (2, 0.004, 1), (3, 0.02, 8 / 64), (4, 0.002, 1)])
@pytest.mark.parametrize("mode", [0, 1])
def test_configs_scaled(cfg, ts, ss, mode, B, oracle_lib):
    """The five BASELINE.json configs at oracle-speed sizes (several tiles, ragged tails)."""
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    p = w.params
    p.l2_mode = mode
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, p)
    geo = _geo(B, w.geometry)
    r = B.process_slice(w.hits, w.seg_offsets, w.run_offsets, geo, _prm(B, p), gather=True)
    _compare(r, o)
    assert r.status == 0
    assert len(o["seeds"]) > 0 and len(o["events"]) > 0
    tagged = np.nonzero(r.flags & 32)[0]
    assert r.gathered.tobytes() == r.sorted[tagged].tobytes()


@pytest.mark.parametrize("cfg,ts,ss", [(1, 0.05, 1), (3, 0.01, 4 / 64), (4, 0.001, 1)])
def test_shuffled_input_radix_path(cfg, ts, ss, B, oracle_lib):
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    hits, _ = W.shuffled(w)
    o = oracle_chain(hits, w.seg_offsets, w.geometry, w.params)
    r = B.process_slice(hits, w.seg_offsets, None, _geo(B, w.geometry), _prm(B, w.params))
    _compare(r, o)


def test_sort_ties_and_extreme_keys(B, oracle_lib):
    rng = np.random.default_rng(3)
    n = 50_000
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, 84, size=n)
    h["pad"] = np.arange(n) & 0xFFFF
    seg = np.array([0, 12345, 12345, n], dtype=np.uint32)
    geo = _geo(B, W.make_geometry("km3"))
    prm = B.make_params()
    for kind in ("ties", "extreme"):
        h["t_ps"] = rng.integers(0, 40, size=n) if kind == "ties" else rng.integers(-2**62, 2**62, size=n)
        if kind == "extreme":
            h["t_ps"][:4] = [-2**63, 2**63 - 1, 0, -1]
        srt, perm = oracle.sort(h, seg)
        d_in = B.hits_to_device(h)
        d_out = torch.empty_like(d_in)
        d_perm = torch.empty(n, dtype=torch.int32, device="cuda")
        st = torch.zeros(1, dtype=torch.int32, device="cuda")
        B.tt_sort_slice(d_in, d_out, d_perm, B.Offsets(seg), None, st)
        torch.cuda.synchronize()
        assert B.hits_to_host(d_out).tobytes() == srt.tobytes()
        assert (d_perm.cpu().numpy().view(np.uint32) == perm).all()
        # sorted-run path on the same keys: each segment sorted per "PMT" first
        order = np.concatenate([np.lexsort((np.arange(a, b), h["t_ps"][a:b], h["pmt_id"][a:b])) + a
                                for a, b in zip(seg[:-1], seg[1:])]) if n else np.zeros(0, dtype=np.int64)
        hr = h[order]
        key = np.concatenate([np.full(b - a, k) for k, (a, b) in enumerate(zip(seg[:-1], seg[1:]))]) * 100 + hr["pmt_id"]
        brk = np.nonzero(np.diff(key))[0] + 1
        runs = np.concatenate([[0], brk, [n]]).astype(np.uint32)
        runs = np.unique(np.concatenate([runs, seg])).astype(np.uint32)
        srt2, perm2 = oracle.sort(hr, seg)
        d_in = B.hits_to_device(hr)
        B.tt_sort_slice(d_in, d_out, d_perm, B.Offsets(seg), B.Offsets(runs), st)
        torch.cuda.synchronize()
        assert B.hits_to_host(d_out).tobytes() == srt2.tobytes()
        assert (d_perm.cpu().numpy().view(np.uint32) == perm2).all()
        assert int(st.item()) == 0


def test_status_codes(B, oracle_lib):
    w = W.make_config(1, time_scale=0.02)
    geo = _geo(B, w.geometry)
    prm = _prm(B, w.params)
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, w.params)
    # seed / event capacity too small: true counts reported, prefix valid
    r = B.process_slice(w.hits, w.seg_offsets, w.run_offsets, geo, prm, seed_cap=3, event_cap=1)
    assert r.status & B.TT_S_SEED_OVERFLOW and r.n_seeds == len(o["seeds"]) and (r.seeds == o["seeds"][:3]).all()
    assert (r.flags & 31 == o["flags"] & 31).all()
    # event capacity alone too small: the true count, the first event_cap events, every flag (INEVT included)
    w2 = W.make_config(1, time_scale=0.2)
    o2 = oracle_chain(w2.hits, w2.seg_offsets, w2.geometry, w2.params)
    assert len(o2["events"]) > 2
    r = B.process_slice(w2.hits, w2.seg_offsets, w2.run_offsets, geo, prm, event_cap=2)
    assert r.status == B.TT_S_EVENT_OVERFLOW
    assert r.n_events == len(o2["events"]) and r.events.tobytes() == o2["events"][:2].tobytes()
    assert r.n_seeds == len(o2["seeds"]) and (r.seeds == o2["seeds"]).all()
    assert (r.flags & 31 == o2["flags"] & 31).all()
    # an unsorted run
    h = w.hits.copy()
    a = int(w.run_offsets[3])
    h[[a, a + 1]] = h[[a + 1, a]]
    assert h["t_ps"][a] > h["t_ps"][a + 1]
    r = B.process_slice(h, w.seg_offsets, w.run_offsets, geo, prm)
    assert r.status & B.TT_S_RUN_UNSORTED
    # pmt_id out of range on an L1 hit
    h = w.hits.copy()
    h["pmt_id"][5] = 500
    h["charge"][5] = 1000
    o2 = oracle_chain(h, w.seg_offsets, w.geometry, w.params)
    r = B.process_slice(h, w.seg_offsets, w.run_offsets, geo, prm)
    assert (r.status & B.TT_S_BAD_PMT) and (o2["status"] & 8)
    assert (r.flags == o2["flags"]).all()


def test_dense_neighbourhood(B, oracle_lib):
    """Bursts of mutually causal L1 hits: windows above 128 candidates (wide path, lazy clique search) and
    above TT_MAX_NEIGHBOURS = 2048 (TT_S_DENSITY: star bit exact, clique bit not decided, status says so)."""
    geo_w = W.make_geometry("km3")
    geo = _geo(B, geo_w)
    rng = np.random.default_rng(9)
    for m, expect_density in ((150, False), (700, False), (2500, True)):
        h = np.zeros(m + 200, dtype=W.HIT_DTYPE)
        h["pmt_id"] = rng.integers(0, 84, size=len(h))
        h["floor"] = geo_w.floor[h["pmt_id"]]
        h["charge"] = 500
        h["t_ps"][:m] = 1_000_000_000 + np.sort(rng.integers(0, 15_000, size=m))  # all within 15 ns: a clique
        h["t_ps"][m:] = np.sort(rng.integers(2_000_000_000, 3_000_000_000, size=200))
        seg = np.array([0, len(h)], dtype=np.uint32)
        p = W.Params(l2_multiplicity=6)
        if expect_density:
            p_star = W.Params(l2_multiplicity=6, l2_mode=1)
            o = oracle_chain(h, seg, geo_w, p_star)  # star bits only (the oracle's clique search is O(k^2) per hit)
        else:
            o = oracle_chain(h, seg, geo_w, p)
        r = B.process_slice(h, seg, None, geo, _prm(B, p))
        assert ((r.flags & 8) == (o["flags"] & 8)).all()
        if expect_density:
            # fail open (R10): the dense hits get L2 := L2STAR, the status says so, and nothing else changes --
            # the 200 isolated hits (> 1 s away: no coincidence or event reaches them) are the oracle's clique-mode bytes
            assert r.status == B.TT_S_DENSITY
            dense = np.arange(len(h)) < m
            assert (((r.flags & 16) != 0)[dense] == ((r.flags & 8) != 0)[dense]).all() and (r.flags & 16)[dense].all()
            iso = oracle_chain(h[m:], np.array([0, 200], dtype=np.uint32), geo_w, p)
            assert (r.flags[m:] == iso["flags"]).all()
            assert (r.seeds == np.concatenate([np.arange(m), iso["seeds"] + m])).all()
            r2 = B.process_slice(h, seg, None, geo, _prm(B, p))  # the same bytes on every run
            assert (r2.flags == r.flags).all() and (r2.seeds == r.seeds).all() and r2.events.tobytes() == r.events.tobytes()
        else:
            assert r.status == 0
            assert (r.flags == o["flags"]).all() and (r.seeds == o["seeds"]).all()
    # a sparse graph on a wide window: many hits, few edges (table entries of 1 ps) -> search must exhaust
    tab = np.full((84, 84), 1, dtype=np.int32)
    tab[:6, :6] = 100_000
    g2 = single_tower_geo(tab)
    h = np.zeros(600, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, 84, size=600)
    h["charge"] = 500
    h["t_ps"] = np.sort(rng.integers(0, 90_000, size=600))
    seg = np.array([0, 600], dtype=np.uint32)
    for N in (3, 4, 6):
        p = W.Params(l2_multiplicity=N)
        o = oracle_chain(h, seg, g2, p)
        r = B.process_slice(h, seg, None, _geo(B, g2), _prm(B, p))
        assert (r.flags == o["flags"]).all() and (r.seeds == o["seeds"]).all() and r.status == 0
        assert 0 < len(o["seeds"]) < 600


def test_host_api_matches_device_api(B, oracle_lib):
    import ctypes

    w = W.make_config(1, time_scale=0.03)
    geo = _geo(B, w.geometry)
    prm = _prm(B, w.params)
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, w.params)
    L = B.load()
    ctx = ctypes.c_void_p(0)
    n = w.n
    assert L.tt_host_ctx_create(ctypes.byref(ctx), n, 4, len(w.run_offsets), n, n) == 0
    srt = np.zeros(n, dtype=B.HIT_DTYPE); fl = np.zeros(n, dtype=np.uint8)
    seeds = np.zeros(n, dtype=np.uint32); ev = np.zeros(n, dtype=B.EVENT_DTYPE); cnt = np.zeros(3, dtype=np.uint32)
    vp = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    seg = np.ascontiguousarray(w.seg_offsets, dtype=np.uint32); runs = np.ascontiguousarray(w.run_offsets, dtype=np.uint32)
    hin = np.ascontiguousarray(w.hits)
    rc = L.tt_process_host(ctx, vp(hin), vp(srt), vp(fl), ctypes.c_uint32(n), vp(seg), ctypes.c_uint32(len(seg) - 1),
                           vp(runs), ctypes.c_uint32(len(runs) - 1), geo.handle, ctypes.byref(prm), vp(seeds), vp(ev),
                           vp(cnt))
    assert rc == 0
    assert srt.tobytes() == o["sorted"].tobytes() and (fl == o["flags"]).all()
    assert cnt[0] == len(o["seeds"]) and (seeds[: cnt[0]] == o["seeds"]).all()
    assert cnt[1] == len(o["events"]) and ev[: cnt[1]].tobytes() == o["events"].tobytes()
    L.tt_host_ctx_destroy(ctx)


def _sort_only(B, h, seg, runs):
    d_in = B.hits_to_device(h)
    d_out = torch.empty_like(d_in)
    d_perm = torch.empty(max(len(h), 1), dtype=torch.int32, device="cuda")
    st = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.tt_sort_slice(d_in, d_out, d_perm, B.Offsets(seg), B.Offsets(runs) if runs is not None else None, st)
    torch.cuda.synchronize()
    return B.hits_to_host(d_out), d_perm.cpu().numpy().view(np.uint32)[: len(h)], int(st.item())


def _as_runs(h, seg, n_pmt):
    """Reorder arbitrary hits into PMT-major, time-ordered runs per segment; returns (hits, run offsets)."""
    parts, offs = [], [0]
    for a, b in zip(seg[:-1], seg[1:]):
        sub = h[a:b]
        o = np.lexsort((np.arange(len(sub)), sub["t_ps"], sub["pmt_id"]))
        sub = sub[o]
        parts.append(sub)
        cnt = np.bincount(sub["pmt_id"], minlength=n_pmt)
        for c in cnt:
            offs.append(offs[-1] + int(c))
    return np.concatenate(parts) if parts else h[:0], np.asarray(offs, dtype=np.uint32)


@pytest.mark.parametrize("kind", ["tie_blocks", "skewed_density", "one_outlier", "three_levels", "many_empty_runs"])
def test_merge_path_edge_cases(kind, B, oracle_lib):
    """The run-merge path off its fast path: tiles that overflow the staging capacity (swept in
    chunks), single timestamps with more hits than a chunk (tie blocks), a timestamp outlier that
    stretches the key range, three merge levels, empty runs."""
    rng = np.random.default_rng(21)
    n_pmt = 84
    if kind == "tie_blocks":
        n = 60_000
        h = np.zeros(n, dtype=W.HIT_DTYPE)
        h["t_ps"] = rng.integers(0, 3, size=n)  # ~20 000 hits per timestamp >> 4096
        seg = np.array([0, 25_000, n], dtype=np.uint32)
    elif kind == "skewed_density":
        n = 80_000
        h = np.zeros(n, dtype=W.HIT_DTYPE)
        t = rng.integers(0, 10**9, size=n)
        t[: n // 2] = rng.integers(5 * 10**8, 5 * 10**8 + 10**6, size=n // 2)  # half of the hits in 0.1 % of the range
        h["t_ps"] = t
        seg = np.array([0, n], dtype=np.uint32)
    elif kind == "one_outlier":
        n = 40_000
        h = np.zeros(n, dtype=W.HIT_DTYPE)
        h["t_ps"] = rng.integers(0, 10**8, size=n)
        h["t_ps"][7] = 2**62
        h["t_ps"][9] = -2**62
        seg = np.array([0, n], dtype=np.uint32)
    elif kind == "three_levels":
        n = 300_000  # every hit its own run: 300 000 > 512^2 runs -> three merge levels
        h = np.zeros(n, dtype=W.HIT_DTYPE)
        h["t_ps"] = rng.integers(0, 10**10, size=n)
        seg = np.array([0, 100_000, n], dtype=np.uint32)
    else:
        n = 30_000
        n_pmt = 3000  # most runs empty
        h = np.zeros(n, dtype=W.HIT_DTYPE)
        h["t_ps"] = rng.integers(0, 10**9, size=n)
        seg = np.array([0, 0, 10_000, n, n], dtype=np.uint32)
    h["pmt_id"] = rng.integers(0, n_pmt, size=n) if kind != "many_empty_runs" else rng.choice(np.arange(0, n_pmt, 7), size=n)
    h["pad"] = np.arange(n) & 0xFFFF
    if kind == "three_levels":
        hr, runs = h, np.arange(n + 1, dtype=np.uint32)
    else:
        hr, runs = _as_runs(h, seg, n_pmt)
    srt, perm = oracle.sort(hr, seg)
    out, gperm, st = _sort_only(B, hr, seg, runs)
    assert st == 0
    assert out.tobytes() == srt.tobytes()
    assert (gperm == perm).all()


def test_many_towers_global_pair_table(B, oracle_lib):
    """More than 128 towers: the tower-pair byte table does not fit the L2 rows kernel's shared memory and the
    pair-block ids are gathered from global memory instead (12 x 12 NEMO towers, 4608 PMTs, 8400-run style
    two-level merge with 4608 runs)."""
    geo = W.make_geometry("nemo", 12, 12)
    assert geo.n_tower == 144
    T_ps = 400_000_000  # 0.4 ms: ~100 k hits
    h, rl, _ = W.make_segment(geo, np.full(geo.n_pmt, 55e3), 0, T_ps, 1, 6, seed=4242)
    h["pad"] = (np.arange(len(h)) & 0xFFFF).astype(np.uint16)
    seg = np.array([0, len(h)], dtype=np.uint32)
    runs = np.zeros(len(rl) + 1, dtype=np.uint32)
    np.cumsum(rl, out=runs[1:])
    p = W.Params(l2_multiplicity=4)
    o = oracle_chain(h, seg, geo, p)
    r = B.process_slice(h, seg, runs, _geo(B, geo), _prm(B, p))
    _compare(r, o)
    assert r.status == 0 and len(o["seeds"]) > 0


@pytest.mark.parametrize("cfg,ts,ss", [(2, 0.01, 1), (3, 0.02, 8 / 64), (4, 0.004, 1)])
def test_reused_dirty_workspaces_and_determinism(cfg, ts, ss, B, oracle_lib):
    """bench.py reuses its workspaces and output buffers from step to step: garbage-filled workspaces and outputs,
    three consecutive runs of the three calls, every run byte-identical to the oracle (hence to each other)."""
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    p = w.params
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, p)
    n = w.n
    geo, prm = _geo(B, w.geometry), _prm(B, p)
    seg, runs = B.Offsets(w.seg_offsets), B.Offsets(w.run_offsets)
    d_in = B.hits_to_device(w.hits)
    d_out = torch.full_like(d_in, -1)
    d_perm = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    d_flags = torch.full((n,), 0xFF, dtype=torch.uint8, device="cuda")
    d_seeds = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    d_ev = torch.full((n, 4), -1, dtype=torch.int64, device="cuda")
    d_cnt = torch.full((4,), -1, dtype=torch.int32, device="cuda")
    ws = {}
    for it in range(3):
        d_cnt[2] = 0  # the status word is the caller's to clear
        for k in ("s", "t", "e"):
            if k in ws:
                ws[k].fill_(0xA5 if it == 1 else 0xFF)  # dirty workspaces: nothing may rely on their content
        ws["s"] = B.tt_sort_slice(d_in, d_out, d_perm, seg, runs, d_cnt[2:3], ws.get("s"))
        ws["t"] = B.tt_trigger_slice(d_out, seg, geo, prm, d_flags, d_seeds, d_cnt[0:1], d_cnt[2:3], ws.get("t"))
        ws["e"] = B.tt_extract_events(d_out, seg, d_seeds, d_cnt[0:1], prm, d_ev, d_cnt[1:2], d_flags, None, None,
                                      d_cnt[2:3], ws.get("e"))
        torch.cuda.synchronize()
        cnt = d_cnt.cpu().numpy().view(np.uint32)
        ns, ne, status = int(cnt[0]), int(cnt[1]), int(cnt[2])
        assert status == 0, (it, status)
        assert B.hits_to_host(d_out).tobytes() == o["sorted"].tobytes(), it
        assert (d_perm.cpu().numpy().view(np.uint32) == o["perm"]).all(), it
        assert (d_flags.cpu().numpy() == o["flags"]).all(), it
        assert ns == len(o["seeds"]) and (d_seeds[:ns].cpu().numpy().view(np.uint32) == o["seeds"]).all(), it
        ev = d_ev[:ne].cpu().numpy().reshape(-1).view(B.EVENT_DTYPE)
        assert ne == len(o["events"]) and ev.tobytes() == o["events"].tobytes(), it
    geo.close()


@pytest.mark.parametrize("cfg,ts,ss", [(1, 0.1, 1), (4, 0.002, 1)])
def test_cuda_graph_replay(cfg, ts, ss, B, oracle_lib):
    """bench.py replays the step as a CUDA graph: the three calls allocate nothing and never synchronise, so they can be
    captured as they are.  Replays onto garbage-filled outputs and workspaces give the oracle's bytes every time."""
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    p = w.params
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, p)
    n = w.n
    geo, prm = _geo(B, w.geometry), _prm(B, p)
    seg, runs = B.Offsets(w.seg_offsets), B.Offsets(w.run_offsets)
    d_in = B.hits_to_device(w.hits)
    d_out = torch.empty_like(d_in)
    d_flags = torch.zeros(n, dtype=torch.uint8, device="cuda")
    d_seeds = torch.zeros(n, dtype=torch.int32, device="cuda")
    d_ev = torch.zeros((n, 4), dtype=torch.int64, device="cuda")
    d_cnt = torch.zeros(4, dtype=torch.int32, device="cuda")
    ws = {}

    def step():
        d_cnt.zero_()
        ws["s"] = B.tt_sort_slice(d_in, d_out, None, seg, runs, d_cnt[2:3], ws.get("s"))
        ws["t"] = B.tt_trigger_slice(d_out, seg, geo, prm, d_flags, d_seeds, d_cnt[0:1], d_cnt[2:3], ws.get("t"))
        ws["e"] = B.tt_extract_events(d_out, seg, d_seeds, d_cnt[0:1], prm, d_ev, d_cnt[1:2], d_flags, None, None,
                                      d_cnt[2:3], ws.get("e"))

    step()  # workspaces allocated, kernel attributes set: outside the capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        step()
    for it in range(3):
        for t in (d_out, d_flags, d_seeds, d_ev, d_cnt, ws["s"], ws["t"], ws["e"]):
            t.fill_(-1 if t.dtype in (torch.int32, torch.int64) else 0xA5)
        g.replay()
        torch.cuda.synchronize()
        cnt = d_cnt.cpu().numpy().view(np.uint32)
        ns, ne, status = int(cnt[0]), int(cnt[1]), int(cnt[2])
        assert status == 0, it
        assert B.hits_to_host(d_out).tobytes() == o["sorted"].tobytes(), it
        assert (d_flags.cpu().numpy() == o["flags"]).all(), it
        assert ns == len(o["seeds"]) and (d_seeds[:ns].cpu().numpy().view(np.uint32) == o["seeds"]).all(), it
        ev = d_ev[:ne].cpu().numpy().reshape(-1).view(B.EVENT_DTYPE)
        assert ne == len(o["events"]) and ev.tobytes() == o["events"].tobytes(), it
    geo.close()
