"""GPU parity of the fused call tt_sort_trigger_slice (last bullet: "a fused call is allowed in
addition; the three calls must exist, be tested, and give identical results"): L1 evaluated by the last merge level on
its time tile in shared memory, the hits near a tile edge finished by l1_boundary_kernel.  Everything is compared with
the oracle byte for byte, and with the three-call path."""
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
    assert len(bad) == 0, (len(bad), bad[:10], r.flags[bad[:10]], o["flags"][bad[:10]])
    assert r.n_seeds == len(o["seeds"]) and (r.seeds == o["seeds"]).all()
    assert r.n_events == len(o["events"])
    assert r.events.tobytes() == o["events"].tobytes()
    assert (r.status & 8) == (o["status"] & 8)


def _same(r, r3):
    assert r.sorted.tobytes() == r3.sorted.tobytes() and (r.perm == r3.perm).all()
    assert (r.flags == r3.flags).all() and r.n_seeds == r3.n_seeds and (r.seeds == r3.seeds).all()
    assert r.n_events == r3.n_events and r.events.tobytes() == r3.events.tobytes() and r.status == r3.status


CASES = directed_cases()


@pytest.mark.parametrize("c", CASES, ids=[c["name"] for c in CASES])
def test_directed_cases_fused(c, B, oracle_lib):
    h, seg = case_arrays(c)
    g = single_tower_geo(c["table"])
    p = W.Params(**c["params"])
    o = oracle_chain(h, seg, g, p)
    geo = _geo(B, g)
    for runs in (None, np.arange(len(h) + 1, dtype=np.uint32)):  # radix path (unfused inside); every hit its own run
        r = B.process_slice(h, seg, runs, geo, _prm(B, p), fused=True)
        _compare(r, o)
        e = c["expect"]
        if "flags" in e:
            assert r.flags.tolist() == e["flags"]
        if "seeds" in e:
            assert r.seeds.tolist() == e["seeds"]
        assert r.status == 0


@pytest.mark.parametrize("cfg,ts,ss", [(0, 0.25, 1), (1, 0.1, 1), (2, 0.004, 1), (3, 0.02, 8 / 64), (4, 0.002, 1)])
@pytest.mark.parametrize("mode", [0, 1])
def test_configs_scaled_fused(cfg, ts, ss, mode, B, oracle_lib):
    """The five BASELINE.json configs at oracle-speed sizes (dozens of time tiles; cfg4 puts ~18 hits inside +-20 ns,
    so hundreds of coincidences straddle tile edges)."""
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    p = w.params
    p.l2_mode = mode
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, p)
    geo = _geo(B, w.geometry)
    r = B.process_slice(w.hits, w.seg_offsets, w.run_offsets, geo, _prm(B, p), fused=True)
    _compare(r, o)
    assert r.status == 0 and len(o["seeds"]) > 0
    _same(r, B.process_slice(w.hits, w.seg_offsets, w.run_offsets, geo, _prm(B, p)))


@pytest.mark.parametrize("lc", [0, 1, 20_000, 3_000_000, 10**9, 2**32 - 1, 2**32, 2**40])
def test_lc_windows_against_tile_width(lc, B, oracle_lib):
    """Coincidence windows from 0 to far wider than a time tile (every hit is then 'near an edge' and finished by the
    exact scans), and at the 32-bit boundary of the in-tile relative times."""
    w = W.make_config(1, time_scale=0.03)
    p = w.params
    p.lc_window_ps = lc
    p.l2_multiplicity = 6 if lc > 10**6 else 5
    if lc > 10**6:  # keep the oracle's L2 affordable: almost every hit is L1 then
        p.l2_mode = 1
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, p)
    r = B.process_slice(w.hits, w.seg_offsets, w.run_offsets, _geo(B, w.geometry), _prm(B, p), fused=True)
    _compare(r, o)


def _as_runs(h, seg, n_pmt):
    parts, offs = [], [0]
    for a, b in zip(seg[:-1], seg[1:]):
        sub = h[a:b]
        o = np.lexsort((np.arange(len(sub)), sub["t_ps"], sub["pmt_id"]))
        sub = sub[o]
        parts.append(sub)
        for c in np.bincount(sub["pmt_id"], minlength=n_pmt):
            offs.append(offs[-1] + int(c))
    return np.concatenate(parts) if parts else h[:0], np.asarray(offs, dtype=np.uint32)


@pytest.mark.parametrize("kind", ["tie_blocks", "skewed_density", "one_outlier", "three_levels", "narrow_tiles"])
def test_general_tiles_fused(kind, B, oracle_lib):
    """Tiles the fast kernel hands to the general one (overflowing tiles, tie blocks, >= 2^32 ps across a tile, tiles
    narrower than the bucket count): their hits get every L1 bit from the exact scans."""
    rng = np.random.default_rng(77)
    geo_w = W.make_geometry("km3")
    n_pmt = 84
    if kind == "tie_blocks":
        n = 30_000
        t = rng.integers(0, 3, size=n) * 15_000  # ~10 000 hits per timestamp, 15 ns apart: all inside LC of each other
        seg = np.array([0, 12_000, n], dtype=np.uint32)
    elif kind == "skewed_density":
        n = 60_000
        t = rng.integers(0, 10**9, size=n)
        t[: n // 2] = rng.integers(5 * 10**8, 5 * 10**8 + 10**7, size=n // 2)
        seg = np.array([0, n], dtype=np.uint32)
    elif kind == "one_outlier":
        n = 40_000
        t = rng.integers(0, 10**9, size=n)
        t[7], t[9] = 2**62, -2**62
        seg = np.array([0, n], dtype=np.uint32)
    elif kind == "three_levels":
        n = 270_000
        t = rng.integers(0, 10**11, size=n)
        seg = np.array([0, 100_000, n], dtype=np.uint32)
    else:
        n = 50_000
        t = rng.integers(0, 30_000, size=n)  # 50 000 hits in 30 ns: tiles of ~2 000 ps < 4096 buckets
        seg = np.array([0, n], dtype=np.uint32)
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["t_ps"] = t
    h["pmt_id"] = rng.integers(0, n_pmt, size=n)
    h["floor"] = geo_w.floor[h["pmt_id"]]
    h["charge"] = rng.integers(50, 320, size=n)
    h["pad"] = np.arange(n) & 0xFFFF
    if kind == "three_levels":
        hr, runs = h, np.arange(n + 1, dtype=np.uint32)
    else:
        hr, runs = _as_runs(h, seg, n_pmt)
    p = W.Params(l2_multiplicity=5, l2_mode=1)  # star mode: dense blocks would make the oracle's clique search slow
    if kind in ("tie_blocks", "narrow_tiles"):
        p.l2_window_ps = 0  # no L2 edges at all between different times: the L1 bits are what is tested here
    o = oracle_chain(hr, seg, geo_w, p)
    r = B.process_slice(hr, seg, runs, _geo(B, geo_w), _prm(B, p), fused=True)
    assert r.status in (0, B.TT_S_DENSITY)
    assert r.sorted.tobytes() == o["sorted"].tobytes() and (r.perm == o["perm"]).all()
    assert ((r.flags & 7) == (o["flags"] & 7)).all()
    if r.status == 0:
        _compare(r, o)


def test_fused_status_and_capacity(B, oracle_lib):
    w = W.make_config(1, time_scale=0.02)
    geo, prm = _geo(B, w.geometry), _prm(B, w.params)
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, w.params)
    r = B.process_slice(w.hits, w.seg_offsets, w.run_offsets, geo, prm, seed_cap=3, event_cap=1, fused=True)
    assert r.status & B.TT_S_SEED_OVERFLOW and r.n_seeds == len(o["seeds"]) and (r.seeds == o["seeds"][:3]).all()
    assert (r.flags & 31 == o["flags"] & 31).all()
    h = w.hits.copy()
    a = int(w.run_offsets[3])
    h[[a, a + 1]] = h[[a + 1, a]]
    r = B.process_slice(h, w.seg_offsets, w.run_offsets, geo, prm, fused=True)
    assert r.status & B.TT_S_RUN_UNSORTED
    # a disorder that stays inside one tile's piece, at every position of a 32-lane group
    for off in range(0, 40, 3):
        h = w.hits.copy()
        a = int(w.run_offsets[5]) + 100 + off
        if h["t_ps"][a] == h["t_ps"][a + 1]:
            continue
        h[[a, a + 1]] = h[[a + 1, a]]
        r = B.process_slice(h, w.seg_offsets, w.run_offsets, geo, prm, fused=True)
        assert r.status & B.TT_S_RUN_UNSORTED, off
    h = w.hits.copy()
    h["pmt_id"][5] = 500
    h["charge"][5] = 1000
    o2 = oracle_chain(h, w.seg_offsets, w.geometry, w.params)
    r = B.process_slice(h, w.seg_offsets, w.run_offsets, geo, prm, fused=True)
    assert (r.status & B.TT_S_BAD_PMT) and (r.flags == o2["flags"]).all()


@pytest.mark.parametrize("fused", [True, False])
@pytest.mark.parametrize("cfg,ts", [(2, 0.004), (4, 0.004)])
def test_l1_capacity(cfg, ts, fused, B, oracle_lib):
    """tt_params.l1_capacity bounds the L1 list (and with it the trigger workspace).  Enough room: the oracle's bytes.
    Too little: TT_S_L1_OVERFLOW, every L1 flag still exact, L2 over the first l1_capacity L1 hits in time order -- so no
    L2 bit the full answer does not have, and the full answer wherever the window of a hit ends before the cut."""
    w = W.make_config(cfg, time_scale=ts)
    g, p = w.geometry, w.params
    o = oracle_chain(w.hits, w.seg_offsets, g, p)
    m = int(((o["flags"] & B.TT_L1) != 0).sum())
    assert m > 200
    geo = _geo(B, g)

    def prm(cap):
        return B.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps,
                             l1_capacity=cap)

    for cap in (m, m + 17, len(w.hits) + 5):  # room for every L1 hit
        r = B.process_slice(w.hits, w.seg_offsets, w.run_offsets, geo, prm(cap), fused=fused)
        assert r.status == 0, cap
        _compare(r, o)
    cap = m // 2
    r = B.process_slice(w.hits, w.seg_offsets, w.run_offsets, geo, prm(cap), fused=fused)
    assert r.status & B.TT_S_L1_OVERFLOW
    assert r.sorted.tobytes() == o["sorted"].tobytes()
    assert ((r.flags & 7) == (o["flags"] & 7)).all()                    # Q, LC, L1: all hits
    l2 = B.TT_L2 | B.TT_L2STAR
    assert ((r.flags & l2) & ~(o["flags"] & l2) == 0).all()             # fewer L1 hits listed: never more L2 bits
    l1_pos = np.nonzero(o["flags"] & B.TT_L1)[0]
    t_cut = int(o["sorted"]["t_ps"][l1_pos[cap]])                        # first L1 hit that is not listed
    reach = min(int(p.l2_window_ps), int(g.blocks.max()))
    early = o["sorted"]["t_ps"] < t_cut - reach                          # windows that end before the cut (one segment)
    assert early.sum() > 0 and ((r.flags & l2)[early] == (o["flags"] & l2)[early]).all()
    assert (r.flags[l1_pos[cap:]] & l2 == 0).all()                       # unlisted L1 hits: no L2 bit
    # the workspace follows the capacity
    n = len(w.hits)
    import ctypes
    need = {}
    for c in (0, cap):
        nb = ctypes.c_size_t(0)
        pr = prm(c)
        rc = B.load().tt_trigger_slice(None, ctypes.c_uint32(n), None, w.seg_offsets.ctypes.data_as(ctypes.c_void_p),
                                       ctypes.c_uint32(len(w.seg_offsets) - 1), geo.handle, ctypes.byref(pr), None, None,
                                       ctypes.c_uint32(n), None, None, ctypes.byref(nb), None, None)
        assert rc == 0
        need[c] = nb.value
    assert need[cap] < need[0] and need[0] - need[cap] >= 60 * (n - cap)
    geo.close()


@pytest.mark.parametrize("cfg,ts,ss", [(2, 0.01, 1), (3, 0.02, 8 / 64), (4, 0.004, 1)])
def test_fused_graph_replay_dirty_buffers(cfg, ts, ss, B, oracle_lib):
    """bench.py's step with the fused call: captured in a CUDA graph, replayed onto garbage-filled outputs and
    workspaces (misaligned flag array on purpose), the oracle's bytes every time."""
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    p = w.params
    o = oracle_chain(w.hits, w.seg_offsets, w.geometry, p)
    n = w.n
    geo, prm = _geo(B, w.geometry), _prm(B, p)
    seg, runs = B.Offsets(w.seg_offsets), B.Offsets(w.run_offsets)
    d_in = B.hits_to_device(w.hits)
    d_out = torch.empty_like(d_in)
    d_flags_buf = torch.zeros(n + 16, dtype=torch.uint8, device="cuda")
    d_flags = d_flags_buf[5:5 + n]  # not 16-byte aligned
    d_seeds = torch.zeros(n, dtype=torch.int32, device="cuda")
    d_ev = torch.zeros((n, 4), dtype=torch.int64, device="cuda")
    d_cnt = torch.zeros(4, dtype=torch.int32, device="cuda")
    ws = {}

    def step():
        d_cnt.zero_()
        ws["f"] = B.tt_sort_trigger_slice(d_in, d_out, None, seg, runs, geo, prm, d_flags, d_seeds, d_cnt[0:1], d_cnt[2:3],
                                          ws.get("f"))
        ws["e"] = B.tt_extract_events(d_out, seg, d_seeds, d_cnt[0:1], prm, d_ev, d_cnt[1:2], d_flags, None, None,
                                      d_cnt[2:3], ws.get("e"))

    step()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        step()
    for it in range(3):
        for t in (d_out, d_flags_buf, d_seeds, d_ev, d_cnt, ws["f"], ws["e"]):
            t.fill_(-1 if t.dtype in (torch.int32, torch.int64) else 0xA5)
        g.replay()
        torch.cuda.synchronize()
        cnt = d_cnt.cpu().numpy().view(np.uint32)
        ns, ne, status = int(cnt[0]), int(cnt[1]), int(cnt[2])
        assert status == 0, it
        assert B.hits_to_host(d_out).tobytes() == o["sorted"].tobytes(), it
        assert (d_flags.cpu().numpy() == o["flags"]).all(), it
        fb = d_flags_buf.cpu().numpy()
        assert (fb[:5] == 0xA5).all() and (fb[5 + n:] == 0xA5).all(), "bytes outside the flag array were written"
        assert ns == len(o["seeds"]) and (d_seeds[:ns].cpu().numpy().view(np.uint32) == o["seeds"]).all(), it
        ev = d_ev[:ne].cpu().numpy().reshape(-1).view(B.EVENT_DTYPE)
        assert ne == len(o["events"]) and ev.tobytes() == o["events"].tobytes(), it
    geo.close()


def test_two_host_threads_two_streams(B, oracle_lib):
    """include/tt.h: calls from several host threads are allowed (per-device set-up under a lock, per-thread plan
    cache).  Two threads, each on its own stream and its own workload, several rounds; both get the oracle's bytes."""
    import threading

    ws_ = [W.make_config(1, time_scale=0.05), W.make_config(3, time_scale=0.02, seg_scale=4 / 64)]
    os_ = [oracle_chain(w.hits, w.seg_offsets, w.geometry, w.params) for w in ws_]
    geos = [_geo(B, w.geometry) for w in ws_]
    errs = []

    def work(k):
        try:
            torch.cuda.set_device(0)
            w, o = ws_[k], os_[k]
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for it in range(4):
                    r = B.process_slice(w.hits, w.seg_offsets, w.run_offsets, geos[k], _prm(B, w.params), fused=bool(it & 1))
                    _compare(r, o)
        except Exception as ex:  # noqa: BLE001
            errs.append((k, repr(ex)))

    th = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    assert not errs, errs


def test_host_pipeline_submit_wait(B, oracle_lib):
    """tt_host_submit / tt_host_wait with two slices in flight (different slices, alternating), against the oracle;
    a third submit is refused; tt_process_host is refused while slices are in flight."""
    import ctypes

    ws_ = [W.make_config(1, time_scale=0.03), W.make_config(1, time_scale=0.05, seed_offset=3)]
    os_ = [oracle_chain(w.hits, w.seg_offsets, w.geometry, w.params) for w in ws_]
    geo = _geo(B, ws_[0].geometry)
    prm = _prm(B, ws_[0].params)
    L = B.load()
    ctx = ctypes.c_void_p(0)
    nmax = max(w.n for w in ws_)
    assert L.tt_host_ctx_create(ctypes.byref(ctx), nmax, 4, len(ws_[0].run_offsets), nmax, nmax) == 0
    vp = lambda a: a.ctypes.data_as(ctypes.c_void_p)
    bufs = []
    for w in ws_:
        bufs.append(dict(hin=np.ascontiguousarray(w.hits), srt=np.zeros(w.n, dtype=B.HIT_DTYPE), fl=np.zeros(w.n, dtype=np.uint8),
                         seeds=np.zeros(nmax, dtype=np.uint32), ev=np.zeros(nmax, dtype=B.EVENT_DTYPE),
                         cnt=np.zeros(3, dtype=np.uint32), seg=np.ascontiguousarray(w.seg_offsets, dtype=np.uint32),
                         runs=np.ascontiguousarray(w.run_offsets, dtype=np.uint32)))

    def submit(k, want_sorted=True):
        b, w = bufs[k], ws_[k]
        return L.tt_host_submit(ctx, vp(b["hin"]), vp(b["srt"]) if want_sorted else ctypes.c_void_p(0), vp(b["fl"]),
                                ctypes.c_uint32(w.n), vp(b["seg"]), ctypes.c_uint32(len(b["seg"]) - 1), vp(b["runs"]),
                                ctypes.c_uint32(len(b["runs"]) - 1), geo.handle, ctypes.byref(prm), vp(b["seeds"]),
                                vp(b["ev"]), vp(b["cnt"]))

    def check(k, want_sorted=True):
        b, o = bufs[k], os_[k]
        if want_sorted:
            assert b["srt"].tobytes() == o["sorted"].tobytes()
        assert (b["fl"] == o["flags"]).all()
        assert b["cnt"][0] == len(o["seeds"]) and (b["seeds"][: b["cnt"][0]] == o["seeds"]).all()
        assert b["cnt"][1] == len(o["events"]) and b["ev"][: b["cnt"][1]].tobytes() == o["events"].tobytes()
        assert b["cnt"][2] == 0

    assert L.tt_host_wait(ctx) == B.TT_E_INVAL  # nothing in flight
    for want_sorted in (True, False):
        assert submit(0, want_sorted) == 0
        for it in range(1, 6):
            assert submit(it & 1, want_sorted) == 0
            if it == 1:
                assert submit(0, want_sorted) == B.TT_E_INVAL  # both slots busy
            assert L.tt_host_wait(ctx) == 0
            check((it - 1) & 1, want_sorted)
            for key in ("srt", "fl", "seeds", "ev", "cnt"):
                bufs[(it - 1) & 1][key][...] = 0 if key != "fl" else 0xEE
        assert L.tt_host_wait(ctx) == 0
        check(5 & 1, want_sorted)
    L.tt_host_ctx_destroy(ctx)
