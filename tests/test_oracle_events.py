"""Pins P9-P12: seeds, event-window merge, injected tracks, chunking invariance."""
import numpy as np
import pytest

import oracle
from oracle import brute
from paper_1411_3968_b200 import workload as W
from util import geo_args, oracle_chain, params_kw

F_L1, F_STAR, F_L2, F_EV = 4, 8, 16, 32


def test_events_brute_force_p11(oracle_lib):
    """Random seeds on tiny inputs: events == union of the closed windows [t-H, t+H] (union-find over
    all pairs, oracle/brute.py); hit ranges and INEVT tags == direct definition."""
    rng = np.random.default_rng(11)
    for trial in range(30):
        n = int(rng.integers(1, 60))
        Hh = int(rng.choice([5, 50, 1000]))
        h = np.zeros(n, dtype=W.HIT_DTYPE)
        h["t_ps"] = rng.integers(-500, 4000, size=n)
        cut = sorted(rng.integers(0, n + 1, size=2).tolist())
        seg = np.array([0, cut[0], cut[1], n], dtype=np.uint32)
        srt, _ = oracle.sort(h, seg)
        is_seed = rng.random(n) < 0.3
        seeds = np.nonzero(is_seed)[0].astype(np.uint32)
        flags = np.zeros(n, dtype=np.uint8)
        ev = oracle.events(srt, seg, seeds, event_half_ps=Hh, flags=flags)
        sg = brute.seg_id(n, seg)
        ref = brute.event_groups(srt["t_ps"][seeds], sg[seeds], Hh)
        assert len(ev) == len(ref)
        t = srt["t_ps"]
        for e, (s, t0, t1, members) in zip(ev, ref):
            assert (int(e["t_start"]), int(e["t_end"])) == (t0, t1)
            assert list(range(int(e["seed_begin"]), int(e["seed_begin"]) + int(e["n_seeds"]))) == members
            inside = np.nonzero((sg == s) & (t >= t0) & (t <= t1))[0]
            assert int(e["hit_begin"]) == inside[0] and int(e["hit_end"]) == inside[-1] + 1
            assert (np.diff(inside) == 1).all()
        # a hit is INEVT <=> some seed of its segment is within H of it
        want = np.zeros(n, dtype=bool)
        for i in range(n):
            want[i] = any(sg[s] == sg[i] and abs(int(t[s]) - int(t[i])) <= Hh for s in seeds)
        assert (((flags & F_EV) != 0) == want).all()


@pytest.mark.parametrize("cfg,ts", [(2, 0.004), (4, 0.0015), (1, 0.05)])
def test_seed_and_event_invariants_p10_p11(cfg, ts, oracle_lib):
    w = W.make_config(cfg, time_scale=ts)
    r = oracle_chain(w.hits, w.seg_offsets, w.geometry, w.params)
    f, seeds, ev, t = r["flags"], r["seeds"], r["events"], r["sorted"]["t_ps"]
    H = w.params.event_half_ps
    # P10: ascending, unique, count = popcount of L2 bits
    assert (np.diff(seeds.astype(np.int64)) > 0).all()
    assert len(seeds) == int(((f & F_L2) != 0).sum()) and ((f[seeds] & F_L2) != 0).all()
    assert len(seeds) > 0
    # P11: ascending and disjoint in time and hit range; every seed in exactly one event;
    # n_events = 1 + #{gaps > 2H}
    assert (ev["t_start"][1:] > ev["t_end"][:-1]).all()
    assert (ev["hit_begin"][1:] >= ev["hit_end"][:-1]).all()
    assert int(ev["n_seeds"].sum()) == len(seeds)
    assert (ev["seed_begin"] == np.concatenate([[0], np.cumsum(ev["n_seeds"])[:-1]])).all()
    gaps = np.diff(t[seeds])
    assert len(ev) == 1 + int((gaps > 2 * H).sum())
    tagged = np.zeros(len(f), dtype=bool)
    for e in ev:
        tagged[int(e["hit_begin"]):int(e["hit_end"])] = True
    assert (((f & F_EV) != 0) == tagged).all()
    ts_ = t[seeds]
    k = np.searchsorted(ts_, t)
    near = np.zeros(len(t), dtype=bool)
    near |= (k < len(ts_)) & (np.abs(ts_[np.minimum(k, len(ts_) - 1)] - t) <= H)
    near |= (k > 0) & (np.abs(ts_[np.maximum(k - 1, 0)] - t) <= H)
    assert (tagged == near).all()


@pytest.mark.parametrize("cfg,ts", [(0, 0.25), (1, 0.1), (4, 0.002)])
def test_injected_tracks_fire_p9(cfg, ts, oracle_lib):
    """Every injected track whose own hits include >= N L1 hits has all of them flagged L2 and inside
    one event (north_star invariant).  The premise -- all pairs of one track's hits are edges,
    |dt| <= d*n/c + 20 ns up to the 1 ns jitter -- is asserted pair by pair from the table."""
    w = W.make_config(cfg, time_scale=ts)
    r = oracle_chain(w.hits, w.seg_offsets, w.geometry, w.params)
    trk = w.track_id[r["perm"]]
    f, srt, ev = r["flags"], r["sorted"], r["events"]
    N = w.params.l2_multiplicity
    geo = w.geometry
    fired = 0
    for k in np.unique(trk[trk >= 0]):
        idx = np.nonzero((trk == k) & ((f & F_L1) != 0))[0]
        if len(idx) < N:
            continue
        pm = srt["pmt_id"][idx].astype(np.int64); tt = srt["t_ps"][idx]
        for a in range(len(idx)):
            for b in range(a + 1, len(idx)):
                ta, tb = pm[a] // geo.pmts_per_tower, pm[b] // geo.pmts_per_tower
                blk = int(geo.pair_block[ta * geo.n_tower + tb])
                if blk < 0:
                    break
                lim = int(geo.blocks[blk, pm[a] % geo.pmts_per_tower, pm[b] % geo.pmts_per_tower])
                assert abs(int(tt[a]) - int(tt[b])) <= lim
            else:
                continue
            break
        else:
            assert ((f[idx] & F_L2) != 0).all()
            e = np.searchsorted(ev["hit_end"], idx, side="right")
            assert (e == e[0]).all() and (ev["hit_begin"][e[0]] <= idx[0])
            fired += 1
    assert fired > 0


def test_chunking_invariance_p12(oracle_lib):
    """Processing a segment as time chunks with a halo of W + LC (flags, seeds) and H + W + LC (INEVT)
    on each side gives identical per-hit results; plus run-twice determinism."""
    w = W.make_config(2, time_scale=0.004)
    p = w.params
    r = oracle_chain(w.hits, w.seg_offsets, w.geometry, p)
    assert r["flags"].tobytes() == oracle_chain(w.hits, w.seg_offsets, w.geometry, p)["flags"].tobytes()
    srt, f = r["sorted"], r["flags"]
    t = srt["t_ps"]
    halo = p.event_half_ps + p.l2_window_ps + p.lc_window_ps
    edges = np.linspace(int(t[0]), int(t[-1]) + 1, 5).astype(np.int64)
    for c0, c1 in zip(edges[:-1], edges[1:]):
        a = int(np.searchsorted(t, c0 - halo, "left")); b = int(np.searchsorted(t, c1 + halo, "left"))
        sub = srt[a:b]
        seg = np.array([0, b - a], dtype=np.uint32)
        tr = oracle.trigger(sub, seg, **geo_args(w.geometry), **params_kw(p))
        fl = tr.flags.copy()
        oracle.events(sub, seg, tr.seeds, event_half_ps=p.event_half_ps, flags=fl)
        own = (sub["t_ps"] >= c0) & (sub["t_ps"] < c1)
        assert (fl[own] == f[a:b][own]).all()
    assert ((f & F_EV) != 0).any() and ((f & F_EV) == 0).any()
