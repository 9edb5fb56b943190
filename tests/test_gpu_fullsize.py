"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (tt_sort_trigger_slice +
tt_extract_events with INEVT tagging, seed / event capacity n / 4; the three separate calls are run too and must give
the same bytes), on all five configs (north_star: "GPU output bit-exact with the oracle on all
five configs").

Three layers, cheapest first:
  * properties that hold at any size, restated in numpy on the downloaded arrays (ordered, a permutation of the input,
    flag implications, seeds = positions of the L2 bit, events = interval merge of the seed windows);
  * two SAMPLED time windows cut out of the input and run through the oracle alone (chunking invariance P12, SURVEY.md
    8(c): halo H + W + LC = 6.02 us) -- a fast pre-check that points at a time range when something is off;
  * the WHOLE input through oracle.sort -> oracle.trigger -> oracle.events (cfg4: ~1 min of one host core) and every
    output compared byte for byte: sorted records, the permutation, every flag byte, the seed list, the event array.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1411_3968_b200 import workload as W
from util import geo_args, params_kw

pytestmark = pytest.mark.gpu

HALO_PS = 6_100_000      # >= H + W + LC = 6.02 us
INTERIOR_PS = 4_000_000  # compared part of a window: centre +- 4 us
N_WINDOWS = 2


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1411_3968_b200 import binding

    binding.load()
    return binding


def _run_bench_config(B, w):
    """Exactly bench.py's step(): returns downloaded sorted hits, flags, seeds, events, status."""
    n = w.n
    g, p = w.geometry, w.params
    geo = B.Geometry(g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks)
    prm = B.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps)
    seg, runs = B.Offsets(w.seg_offsets), B.Offsets(w.run_offsets)
    d_in = B.hits_to_device(w.hits)
    d_out = torch.empty_like(d_in)
    cap = max(n // 4, 1024)
    d_flags = torch.zeros(n, dtype=torch.uint8, device="cuda")
    d_seeds = torch.zeros(cap, dtype=torch.int32, device="cuda")
    d_ev = torch.zeros((cap, 4), dtype=torch.int64, device="cuda")
    d_cnt = torch.zeros(4, dtype=torch.int32, device="cuda")
    # bench.py's step: the fused call + events
    d_flags.fill_(0xEE)  # every byte is written by the fused call
    B.tt_sort_trigger_slice(d_in, d_out, None, seg, runs, geo, prm, d_flags, d_seeds, d_cnt[0:1], d_cnt[2:3])
    B.tt_extract_events(d_out, seg, d_seeds, d_cnt[0:1], prm, d_ev, d_cnt[1:2], d_flags, None, None, d_cnt[2:3])
    torch.cuda.synchronize()
    cnt = d_cnt.cpu().numpy().view(np.uint32)
    ns, ne, status = int(cnt[0]), int(cnt[1]), int(cnt[2])
    assert ns <= cap and ne <= cap
    srt = B.hits_to_host(d_out)
    flags = d_flags.cpu().numpy()
    seeds = d_seeds[:ns].cpu().numpy().view(np.uint32)
    events = d_ev[:ne].cpu().numpy().reshape(-1).view(B.EVENT_DTYPE).copy()
    # the three separate calls (bench.py --fused off) give the same bytes
    d_cnt.zero_(); d_out.fill_(-1); d_flags.fill_(0); d_seeds.fill_(-1); d_ev.fill_(-1)
    B.tt_sort_slice(d_in, d_out, None, seg, runs, d_cnt[2:3])
    B.tt_trigger_slice(d_out, seg, geo, prm, d_flags, d_seeds, d_cnt[0:1], d_cnt[2:3])
    B.tt_extract_events(d_out, seg, d_seeds, d_cnt[0:1], prm, d_ev, d_cnt[1:2], d_flags, None, None, d_cnt[2:3])
    torch.cuda.synchronize()
    cnt3 = d_cnt.cpu().numpy().view(np.uint32)
    assert (int(cnt3[0]), int(cnt3[1]), int(cnt3[2])) == (ns, ne, status), "three calls and fused call: counts differ"
    assert torch.equal(d_flags, torch.from_numpy(flags).cuda()), "three calls and fused call: flags differ"
    assert B.hits_to_host(d_out).tobytes() == srt.tobytes(), "three calls and fused call: sorted records differ"
    assert (d_seeds[:ns].cpu().numpy().view(np.uint32) == seeds).all(), "three calls and fused call: seeds differ"
    assert d_ev[:ne].cpu().numpy().reshape(-1).view(B.EVENT_DTYPE).tobytes() == events.tobytes(), "events differ"
    del d_flags, d_seeds, d_ev
    # the permutation output (bench.py does not ask for it): a second sort call into a scratch buffer
    d_out.fill_(-1)
    d_perm = torch.full((n,), -1, dtype=torch.int32, device="cuda")
    st2 = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.tt_sort_slice(d_in, d_out, d_perm, seg, runs, st2)
    torch.cuda.synchronize()
    assert int(st2.item()) == 0
    assert B.hits_to_host(d_out).tobytes() == srt.tobytes(), "sort with and without the permutation output differ"
    perm = d_perm.cpu().numpy().view(np.uint32)
    geo.close()
    return srt, perm, flags, seeds, events, status


def _checksum(h):
    """Order-independent 64-bit checksums of whole 16-byte records (sum and xor of a mixed word)."""
    a = h.view(np.uint64).reshape(-1, 2)
    with np.errstate(over="ignore"):
        x = a[:, 0] * np.uint64(0x9E3779B97F4A7C15) + (a[:, 1] ^ np.uint64(0xC2B2AE3D27D4EB4F)) * np.uint64(0x165667B19E3779F9)
        x ^= x >> np.uint64(29)
        return int(np.add.reduce(x, dtype=np.uint64)), int(np.bitwise_xor.reduce(x))


@pytest.mark.parametrize("cfg", [0, 1, 2, 3, 4])
def test_full_size_config(cfg, B, oracle_lib):
    w = W.make_config(cfg)
    p, g = w.params, w.geometry
    srt, perm, flags, seeds, events, status = _run_bench_config(B, w)
    assert status == 0
    n, seg = w.n, np.asarray(w.seg_offsets, dtype=np.int64)
    t = srt["t_ps"]

    # ---- properties at full size ---------------------------------------------------------------------
    for s in range(len(seg) - 1):  # ordered inside each segment, and a permutation of that segment's input
        a, b = seg[s], seg[s + 1]
        assert (np.diff(t[a:b]) >= 0).all(), f"segment {s} not time-ordered"
        if len(seg) - 1 > 1:
            assert _checksum(srt[a:b]) == _checksum(w.hits[a:b]), f"segment {s} is not a permutation of its input"
    assert _checksum(srt) == _checksum(w.hits)
    q, lc, l1, star, l2, inevt = [(flags & m) != 0 for m in (1, 2, 4, 8, 16, 32)]
    assert ((flags & 0xC0) == 0).all()
    assert (q == (srt["charge"] >= p.q_thresh)).all()
    assert (l1 == (q | lc)).all()
    assert not (star & ~l1).any() and not (l2 & ~star).any()  # L2 within L2STAR within L1 (P8)
    assert not (l2 & ~inevt).any()                            # a seed lies in its own event window
    assert (np.nonzero(l2)[0] == seeds).all()                 # ascending, unique, = the L2 bits (P10)
    # events = interval merge of the closed seed windows (R11-R13), restated on the downloaded arrays
    H = p.event_half_ps
    ts = t[seeds]
    sseg = np.searchsorted(seg, seeds, side="right") - 1
    head = np.ones(len(seeds), dtype=bool)
    if len(seeds) > 1:
        head[1:] = (np.diff(ts) > 2 * H) | (np.diff(sseg) != 0)
    first = np.nonzero(head)[0]
    last = np.append(first[1:], len(seeds)) - 1
    assert len(events) == len(first)
    assert (events["seed_begin"] == first).all() and (events["n_seeds"] == last - first + 1).all()
    assert (events["t_start"] == ts[first] - H).all() and (events["t_end"] == ts[last] + H).all()
    hb, he = np.empty(len(first), dtype=np.int64), np.empty(len(first), dtype=np.int64)
    for s in np.unique(sseg[first]):
        a, b = seg[s], seg[s + 1]
        m = sseg[first] == s
        hb[m] = a + np.searchsorted(t[a:b], ts[first][m] - H, side="left")
        he[m] = a + np.searchsorted(t[a:b], ts[last][m] + H, side="right")
    assert (events["hit_begin"] == hb).all() and (events["hit_end"] == he).all()
    tag = np.zeros(n + 1, dtype=np.int32)
    np.add.at(tag, hb, 1)
    np.add.at(tag, he, -1)
    assert (inevt == (np.cumsum(tag)[:n] > 0)).all()

    # ---- sampled windows against the oracle --------------------------------------------------------------
    rng = np.random.default_rng(1000 + cfg)
    tin = w.hits["t_ps"]
    n_seg = len(seg) - 1
    compared = 0
    for k in range(N_WINDOWS):
        s = int(rng.integers(0, n_seg))
        a, b = seg[s], seg[s + 1]
        seg_t = tin[a:b]
        in_seg_tracks = seg_t[w.track_id[a:b] >= 0]
        if k % 2 == 0 and len(in_seg_tracks):
            c = int(in_seg_tracks[rng.integers(0, len(in_seg_tracks))])  # around an injected track
        else:
            c = int(seg_t[rng.integers(0, len(seg_t))])
        lo_t, hi_t = c - INTERIOR_PS - HALO_PS, c + INTERIOR_PS + HALO_PS
        sel = (seg_t >= lo_t) & (seg_t <= hi_t)
        chunk = np.ascontiguousarray(w.hits[a:b][sel])  # input order = run-major: the oracle's stable order
        rank = int(a + np.count_nonzero(seg_t < lo_t))
        m = len(chunk)
        cseg = np.array([0, m], dtype=np.uint32)
        osrt, _ = oracle.sort(chunk, cseg)
        assert srt[rank:rank + m].tobytes() == osrt.tobytes(), f"window {k}: sorted records differ"
        tr = oracle.trigger(osrt, cseg, **geo_args(g), **params_kw(p))
        ofl = tr.flags.copy()
        oracle.events(osrt, cseg, tr.seeds, event_half_ps=p.event_half_ps, flags=ofl)
        ot = osrt["t_ps"]
        # interior: what the halo decides; the slice ends need no halo on their own side
        i0 = 0 if lo_t <= seg_t.min() else int(np.searchsorted(ot, c - INTERIOR_PS, side="left"))
        i1 = m if hi_t >= seg_t.max() else int(np.searchsorted(ot, c + INTERIOR_PS, side="right"))
        assert i1 > i0
        bad = np.nonzero(flags[rank + i0:rank + i1] != ofl[i0:i1])[0]
        assert len(bad) == 0, (k, bad[:8], flags[rank + i0:rank + i1][bad[:8]], ofl[i0:i1][bad[:8]])
        oseeds = tr.seeds[(tr.seeds >= i0) & (tr.seeds < i1)].astype(np.int64) + rank
        gseeds = seeds[(seeds >= rank + i0) & (seeds < rank + i1)].astype(np.int64)
        assert (oseeds == gseeds).all() if len(oseeds) == len(gseeds) else False
        compared += i1 - i0
    assert compared > 0

    # ---- the whole input through the oracle, every byte ---------------------------------------------------
    o_srt, o_perm = oracle.sort(w.hits, w.seg_offsets)
    assert srt.tobytes() == o_srt.tobytes(), "sorted records differ from the oracle"
    assert perm.tobytes() == o_perm.tobytes(), "permutation differs from the oracle (stability of ties)"
    del perm, o_perm
    tr = oracle.trigger(o_srt, w.seg_offsets, **geo_args(g), **params_kw(p))
    assert tr.status == 0
    o_flags = tr.flags.copy()
    o_ev = oracle.events(o_srt, w.seg_offsets, tr.seeds, event_half_ps=p.event_half_ps, flags=o_flags)
    bad = np.nonzero(flags != o_flags)[0]
    assert len(bad) == 0, (len(bad), bad[:8], flags[bad[:8]], o_flags[bad[:8]])
    assert len(seeds) == len(tr.seeds) and seeds.tobytes() == tr.seeds.tobytes(), "seed list differs"
    assert len(events) == len(o_ev) and events.tobytes() == o_ev.tobytes(), "event array differs"
    assert len(seeds) > 0 and len(events) > 0
