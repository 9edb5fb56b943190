"""Pin for DESIGN.md reading R1 ("timestamps are any int64"): oracle_trigger and oracle_events on clusters of hits
placed at -2^62, +2^62 and at both ends of the int64 range, against the brute-force checkers of oracle/brute.py, which
compute every time difference with Python integers (no width).  A signed 64-bit subtraction anywhere in the oracle's
L1 / L2 / event code gives a wrong neighbour, edge or merge here (the spans between clusters are 2^63 .. 2^64 - 1)."""
import numpy as np

import oracle
from oracle import brute
from paper_1411_3968_b200 import workload as W
from util import geo_args

F_Q, F_LC, F_L1, F_STAR, F_L2, F_EV = 1, 2, 4, 8, 16, 32
LO64, HI64 = -(1 << 63), (1 << 63) - 1


def _clusters(seed, per=7):
    geo = W.make_geometry("nemo")
    rng = np.random.default_rng(seed)
    bases = [LO64, -(1 << 62), -40_000, (1 << 62), HI64 - 200_000]
    t, pm = [], []
    for b in bases:
        t += [int(b) + int(x) for x in rng.integers(0, 200_000, size=per)]
        pm += [int(x) for x in rng.integers(0, geo.n_pmt, size=per)]
    n = len(t)
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["t_ps"] = np.array(t, dtype=np.int64)
    h["pmt_id"] = pm
    h["floor"] = geo.floor[h["pmt_id"]]
    h["charge"] = np.where(rng.random(n) < 0.7, 400, 100)
    o = rng.permutation(n)
    return geo, h[o]


def test_extreme_timestamps_against_brute_force(oracle_lib):
    for seed in range(8):
        geo, h = _clusters(seed)
        n = len(h)
        seg = np.array([0, n], dtype=np.uint32) if seed % 2 == 0 else np.array([0, n // 3, n], dtype=np.uint32)
        srt, _ = oracle.sort(h, seg)
        N = 2 + seed % 3
        tr = oracle.trigger(srt, seg, **geo_args(geo), l2_multiplicity=N, lc_window_ps=20_000, q_thresh=300)
        assert ((tr.flags & 7) == brute.l1_flags(srt, seg, 300, 20_000)).all()
        l1 = (tr.flags & F_L1) != 0
        star, clique = brute.l2_flags(srt, seg, l1, geo.dense_table(), 3_000_000, N)
        assert (((tr.flags & F_STAR) != 0) == star).all()
        assert (((tr.flags & F_L2) != 0) == clique).all()
        assert clique.any()
        flags = tr.flags.copy()
        Hh = 3_000_000
        ev = oracle.events(srt, seg, tr.seeds, event_half_ps=Hh, flags=flags)
        sg = brute.seg_id(n, seg)
        t = [int(x) for x in srt["t_ps"]]
        ref = brute.event_groups([t[s] for s in tr.seeds], sg[tr.seeds], Hh)
        assert len(ev) == len(ref)
        for e, (s, t0, t1, members) in zip(ev, ref):
            # reported bounds: the exact values modulo 2^64 (R13: unclipped)
            assert (int(e["t_start"]) - t0) % (1 << 64) == 0 and (int(e["t_end"]) - t1) % (1 << 64) == 0
            assert list(range(int(e["seed_begin"]), int(e["seed_begin"]) + int(e["n_seeds"]))) == members
            inside = [i for i in range(n) if sg[i] == s and t0 <= t[i] <= t1]
            assert int(e["hit_begin"]) == inside[0] and int(e["hit_end"]) == inside[-1] + 1
        want = np.array([any(sg[s] == sg[i] and abs(t[s] - t[i]) <= Hh for s in tr.seeds) for i in range(n)])
        assert (((flags & F_EV) != 0) == want).all()
