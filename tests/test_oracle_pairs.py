"""Pins P18-P22 for oracle_pair_seeds (SC / FC / AFC) and oracle_l0_combine."""
import math

import numpy as np
import pytest

import oracle
from oracle import brute
from paper_1411_3968_b200 import workload as W
from util import geo_args, mk_hits

SC, FC, AFC, CAND_A, CAND_B = 1, 2, 4, 8, 16


def _cluster(seed, n, span_ps, geo, n_seg=1):
    rng = np.random.default_rng(seed)
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, geo.n_pmt, size=n)
    h["floor"] = geo.floor[h["pmt_id"]]
    h["charge"] = 100
    h["t_ps"] = rng.integers(0, span_ps, size=n) - span_ps // 2
    seg = np.array([0, n], dtype=np.uint32) if n_seg == 1 else np.array([0, n // 2, n // 2, n], dtype=np.uint32)
    srt, _ = oracle.sort(h, seg)
    return srt, seg


@pytest.mark.parametrize("kind,nx", [("nemo", 1), ("km3", 1), ("km3", 2)])
def test_pair_seeds_brute_force_p18(kind, nx, oracle_lib):
    """P18: all ordered pairs (oracle/brute.py); two towers exercise the same-tower conditions of SC and AFC."""
    geo = W.make_geometry(kind, nx=nx)
    adj, ppt = geo.adjacency(), geo.pmts_per_tower
    seen = 0
    for seed in range(6):
        srt, seg = _cluster(seed, 60, (400_000, 2_000_000, 6_000_000)[seed % 3], geo, n_seg=1 + seed % 2)
        for w in [(20_000, 100_000, 250_000), (250_000, 20_000, 100_000), (0, 0, 0)]:
            got = oracle.pair_seeds(srt, seg, ppt, adj, sc_window_ps=w[0], fc_window_ps=w[1], afc_window_ps=w[2])
            ref = brute.pair_seeds(srt, seg, ppt, adj, *w)
            assert (got == ref).all()
            seen |= int(np.bitwise_or.reduce(ref)) if len(ref) else 0
    assert seen == SC | FC | AFC  # every rule fired somewhere


def test_pair_seeds_directed_p19(oracle_lib):
    """P19: hand-written cases on the KM3NeT-It tower (6 PMTs per floor on a bar; floor = pmt // 6)."""
    geo = W.make_geometry("km3", nx=2)
    adj, ppt = geo.adjacency(), geo.pmts_per_tower
    one = lambda n: np.array([0, n], dtype=np.uint32)
    run = lambda rows, seg=None: oracle.pair_seeds(mk_hits(rows), seg if seg is not None else one(len(rows)), ppt,
                                                   adj).tolist()
    # PMTs 0 and 1: adjacent on floor 0.  dt = 20 ns: SC and FC; 20 ns + 1 ps: FC only; 100 ns + 1 ps: nothing
    assert run([(0, 0, 0, 0), (20_000, 1, 0, 0)]) == [SC | FC, SC | FC]
    assert run([(0, 0, 0, 0), (20_001, 1, 0, 0)]) == [FC, FC]
    assert run([(0, 0, 0, 0), (100_000, 1, 0, 0)]) == [FC, FC]
    assert run([(0, 0, 0, 0), (100_001, 1, 0, 0)]) == [0, 0]
    # PMTs 0 and 2: same floor, not adjacent
    assert run([(0, 0, 0, 0), (5_000, 2, 0, 0)]) == [FC, FC]
    # the same PMT twice: no rule ("two PMTs")
    assert run([(0, 0, 0, 0), (5_000, 0, 0, 0)]) == [0, 0]
    # floors 0 and 1 of one tower: AFC up to 250 ns inclusive; floors 0 and 2: nothing
    assert run([(0, 0, 0, 0), (250_000, 6, 1, 0)]) == [AFC, AFC]
    assert run([(0, 0, 0, 0), (250_001, 6, 1, 0)]) == [0, 0]
    assert run([(0, 0, 0, 0), (1_000, 12, 2, 0)]) == [0, 0]
    # last floor of tower 0 (global floor 13) and first floor of tower 1 (global floor 14): consecutive ids, other tower
    assert run([(0, 78, 13, 0), (1_000, 84, 14, 0)]) == [0, 0]
    # PMT 0 of tower 0 and PMT 1 of tower 1: adjacent local indices, other tower
    assert run([(0, 0, 0, 0), (1_000, 85, 14, 0)]) == [0, 0]
    # never across a segment
    assert run([(0, 0, 0, 0), (1_000, 1, 0, 0)], np.array([0, 1, 2], dtype=np.uint32)) == [0, 0]
    # a partner 250 ns away is found behind a closer hit that matches nothing
    assert run([(0, 0, 0, 0), (10, 30, 5, 0), (250_000, 7, 1, 0)]) == [AFC, 0, AFC]


def test_fc_is_the_l1_coincidence_p20(oracle_lib):
    """P20: FC with the window of L1's local coincidence is the LC bit of oracle_trigger (already pinned, P4 / P5)."""
    w = W.make_config(1, time_scale=0.05)
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    g = w.geometry
    tr = oracle.trigger(srt, w.seg_offsets, **geo_args(g), lc_window_ps=20_000)
    bits = oracle.pair_seeds(srt, w.seg_offsets, g.pmts_per_tower, g.adjacency(), fc_window_ps=20_000)
    assert (((bits & FC) != 0) == ((tr.flags & 2) != 0)).all() and (bits & FC).any()


def test_pair_seed_poisson_rates_p21(oracle_lib):
    """P21: Poisson background at 55 kHz per PMT on the 84-PMT tower.  A hit is flagged by a rule with
    probability 1 - exp(-2 W R k), k = number of partner PMTs of the rule (north_star's 2 R1 R2 dt, per hit)."""
    geo = W.make_geometry("km3")
    adj, ppt = geo.adjacency(), geo.pmts_per_tower
    R, T = 55e3, 0.4
    rng = np.random.default_rng(1411)
    counts = rng.poisson(R * T, size=ppt)
    n = int(counts.sum())
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = np.repeat(np.arange(ppt), counts)
    h["floor"] = geo.floor[h["pmt_id"]]
    h["t_ps"] = rng.integers(0, int(T * 1e12), size=n)
    seg = np.array([0, n], dtype=np.uint32)
    srt, _ = oracle.sort(h, seg)
    bits = oracle.pair_seeds(srt, seg, ppt, adj)
    floors = int(geo.floor[:ppt].max()) + 1
    for bit, W_s, partners in [
        (SC, 20e-9, adj.sum(axis=1)),                                             # 1 or 2 bar neighbours
        (FC, 100e-9, np.full(ppt, 5)),                                            # the 5 other PMTs of the floor
        (AFC, 250e-9, np.where((geo.floor[:ppt] == 0) | (geo.floor[:ppt] == floors - 1), 6, 12)),
    ]:
        exp = float((counts * (1.0 - np.exp(-2.0 * W_s * R * partners))).sum())
        got = int((bits & bit).astype(bool).sum())
        assert abs(got - exp) < 5 * math.sqrt(2 * exp), (bit, got, exp)  # pairs flag two hits: variance <= 2 x Poisson


def test_l0_combine_p22(oracle_lib):
    """P22: python restatement on random bytes + a hand case."""
    rng = np.random.default_rng(3)
    for N in (1, 3, 7):
        n = 300
        l0 = np.zeros(n, dtype=np.uint8)
        l0[: n - N + 1] = rng.integers(0, 2, size=n - N + 1) * 3
        pb = (rng.integers(0, 8, size=n) * (rng.random(n) < 0.3)).astype(np.uint8)
        assert (oracle.l0_combine(l0, pb, N) == brute.l0_combine(l0, pb, N)).all()
    # window 0..2 holds SC (hit 1) and AFC (hit 2): candidate A; window 3..5 holds FC and AFC: candidate B
    l0 = np.array([3, 2, 2, 3, 2, 2, 0], dtype=np.uint8)
    pb = np.array([0, SC, AFC, FC, 0, AFC, SC | AFC], dtype=np.uint8)
    assert oracle.l0_combine(l0, pb, 3).tolist() == [CAND_A, 0, 0, CAND_B, 0, 0, 0]
    with pytest.raises(ValueError):
        oracle.l0_combine(np.array([0, 1], dtype=np.uint8), np.zeros(2, dtype=np.uint8), 3)  # start without a window
