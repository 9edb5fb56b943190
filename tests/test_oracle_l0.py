"""Pins P14-P17 for oracle_l0_ntw, the level-0 N-in-TW trigger (PAPER.md:59 'N7TW1000: looking for 7 hits in
TW = 1000 ns', PAPER.md:73 N7TW500, PAPER.md:67 'as level 0 trigger'; reading R14 / R20: t[k+N-1] - t[k] < TW)."""
import math

import numpy as np
import pytest

import oracle
from oracle import brute
from paper_1411_3968_b200 import workload as W
from util import geo_args, mk_hits, single_tower_geo

START, MEMBER = 1, 2


def _random_sorted(seed, n, span_ps, n_seg=1, ties=False):
    rng = np.random.default_rng(seed)
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, 32, size=n)
    h["charge"] = 100
    t = rng.integers(0, span_ps, size=n)
    if ties:
        t = (t // (span_ps // 12 + 1)) * (span_ps // 12 + 1)  # a dozen distinct values: many equal timestamps
    h["t_ps"] = t - span_ps // 3  # negative times too
    seg = np.array([0, n], dtype=np.uint32) if n_seg == 1 else np.array([0, n // 3, n // 3, n], dtype=np.uint32)
    srt, _ = oracle.sort(h, seg)
    return srt, seg


@pytest.mark.parametrize("N,tw", [(7, 1_000_000), (7, 500_000), (3, 200_000), (2, 50_000), (1, 1), (5, 0)])
def test_l0_brute_force_p14(N, tw, oracle_lib):
    """P14: counting formulation on time intervals (oracle/brute.py), tiny inputs, with ties and segments."""
    fired = 0
    for seed in range(8):
        srt, seg = _random_sorted(100 * N + seed, 40, (3_000_000, 800_000)[seed % 2], n_seg=1 + seed % 2,
                                  ties=seed >= 6)
        l0, ns = oracle.l0_ntw(srt, seg, multiplicity=N, window_ps=tw)
        ref = brute.l0_ntw(srt, seg, N, tw)
        assert (l0 == ref).all()
        assert ns == int((ref & START).astype(bool).sum())
        fired += ns
    assert (fired > 0) == (tw > 0)


def test_l0_directed_boundaries_p15(oracle_lib):
    """P15: hand-written cases.  Strict '<' as printed; a window never crosses a segment."""
    # 3-in-100: hits at 0, 40, 99 fire (span 99 < 100); 0, 40, 100 do not (span 100)
    seg = np.array([0, 3], dtype=np.uint32)
    l0, ns = oracle.l0_ntw(mk_hits([(0, 0, 0, 0), (40, 1, 0, 0), (99, 2, 0, 0)]), seg, multiplicity=3, window_ps=100)
    assert l0.tolist() == [START | MEMBER, MEMBER, MEMBER] and ns == 1
    l0, ns = oracle.l0_ntw(mk_hits([(0, 0, 0, 0), (40, 1, 0, 0), (100, 2, 0, 0)]), seg, multiplicity=3, window_ps=100)
    assert l0.tolist() == [0, 0, 0] and ns == 0
    # two overlapping windows: starts at 0 and 1, members 0..3, the last hit is too late
    h = mk_hits([(0, 0, 0, 0), (10, 0, 0, 0), (20, 0, 0, 0), (105, 0, 0, 0), (300, 0, 0, 0)])
    l0, ns = oracle.l0_ntw(h, np.array([0, 5], dtype=np.uint32), multiplicity=3, window_ps=100)
    assert l0.tolist() == [START | MEMBER, START | MEMBER, MEMBER, MEMBER, 0] and ns == 2
    # the same five hits cut into segments 0..1 | 2..4: no window of three inside either one
    l0, ns = oracle.l0_ntw(h, np.array([0, 2, 5], dtype=np.uint32), multiplicity=3, window_ps=100)
    assert l0.tolist() == [0] * 5 and ns == 0
    # equal timestamps: span 0 < 1
    h = mk_hits([(7, 0, 0, 0)] * 4)
    l0, ns = oracle.l0_ntw(h, np.array([0, 4], dtype=np.uint32), multiplicity=4, window_ps=1)
    assert l0.tolist() == [START | MEMBER, MEMBER, MEMBER, MEMBER] and ns == 1
    # N larger than the slice, empty slice, N = 1 (every hit is its own window when TW > 0)
    assert oracle.l0_ntw(h, np.array([0, 4], dtype=np.uint32), multiplicity=5, window_ps=10)[1] == 0
    assert oracle.l0_ntw(h[:0], np.array([0, 0], dtype=np.uint32), multiplicity=3, window_ps=10)[1] == 0
    l0, ns = oracle.l0_ntw(h, np.array([0, 4], dtype=np.uint32), multiplicity=1, window_ps=1)
    assert l0.tolist() == [START | MEMBER] * 4 and ns == 4
    # extreme timestamps: the span is taken exactly (no int64 wrap): 2^63-1 - (-2^63) is not < TW
    big = mk_hits([(-2**63, 0, 0, 0), (2**63 - 1, 0, 0, 0)])
    assert oracle.l0_ntw(big, np.array([0, 2], dtype=np.uint32), multiplicity=2, window_ps=2**63 - 1)[1] == 0


def test_l0_equals_clique_on_constant_table_p16(oracle_lib):
    """P16: with every hit L1 and a constant causality table C, 'N hits pairwise within C' is 'N consecutive hits
    spanning <= C' -- the N-in-TW test with TW = C + 1 on integer times (the paper's own form).  The two
    oracle functions share no code: oracle_trigger finds the cliques by search."""
    C = 180_000
    geo = single_tower_geo(np.full((32, 32), C, dtype=np.int32))
    for seed in range(5):
        srt, seg = _random_sorted(900 + seed, 300, 6_000_000, n_seg=1 + seed % 2)
        for N in (2, 4, 6):
            tr = oracle.trigger(srt, seg, **geo_args(geo), q_thresh=0, l2_multiplicity=N, l2_mode=0)
            l0, _ = oracle.l0_ntw(srt, seg, multiplicity=N, window_ps=C + 1)
            assert (((tr.flags & 16) != 0) == ((l0 & MEMBER) != 0)).all()
            assert (l0 & MEMBER).any()


def test_l0_poisson_rate_p17(oracle_lib):
    """P17: for a Poisson stream of rate R the span of N consecutive hits is Erlang(N-1, R), so a start fires with
    probability P(Poisson(R TW) >= N-1).  NEMO tower: 32 PMTs x 55 kHz, N7TW1000."""
    R, T, N, tw = 32 * 55e3, 0.2, 7, 1_000_000
    rng = np.random.default_rng(14113968)
    n = rng.poisson(R * T)
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["t_ps"] = np.sort(rng.integers(0, int(T * 1e12), size=n))
    l0, ns = oracle.l0_ntw(h, np.array([0, n], dtype=np.uint32), multiplicity=N, window_ps=tw)
    lam = R * tw * 1e-12
    p = 1.0 - sum(math.exp(-lam) * lam**k / math.factorial(k) for k in range(N - 1))
    exp = n * p
    # starts are positively correlated over ~N neighbours: allow 5 sigma of a variance inflated by 2N
    assert abs(ns - exp) < 5 * math.sqrt(exp * 2 * N), (ns, exp)
    assert ns == int((l0 & START).astype(bool).sum())
    assert ((l0 & START) == 0)[(l0 & MEMBER) == 0].all()  # a start is a member
