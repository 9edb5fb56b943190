"""Pins P23-P25 for oracle_l0_dntw, the distinct-PMT level-0 trigger (PAPER.md:60 'DN7TW1000: looking for 7 hits from
different PMTs within TW = 1000 ns'; reading R23)."""
import numpy as np
import pytest

import oracle
from oracle import brute
from paper_1411_3968_b200 import workload as W
from util import mk_hits

START, MEMBER = 1, 2


def _random_sorted(seed, n, span_ps, n_pmt, n_seg=1):
    rng = np.random.default_rng(seed)
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, n_pmt, size=n)
    h["t_ps"] = rng.integers(0, span_ps, size=n) - span_ps // 2
    seg = np.array([0, n], dtype=np.uint32) if n_seg == 1 else np.array([0, n // 3, n // 3, n], dtype=np.uint32)
    srt, _ = oracle.sort(h, seg)
    return srt, seg


@pytest.mark.parametrize("N,tw,n_pmt", [(7, 1_000_000, 32), (3, 300_000, 4), (2, 100_000, 2), (1, 1, 5), (4, 0, 8),
                                        (5, 2_000_000, 5)])
def test_dn_brute_force_p23(N, tw, n_pmt, oracle_lib):
    """P23: set formulation (oracle/brute.py); few PMTs so that repeated PMTs inside a window are the rule."""
    fired = 0
    for seed in range(6):
        srt, seg = _random_sorted(50 * N + seed, 40, (3_000_000, 900_000)[seed % 2], n_pmt, n_seg=1 + seed % 2)
        l0, ns = oracle.l0_dntw(srt, seg, multiplicity=N, window_ps=tw)
        ref = brute.l0_dntw(srt, seg, N, tw)
        assert (l0 == ref).all()
        assert ns == int((ref & START).astype(bool).sum())
        fired += ns
    assert (fired > 0) == (tw > 0)


def test_dn_directed_p24(oracle_lib):
    """P24: hand-written cases."""
    one = lambda n: np.array([0, n], dtype=np.uint32)
    # three hits, PMTs 0 0 1, DN2 in 100: start 0 needs the third hit (members 0..2), start 1 fires with hit 2
    h = mk_hits([(0, 0, 0, 0), (10, 0, 0, 0), (20, 1, 0, 0)])
    l0, ns = oracle.l0_dntw(h, one(3), multiplicity=2, window_ps=100)
    assert l0.tolist() == [START | MEMBER, START | MEMBER, MEMBER] and ns == 2
    # the second PMT arrives exactly at t_k + TW: strict '<', no fire; one ps earlier: fire
    h = mk_hits([(0, 0, 0, 0), (100, 1, 0, 0)])
    assert oracle.l0_dntw(h, one(2), multiplicity=2, window_ps=100)[1] == 0
    assert oracle.l0_dntw(h, one(2), multiplicity=2, window_ps=101)[0].tolist() == [START | MEMBER, MEMBER]
    # seven hits of one PMT never make DN2, whatever the window
    h = mk_hits([(i, 3, 0, 0) for i in range(7)])
    assert oracle.l0_dntw(h, one(7), multiplicity=2, window_ps=10**9)[1] == 0
    # never across a segment
    h = mk_hits([(0, 0, 0, 0), (10, 1, 0, 0)])
    assert oracle.l0_dntw(h, np.array([0, 1, 2], dtype=np.uint32), multiplicity=2, window_ps=100)[1] == 0
    # N = 1: every hit is its own window when TW > 0
    assert oracle.l0_dntw(h, one(2), multiplicity=1, window_ps=1)[0].tolist() == [START | MEMBER] * 2


def test_dn_equals_plain_when_all_pmts_differ_p25(oracle_lib):
    """P25: with a different PMT on every hit DNnTW is the pinned plain N-in-TW (P14-P17); with repeats it fires on a
    subset of the plain starts."""
    for seed in range(4):
        srt, seg = _random_sorted(300 + seed, 400, 8_000_000, 32, n_seg=1 + seed % 2)
        uniq = srt.copy()
        uniq["pmt_id"] = np.arange(len(uniq))
        for N in (2, 5, 7):
            plain, ns = oracle.l0_ntw(uniq, seg, multiplicity=N, window_ps=250_000)
            dn, nd = oracle.l0_dntw(uniq, seg, multiplicity=N, window_ps=250_000)
            assert (plain == dn).all() and ns == nd and ns > 0
            plain2, _ = oracle.l0_ntw(srt, seg, multiplicity=N, window_ps=250_000)
            dn2, _ = oracle.l0_dntw(srt, seg, multiplicity=N, window_ps=250_000)
            assert not ((dn2 & START) & ~(plain2 & START)).any()
