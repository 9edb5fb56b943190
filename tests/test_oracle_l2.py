"""Pins P6 / P7 / P8 for the L2 part of oracle_trigger."""
import numpy as np
import pytest

import oracle
from oracle import brute
from paper_1411_3968_b200 import workload as W
from util import geo_args, single_tower_geo

F_L1, F_STAR, F_L2 = 4, 8, 16


def _cluster_case(seed, n, span_ps, geo, n_seg=1):
    """n hits, all L1 through the Q bit, random PMTs, random times in a short span."""
    rng = np.random.default_rng(seed)
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, geo.n_pmt, size=n)
    h["floor"] = geo.floor[h["pmt_id"]]
    h["charge"] = np.where(rng.random(n) < 0.8, 400, 100)
    h["t_ps"] = rng.integers(0, span_ps, size=n)
    seg = np.array([0, n], dtype=np.uint32) if n_seg == 1 else np.array([0, n // 2, n], dtype=np.uint32)
    srt, _ = oracle.sort(h, seg)
    return srt, seg


@pytest.mark.parametrize("kind,N", [("nemo", 4), ("km3", 5), ("km3", 3), ("nemo", 2)])
def test_l2_brute_force_p6(kind, N, oracle_lib):
    geo = W.make_geometry(kind)
    table = geo.dense_table()
    seen = [0, 0, 0]
    for seed in range(6):
        span = (400_000, 900_000, 2_000_000, 5_000_000)[seed % 4]
        srt, seg = _cluster_case(seed + 10 * N, 22, span, geo, n_seg=1 + seed % 2)
        for mode in (0, 1):
            tr = oracle.trigger(srt, seg, **geo_args(geo), l2_multiplicity=N, l2_mode=mode, lc_window_ps=20_000)
            l1 = (tr.flags & F_L1) != 0
            star, clique = brute.l2_flags(srt, seg, l1, table, 3_000_000, N)
            assert (((tr.flags & F_STAR) != 0) == star).all()
            assert (((tr.flags & F_L2) != 0) == (clique if mode == 0 else star)).all()
            assert (tr.seeds == np.nonzero(tr.flags & F_L2)[0]).all()
        seen[0] += int(star.sum()); seen[1] += int(clique.sum()); seen[2] += int((star & ~clique).sum())
    assert seen[0] > 0 and seen[1] > 0  # both outcomes occur
    if N > 3:
        assert seen[2] > 0  # stars that are not cliques occur (R7 matters)


def test_l2_window_binds(oracle_lib):
    """min(dtmax, W): with W smaller than the table the window is what limits the edge (R9)."""
    geo = W.make_geometry("km3")
    table = geo.dense_table()
    srt, seg = _cluster_case(77, 20, 1_500_000, geo)
    tr = oracle.trigger(srt, seg, **geo_args(geo), l2_multiplicity=3, l2_window_ps=150_000)
    star, clique = brute.l2_flags(srt, seg, (tr.flags & F_L1) != 0, table, 150_000, 3)
    assert (((tr.flags & F_L2) != 0) == clique).all() and clique.any()
    tr_big = oracle.trigger(srt, seg, **geo_args(geo), l2_multiplicity=3)
    assert ((tr_big.flags & F_L2) != 0).sum() > clique.sum()


def test_l2_special_cases_p7(oracle_lib):
    geo = W.make_geometry("km3")
    w = W.make_config(1, time_scale=0.02)
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ga = geo_args(geo)
    # N = 1: L2 == L1
    tr = oracle.trigger(srt, w.seg_offsets, **ga, l2_multiplicity=1)
    assert (((tr.flags & F_L2) != 0) == ((tr.flags & F_L1) != 0)).all()
    # N = 2: clique == star == "has at least one edge"
    a = oracle.trigger(srt, w.seg_offsets, **ga, l2_multiplicity=2, l2_mode=0)
    b = oracle.trigger(srt, w.seg_offsets, **ga, l2_multiplicity=2, l2_mode=1)
    assert (a.flags == b.flags).all() and (((a.flags & F_L2) != 0) == ((a.flags & F_STAR) != 0)).all()
    assert len(a.seeds) > 0


@pytest.mark.parametrize("N,C", [(3, 150_000), (5, 700_000), (7, 1_000_000)])
def test_l2_constant_table_is_n_in_tw_p7(N, C, oracle_lib):
    """Constant table C: clique == the paper's N-in-TW sliding test on the L1 list,
    t[k+N-1] - t[k] <= C for some window containing i (PAPER.md:59 with DESIGN.md reading R14)."""
    P = 84
    geo = single_tower_geo(np.full((P, P), C, dtype=np.int32))
    w = W.make_config(2, time_scale=0.002)  # burst density: plenty of L1 hits
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    tr = oracle.trigger(srt, w.seg_offsets, **geo_args(geo), l2_multiplicity=N)
    l1 = np.nonzero(tr.flags & F_L1)[0]
    t = srt["t_ps"][l1]
    ok = np.zeros(len(l1), dtype=bool)
    for k in range(len(l1) - N + 1):
        if t[k + N - 1] - t[k] <= C:
            ok[k:k + N] = True
    got = ((tr.flags & F_L2) != 0)[l1]
    assert (got == ok).all() and ok.any() and not ok.all()


def test_l2_invariants_p8(oracle_lib):
    w = W.make_config(2, time_scale=0.003)
    geo = w.geometry
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ga = geo_args(geo)
    base = oracle.trigger(srt, w.seg_offsets, **ga, l2_multiplicity=4)
    f = base.flags
    l1, st, l2 = (f & F_L1) != 0, (f & F_STAR) != 0, (f & F_L2) != 0
    assert (l2 <= st).all() and (st <= l1).all() and l2.any() and (st & ~l2).any()
    # monotone in N, in the window and in the table
    f5 = oracle.trigger(srt, w.seg_offsets, **ga, l2_multiplicity=5).flags
    assert (((f5 & F_L2) != 0) <= l2).all() and (((f5 & F_STAR) != 0) <= st).all()
    fw = oracle.trigger(srt, w.seg_offsets, **ga, l2_multiplicity=4, l2_window_ps=300_000).flags
    assert (((fw & F_L2) != 0) <= l2).all()
    ga_small = dict(ga, blocks=np.maximum(ga["blocks"] // 2, 0))
    fs = oracle.trigger(srt, w.seg_offsets, **ga_small, l2_multiplicity=4).flags
    assert (((fs & F_L2) != 0) <= l2).all() and ((fs & F_L2) != 0).sum() < l2.sum()
    # time translation changes nothing
    sh = srt.copy()
    sh["t_ps"] += 123_456_789_012_345
    assert (oracle.trigger(sh, w.seg_offsets, **ga, l2_multiplicity=4).flags == f).all()
    sh["t_ps"] -= 2 * 123_456_789_012_345  # negative times
    assert (oracle.trigger(sh, w.seg_offsets, **ga, l2_multiplicity=4).flags == f).all()
    # relabelling PMTs with the table permuted changes nothing
    rng = np.random.default_rng(5)
    pi = rng.permutation(geo.n_pmt)  # old id -> new id
    rel = srt.copy()
    rel["pmt_id"] = pi[srt["pmt_id"]]
    tab = geo.dense_table()
    inv = np.argsort(pi)
    geo2 = single_tower_geo(tab[np.ix_(inv, inv)])
    assert (oracle.trigger(rel, w.seg_offsets, **geo_args(geo2), l2_multiplicity=4).flags == f).all()
    # dtmax = -1 everywhere: no edges, no L2 (but N=1 still gives L2 = L1)
    geo3 = single_tower_geo(np.full((84, 84), -1, dtype=np.int32))
    f3 = oracle.trigger(srt, w.seg_offsets, **geo_args(geo3), l2_multiplicity=2).flags
    assert not (f3 & (F_L2 | F_STAR)).any()


def test_l2_multitower_block_table(oracle_lib):
    """cfg4 geometry: the block-sparse lookup equals a dense table built independently from positions."""
    w = W.make_config(4, time_scale=0.0004)
    geo = w.geometry
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    tr = oracle.trigger(srt, w.seg_offsets, **geo_args(geo), l2_multiplicity=3)
    l1 = np.nonzero(tr.flags & F_L1)[0]
    pos, tow = geo.pos, geo.tower
    org = pos[::84][:, :2]  # tower origins + local x of pmt 0 (same offset for every tower)
    t = srt["t_ps"][l1].astype(np.int64); pm = srt["pmt_id"][l1].astype(np.int64)
    m = len(l1)
    deg = np.zeros(m, dtype=np.int64)
    adj = np.zeros((m, m), dtype=bool)
    for a in range(m):
        d = np.linalg.norm(pos[pm] - pos[pm[a]], axis=1)
        lim = np.rint((d * 1.35 / 299792458.0 + 20e-9) * 1e12).astype(np.int64)
        far = np.linalg.norm(org[tow[pm]] - org[tow[pm[a]]], axis=1) > 300.0 + 1e-9
        e = (np.abs(t - t[a]) <= np.minimum(lim, 3_000_000)) & ~far
        e[a] = False
        adj[a] = e
    star = adj.sum(1) >= 2
    tri = ((adj.astype(np.int64) @ adj.astype(np.int64)) * adj).sum(1) > 0  # in a triangle
    assert (((tr.flags & F_STAR) != 0)[l1] == star).all()
    assert (((tr.flags & F_L2) != 0)[l1] == tri).all()
    assert tri.any() and m > 100
