"""Directed boundary cases (SURVEY.md sect. 8(c) "Directed boundary tests"): hand-built inputs of a
few hits with the expected output written by hand.  Each pins one inclusive / exclusive choice of
the readings R1-R13 in DESIGN.md.  Used twice: against the oracle (tests/test_oracle_directed.py,
CPU) and against the CUDA path (tests/test_gpu_parity.py).

A case is a dict: hits rows (t_ps, pmt_id, floor, charge) in INPUT order, seg offsets, a dense
(P,P) table, parameter overrides, and `expect`: any of
  order   -- input indices in sorted order (the stable permutation)
  flags   -- per sorted hit, full flag byte (Q=1 LC=2 L1=4 L2STAR=8 L2=16 INEVT=32)
  seeds   -- sorted-array indices
  events  -- list of (t_start, t_end, hit_begin, hit_end, seed_begin, n_seeds)
"""
from __future__ import annotations

import numpy as np

Q, LC, L1, STAR, L2, EV = 1, 2, 4, 8, 16, 32
H = 3_000_000
W = 3_000_000


def _table(P, fill=100_000, diag=20_000):
    t = np.full((P, P), fill, dtype=np.int32)
    np.fill_diagonal(t, diag)
    return t


def directed_cases():
    cs = []

    # --- R3: charge = Q-1 and Q; one PMT only: no LC possible (R5) -------------------------------
    cs.append(dict(
        name="charge_threshold_inclusive",
        rows=[(1000, 0, 0, 299), (2000, 0, 0, 300), (3000, 0, 0, 301)],
        seg=[0, 3], table=_table(4), params=dict(l2_multiplicity=4),
        expect=dict(order=[0, 1, 2], flags=[0, Q | L1, Q | L1], seeds=[], events=[])))

    # --- R4: same-floor pair at exactly LC and at LC+1; R5 same-PMT pair never LC ----------------
    cs.append(dict(
        name="lc_window_inclusive",
        rows=[(0, 0, 0, 100), (20_000, 1, 0, 100),          # dt = LC      -> both LC
              (1_000_000, 0, 0, 100), (1_020_001, 1, 0, 100),  # dt = LC+1 -> none
              (2_000_000, 2, 0, 100), (2_010_000, 2, 0, 100),  # same PMT  -> none (R5)
              (3_000_000, 0, 0, 100), (3_010_000, 4, 1, 100)],  # other floor -> none (R6)
        seg=[0, 8], table=_table(8), params=dict(l2_multiplicity=4),
        expect=dict(flags=[LC | L1, LC | L1, 0, 0, 0, 0, 0, 0], seeds=[])))

    # --- R2: all hits share one timestamp: stable order = input order; LC all-to-all --------------
    cs.append(dict(
        name="all_equal_timestamps",
        rows=[(5000, p % 4, 0, 100) for p in range(12)],
        seg=[0, 12], table=_table(4), params=dict(l2_multiplicity=13),
        expect=dict(order=list(range(12)), flags=[LC | L1] * 12, seeds=[])))

    # --- R8: same-PMT pair gives an L2 edge through the table diagonal (20 ns), not an LC ---------
    cs.append(dict(
        name="same_pmt_diagonal_edge",
        rows=[(0, 3, 0, 400), (20_000, 3, 0, 400), (5_000_000, 3, 0, 400), (5_020_001, 3, 0, 400)],
        seg=[0, 4], table=_table(4), params=dict(l2_multiplicity=2),
        # seeds at 0 and 20 000 -> event [-H, 20 000 + H] = [-3.0, 3.02] us; hit 2 at 5.0 us is outside
        expect=dict(flags=[Q | L1 | STAR | L2 | EV, Q | L1 | STAR | L2 | EV, Q | L1, Q | L1],
                    seeds=[0, 1],
                    events=[(-H, 20_000 + H, 0, 2, 0, 2)])))

    # --- pair at dt = dtmax and dtmax+1; dtmax = -1 pair ----------------------------------------
    t = _table(4, fill=50_000)
    t[2, 3] = t[3, 2] = -1
    cs.append(dict(
        name="dtmax_inclusive_and_unconnected",
        rows=[(0, 0, 0, 400), (50_000, 1, 1, 400),                    # dt = dtmax   -> edge
              (10_000_000, 0, 0, 400), (10_050_001, 1, 1, 400),        # dt = dtmax+1 -> none
              (20_000_000, 2, 2, 400), (20_000_010, 3, 3, 400)],       # dtmax = -1   -> none
        seg=[0, 6], table=t, params=dict(l2_multiplicity=2),
        expect=dict(flags=[Q | L1 | STAR | L2 | EV, Q | L1 | STAR | L2 | EV, Q | L1, Q | L1, Q | L1, Q | L1],
                    seeds=[0, 1], events=[(-H, 50_000 + H, 0, 2, 0, 2)])))

    # --- R7: a path a-b-c-d is a star for b,c (N=3) but holds no 3-clique ------------------------
    # hits 40 us apart in pairs cannot be edges: table = 45 000 everywhere; times 0, 40k, 80k, 120k ps
    cs.append(dict(
        name="star_not_clique_path",
        rows=[(0, 0, 0, 400), (40_000, 1, 1, 400), (80_000, 2, 2, 400), (120_000, 3, 3, 400)],
        seg=[0, 4], table=_table(4, fill=45_000), params=dict(l2_multiplicity=3, l2_mode=0),
        expect=dict(flags=[Q | L1, Q | L1 | STAR, Q | L1 | STAR, Q | L1], seeds=[], events=[])))
    cs.append(dict(
        name="star_mode_path",
        rows=[(0, 0, 0, 400), (40_000, 1, 1, 400), (80_000, 2, 2, 400), (120_000, 3, 3, 400)],
        seg=[0, 4], table=_table(4, fill=45_000), params=dict(l2_multiplicity=3, l2_mode=1),
        expect=dict(flags=[Q | L1 | EV, Q | L1 | STAR | L2 | EV, Q | L1 | STAR | L2 | EV, Q | L1 | EV], seeds=[1, 2],
                    events=[(40_000 - H, 80_000 + H, 0, 4, 0, 2)])))
    # a triangle is a 3-clique
    cs.append(dict(
        name="triangle_clique",
        rows=[(0, 0, 0, 400), (40_000, 1, 1, 400), (45_000, 2, 2, 400), (9_000_000, 3, 3, 400)],
        seg=[0, 4], table=_table(4, fill=45_000), params=dict(l2_multiplicity=3),
        expect=dict(flags=[Q | L1 | STAR | L2 | EV] * 3 + [Q | L1], seeds=[0, 1, 2],
                    events=[(-H, 45_000 + H, 0, 3, 0, 3)])))

    # --- N larger than the number of hits ---------------------------------------------------------
    cs.append(dict(
        name="multiplicity_larger_than_n",
        rows=[(0, 0, 0, 400), (10, 1, 1, 400), (20, 2, 2, 400)],
        seg=[0, 3], table=_table(4), params=dict(l2_multiplicity=9),
        expect=dict(flags=[Q | L1] * 3, seeds=[], events=[])))

    # --- R12: seeds exactly 2H apart merge, 2H+1 apart do not; R13 hit exactly at t_seed +- H -----
    cs.append(dict(
        name="event_merge_gap_inclusive",
        rows=[(10_000_000 - H, 5, 1, 100),          # hit exactly at t_seed0 - H   -> inside (closed)
              (10_000_000 - H - 1, 6, 2, 100),      # one ps earlier               -> outside
              (10_000_000, 0, 0, 400),              # seed 0
              (10_000_000 + 2 * H, 0, 0, 400),      # seed 1: gap = 2H   -> same event
              (10_000_000 + 4 * H + 1, 0, 0, 400),  # seed 2: gap = 2H+1 -> new event
              (10_000_000 + 5 * H + 1, 7, 3, 100),  # exactly t_seed2 + H          -> inside
              (10_000_000 + 5 * H + 2, 7, 3, 100)],  # one ps later                 -> outside
        seg=[0, 7], table=_table(8), params=dict(l2_multiplicity=1),
        expect=dict(order=[1, 0, 2, 3, 4, 5, 6],
                    flags=[0, EV, Q | L1 | STAR | L2 | EV, Q | L1 | STAR | L2 | EV, Q | L1 | STAR | L2 | EV, EV, 0],
                    seeds=[2, 3, 4],
                    events=[(10_000_000 - H, 10_000_000 + 3 * H, 1, 4, 0, 2),
                            (10_000_000 + 3 * H + 1, 10_000_000 + 5 * H + 1, 4, 6, 2, 1)])))

    # --- two segments whose hits would coincide if merged: no cross-segment LC / L2 / event -------
    cs.append(dict(
        name="segments_are_independent",
        rows=[(100, 0, 0, 100), (500_000, 2, 1, 400),      # segment 0
              (110, 1, 0, 100), (500_010, 3, 1, 400)],     # segment 1 (same floor, 10 ps away)
        seg=[0, 2, 4], table=_table(4), params=dict(l2_multiplicity=2),
        expect=dict(order=[0, 1, 2, 3], flags=[0, Q | L1, 0, Q | L1], seeds=[], events=[])))
    cs.append(dict(
        name="segments_merged_do_coincide",
        rows=[(100, 0, 0, 100), (500_000, 2, 1, 400), (110, 1, 0, 100), (500_010, 3, 1, 400)],
        seg=[0, 4], table=_table(4), params=dict(l2_multiplicity=2),
        # merged: (r0, r2) are a same-floor pair 10 ps apart, (r1, r3) too; both pairs are L2 edges
        expect=dict(order=[0, 2, 1, 3],
                    flags=[LC | L1 | STAR | L2 | EV, LC | L1 | STAR | L2 | EV, Q | LC | L1 | STAR | L2 | EV,
                           Q | LC | L1 | STAR | L2 | EV], seeds=[0, 1, 2, 3],
                    events=[(100 - H, 500_010 + H, 0, 4, 0, 4)])))
    # an event per segment, seeds at the same time: never merged across the boundary (R13)
    cs.append(dict(
        name="events_do_not_cross_segments",
        rows=[(0, 0, 0, 400), (10, 1, 1, 400), (5, 0, 0, 400), (15, 1, 1, 400)],
        seg=[0, 2, 4], table=_table(4), params=dict(l2_multiplicity=2),
        expect=dict(flags=[Q | L1 | STAR | L2 | EV] * 4, seeds=[0, 1, 2, 3],
                    events=[(-H, 10 + H, 0, 2, 0, 2), (5 - H, 15 + H, 2, 4, 2, 2)])))

    # --- R1: negative and > 2^40 timestamps; t_start / t_end unclipped ---------------------------
    big = 1 << 45
    cs.append(dict(
        name="negative_and_large_timestamps",
        rows=[(big + 10, 1, 0, 400), (-big, 0, 0, 400), (big, 0, 0, 400), (-big + 15_000, 1, 0, 100)],
        seg=[0, 4], table=_table(4), params=dict(l2_multiplicity=2),
        expect=dict(order=[1, 3, 2, 0],
                    flags=[Q | LC | L1 | STAR | L2 | EV, LC | L1 | STAR | L2 | EV, Q | LC | L1 | STAR | L2 | EV,
                           Q | LC | L1 | STAR | L2 | EV],
                    seeds=[0, 1, 2, 3],
                    events=[(-big - H, -big + 15_000 + H, 0, 2, 0, 2), (big - H, big + 10 + H, 2, 4, 2, 2)])))

    # --- R1: a span of 2^63 ps between two clusters: t_hi - t_lo does not fit int64 (unsigned differences) ----
    big2 = 1 << 62
    cs.append(dict(
        name="span_2_63_between_clusters",
        rows=[(big2 + 10, 1, 0, 400), (-big2, 0, 0, 400), (big2, 0, 0, 400), (-big2 + 15_000, 1, 0, 100)],
        seg=[0, 4], table=_table(4), params=dict(l2_multiplicity=2),
        expect=dict(order=[1, 3, 2, 0],
                    flags=[Q | LC | L1 | STAR | L2 | EV, LC | L1 | STAR | L2 | EV, Q | LC | L1 | STAR | L2 | EV,
                           Q | LC | L1 | STAR | L2 | EV],
                    seeds=[0, 1, 2, 3],
                    events=[(-big2 - H, -big2 + 15_000 + H, 0, 2, 0, 2), (big2 - H, big2 + 10 + H, 2, 4, 2, 2)])))

    # --- R1 / R13: hits at both ends of int64: the span is 2^64 - 1, and t_start / t_end (unclipped) leave int64 --
    # reported modulo 2^64, while the hit ranges follow the exact (unwrapped) window
    lo64, hi64 = -(1 << 63), (1 << 63) - 1
    cs.append(dict(
        name="int64_extremes_windows_wrap",
        rows=[(hi64, 1, 1, 400), (lo64, 0, 0, 400), (hi64 - 10, 0, 0, 400), (lo64 + 10, 1, 1, 400)],
        seg=[0, 4], table=_table(4), params=dict(l2_multiplicity=2),
        expect=dict(order=[1, 3, 2, 0],
                    flags=[Q | L1 | STAR | L2 | EV] * 4,
                    seeds=[0, 1, 2, 3],
                    events=[(lo64 - H + (1 << 64), lo64 + 10 + H, 0, 2, 0, 2),
                            (hi64 - 10 - H, hi64 + H - (1 << 64), 2, 4, 2, 2)])))

    # --- R9: the window binds before the table ----------------------------------------------------
    cs.append(dict(
        name="l2_window_binds",
        rows=[(0, 0, 0, 400), (30_000, 1, 1, 400), (30_001 + 30_000, 2, 2, 400)],
        seg=[0, 3], table=_table(4, fill=100_000), params=dict(l2_multiplicity=2, l2_window_ps=30_000),
        expect=dict(flags=[Q | L1 | STAR | L2 | EV, Q | L1 | STAR | L2 | EV, Q | L1 | EV], seeds=[0, 1])))

    # --- empty input and single hit ---------------------------------------------------------------
    cs.append(dict(name="empty", rows=[], seg=[0, 0], table=_table(4), params=dict(l2_multiplicity=2),
                   expect=dict(order=[], flags=[], seeds=[], events=[])))
    cs.append(dict(name="single_hit_n1", rows=[(7, 0, 0, 400)], seg=[0, 1], table=_table(4),
                   params=dict(l2_multiplicity=1),
                   expect=dict(order=[0], flags=[Q | L1 | STAR | L2 | EV], seeds=[0], events=[(7 - H, 7 + H, 0, 1, 0, 1)])))
    cs.append(dict(name="empty_segment_between", rows=[(7, 0, 0, 400), (9, 0, 0, 400)], seg=[0, 1, 1, 2],
                   table=_table(4), params=dict(l2_multiplicity=1),
                   expect=dict(order=[0, 1], seeds=[0, 1],
                               events=[(7 - H, 7 + H, 0, 1, 0, 1), (9 - H, 9 + H, 1, 2, 1, 1)])))

    return cs


def case_arrays(c):
    from paper_1411_3968_b200 import workload as Wl

    rows = c["rows"]
    h = np.zeros(len(rows), dtype=Wl.HIT_DTYPE)
    for k, r in enumerate(rows):
        h[k] = (r[0], r[1], r[2], r[3], (k * 257 + 1) & 0xFFFF)
    seg = np.asarray(c["seg"], dtype=np.uint32)
    return h, seg
