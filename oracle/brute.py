"""Brute-force checkers that pin oracle/tt_oracle.cpp -- TEST INFRASTRUCTURE.

Written separately from the oracle (different language, different formulation: exhaustive
pair / subset enumeration straight from the definitions in BASELINE.json:north_star) so that
a mistake cannot be shared.  Tiny inputs only (O(n^2) and O(C(n,N))).
"""
from __future__ import annotations

import itertools

import numpy as np


def seg_id(n: int, seg_offsets) -> np.ndarray:
    s = np.zeros(n, dtype=np.int64)
    for k in range(len(seg_offsets) - 1):
        s[int(seg_offsets[k]):int(seg_offsets[k + 1])] = k
    return s


def l1_flags(h: np.ndarray, seg_offsets, q_thresh: int, lc_ps: int) -> np.ndarray:
    """north_star: 'a charge-over-threshold test and a same-floor local coincidence (L1)'.
    All ordered pairs, no use of the time order."""
    n = len(h)
    sg = seg_id(n, seg_offsets)
    t = h["t_ps"].astype(object)  # python ints: no overflow
    out = np.zeros(n, dtype=np.uint8)
    for i in range(n):
        f = 1 if int(h["charge"][i]) >= q_thresh else 0
        for j in range(n):
            if j == i or sg[j] != sg[i]:
                continue
            if h["floor"][j] == h["floor"][i] and h["pmt_id"][j] != h["pmt_id"][i] and abs(t[j] - t[i]) <= lc_ps:
                f |= 2
                break
        if f:
            f |= 4
        out[i] = f
    return out


def l2_flags(h: np.ndarray, seg_offsets, l1: np.ndarray, table: np.ndarray, W: int, N: int):
    """north_star: 'at least N L1 hits pairwise satisfying |dt| <= dt_max(pmt_i, pmt_j)' within
    the <= 3 us window.  Returns (star, clique) boolean arrays by enumerating every pair and every
    N-subset of L1 hits.  table is the dense (P,P) integer table, -1 = never."""
    n = len(h)
    sg = seg_id(n, seg_offsets)
    idx = [i for i in range(n) if l1[i]]
    t = [int(x) for x in h["t_ps"]]
    pm = [int(x) for x in h["pmt_id"]]
    P = table.shape[0]

    def edge(a, b):
        if sg[a] != sg[b] or pm[a] >= P or pm[b] >= P:
            return False
        lim = int(table[pm[a], pm[b]])
        if lim < 0:
            return False
        return abs(t[a] - t[b]) <= min(lim, W)

    star = np.zeros(n, dtype=bool)
    clique = np.zeros(n, dtype=bool)
    for a in idx:
        deg = sum(1 for b in idx if b != a and edge(a, b))
        star[a] = deg >= N - 1
    if N == 1:
        clique[idx] = True
        return star, clique
    for sub in itertools.combinations(idx, N):
        if all(edge(a, b) for a, b in itertools.combinations(sub, 2)):
            clique[list(sub)] = True
    return star, clique


def event_groups(seed_t, seed_seg, H: int):
    """Union of the closed windows [t-H, t+H] of the seeds, per segment: two seeds share an event
    iff they are linked by a chain of overlapping (or touching) windows.  Union-find over all pairs.
    Returns a list of (segment, t_start, t_end, [seed positions])."""
    m = len(seed_t)
    parent = list(range(m))

    def find(x):
        while parent[x] != x:
            parent[x] = parent[parent[x]]
            x = parent[x]
        return x

    for a in range(m):
        for b in range(a + 1, m):
            # windows [ta-H, ta+H] and [tb-H, tb+H] intersect iff |ta-tb| <= 2H
            if seed_seg[a] == seed_seg[b] and abs(int(seed_t[a]) - int(seed_t[b])) <= 2 * H:
                parent[find(a)] = find(b)
    groups: dict[int, list[int]] = {}
    for a in range(m):
        groups.setdefault(find(a), []).append(a)
    out = []
    for members in groups.values():
        ts = [int(seed_t[a]) for a in members]
        out.append((int(seed_seg[members[0]]), min(ts) - H, max(ts) + H, sorted(members)))
    out.sort(key=lambda e: (e[0], e[1]))
    return out


def l0_ntw(h: np.ndarray, seg_offsets, N: int, tw_ps: int) -> np.ndarray:
    """PAPER.md:59 'looking for 7 hits in TW'.  Counting formulation on half-open time intervals, no k+N-1
    indexing: hit k is a firing start <=> at least N hits of its segment with index >= k have t < t_k + TW;
    hit i is a member <=> some hit a of its segment has t_a <= t_i < t_a + TW and at least N hits of the segment
    lie in [t_a, t_a + TW)  (the hits of such an interval are consecutive in time order, so N consecutive ones
    containing i span less than TW)."""
    n = len(h)
    sg = seg_id(n, seg_offsets)
    t = [int(x) for x in h["t_ps"]]
    out = np.zeros(n, dtype=np.uint8)
    for k in range(n):
        c = sum(1 for j in range(k, n) if sg[j] == sg[k] and t[j] < t[k] + tw_ps)
        if tw_ps > 0 and c >= N:
            out[k] |= 1
    for i in range(n):
        for a in range(n):
            if sg[a] != sg[i] or not (t[a] <= t[i] < t[a] + tw_ps):
                continue
            c = sum(1 for j in range(n) if sg[j] == sg[a] and t[a] <= t[j] < t[a] + tw_ps)
            if c >= N:
                out[i] |= 2
                break
    return out


def pair_seeds(h: np.ndarray, seg_offsets, ppt: int, adj: np.ndarray, w_sc: int, w_fc: int, w_afc: int) -> np.ndarray:
    """PAPER.md:61-63 SC / FC / AFC straight from the sentences: all ordered pairs of a segment, no use of the time
    order, one rule at a time."""
    n = len(h)
    sg = seg_id(n, seg_offsets)
    t = [int(x) for x in h["t_ps"]]
    pmt = [int(x) for x in h["pmt_id"]]
    fl = [int(x) for x in h["floor"]]
    out = np.zeros(n, dtype=np.uint8)
    for i in range(n):
        for j in range(n):
            if i == j or sg[i] != sg[j] or pmt[i] == pmt[j]:
                continue
            dt = abs(t[i] - t[j])
            tower_i, tower_j = pmt[i] // ppt, pmt[j] // ppt
            # SC: "two hits occurred in two adjacent PMTs within 20 ns"
            if dt <= w_sc and tower_i == tower_j and adj[pmt[i] % ppt][pmt[j] % ppt]:
                out[i] |= 1
            # FC: "two PMTs in the same floor within 100 ns"
            if dt <= w_fc and fl[i] == fl[j]:
                out[i] |= 2
            # AFC: "two PMTs located at two consecutive floors within 250 ns"
            if dt <= w_afc and tower_i == tower_j and abs(fl[i] - fl[j]) == 1:
                out[i] |= 4
    return out


def l0_combine(l0: np.ndarray, pair_bits: np.ndarray, N: int) -> np.ndarray:
    """PAPER.md:65 'applying N7TW1000, and if it is satisfied, we apply [SC and AFC] or [FC and AFC]'."""
    out = np.zeros(len(l0), dtype=np.uint8)
    for k in range(len(l0)):
        if l0[k] & 1:
            window = [int(b) for b in pair_bits[k:k + N]]
            has = lambda bit: any(b & bit for b in window)
            if has(1) and has(4):
                out[k] |= 8
            if has(2) and has(4):
                out[k] |= 16
    return out


def l0_dntw(h: np.ndarray, seg_offsets, N: int, tw_ps: int) -> np.ndarray:
    """PAPER.md:60 'N hits from different PMTs within TW'.  Set formulation: start k fires <=> the set of pmt_id over
    the hits of its segment with index >= k and t < t_k + TW has at least N elements; its members run from k to the
    smallest index e for which the set over [k, e] already has N elements."""
    n = len(h)
    sg = seg_id(n, seg_offsets)
    t = [int(x) for x in h["t_ps"]]
    pmt = [int(x) for x in h["pmt_id"]]
    out = np.zeros(n, dtype=np.uint8)
    for k in range(n):
        inside = [j for j in range(k, n) if sg[j] == sg[k] and t[j] < t[k] + tw_ps]
        if tw_ps <= 0 or len({pmt[j] for j in inside}) < N:
            continue
        e = next(j for j in inside if len({pmt[m] for m in inside if m <= j}) >= N)
        out[k] |= 1
        for m in range(k, e + 1):
            out[m] |= 2
    return out
