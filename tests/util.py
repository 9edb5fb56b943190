"""Shared test helpers: run the oracle chain on a workload / raw arrays."""
from __future__ import annotations

import numpy as np

import oracle
from paper_1411_3968_b200 import workload as W


def geo_args(geo: W.Geometry):
    return dict(n_pmt=geo.n_pmt, n_tower=geo.n_tower, ppt=geo.pmts_per_tower, pair_block=geo.pair_block,
                blocks=geo.blocks)


def params_kw(p: W.Params):
    return dict(q_thresh=p.q_thresh, lc_window_ps=p.lc_window_ps, l2_window_ps=p.l2_window_ps,
                l2_multiplicity=p.l2_multiplicity, l2_mode=p.l2_mode, event_half_ps=p.event_half_ps)


def oracle_chain(hits, seg_offsets, geo: W.Geometry, p: W.Params, tag=True):
    srt, perm = oracle.sort(hits, seg_offsets)
    tr = oracle.trigger(srt, seg_offsets, **geo_args(geo), **params_kw(p))
    flags = tr.flags.copy()
    ev = oracle.events(srt, seg_offsets, tr.seeds, event_half_ps=p.event_half_ps, flags=flags if tag else None)
    return dict(sorted=srt, perm=perm, flags=flags, seeds=tr.seeds, events=ev, status=tr.status)


def single_tower_geo(table: np.ndarray, name="custom") -> W.Geometry:
    """Geometry with one tower and the given dense (P,P) int32 table (positions unused)."""
    P = table.shape[0]
    return W.Geometry(name, np.zeros((P, 3)), np.zeros(P, dtype=np.int32), np.zeros(P, dtype=np.uint16), 1, P,
                      np.zeros(1, dtype=np.int32), np.ascontiguousarray(table, dtype=np.int32)[None])


def mk_hits(rows):
    """rows: iterable of (t_ps, pmt_id, floor, charge)"""
    h = np.zeros(len(rows), dtype=W.HIT_DTYPE)
    for k, r in enumerate(rows):
        h[k] = (r[0], r[1], r[2], r[3], k & 0xFFFF)
    return h
