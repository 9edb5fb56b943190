"""Pins P1 / P2 for oracle_sort: invariants and library stable sorts."""
import numpy as np
import pytest
import torch

import oracle
from paper_1411_3968_b200 import workload as W


def _check_invariants(h, seg, out, perm):
    n = len(h)
    assert sorted(perm.tolist()) == list(range(n))  # a permutation
    assert (out == h[perm]).all()  # pure permutation of whole 16-byte records
    assert out.tobytes() == h[perm].tobytes()
    for s in range(len(seg) - 1):
        a, b = int(seg[s]), int(seg[s + 1])
        t = out["t_ps"][a:b]
        assert (np.diff(t) >= 0).all()
        assert ((perm[a:b] >= a) & (perm[a:b] < b)).all()
        eq = np.diff(t) == 0
        assert (np.diff(perm[a:b].astype(np.int64))[eq] > 0).all()  # stability: ties keep input order
    out2, perm2 = oracle.sort(out, seg)
    assert (perm2 == np.arange(n)).all()  # sorting the output is the identity


@pytest.mark.parametrize("cfg,ts,ss", [(0, 0.1, 1), (1, 0.05, 1), (3, 0.01, 4 / 64), (4, 0.001, 1)])
def test_sort_invariants_and_library(cfg, ts, ss, oracle_lib):
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    for hits in (w.hits, W.shuffled(w)[0]):
        out, perm = oracle.sort(hits, w.seg_offsets)
        _check_invariants(hits, w.seg_offsets, out, perm)
        for s in range(len(w.seg_offsets) - 1):
            a, b = int(w.seg_offsets[s]), int(w.seg_offsets[s + 1])
            ref = np.argsort(hits["t_ps"][a:b], kind="stable") + a
            assert (perm[a:b] == ref).all()
            tref = torch.sort(torch.from_numpy(hits["t_ps"][a:b].copy()), stable=True).indices.numpy() + a
            assert (perm[a:b] == tref).all()
    # each run's internal order is preserved: within a run, output positions ascend
    out, perm = oracle.sort(w.hits, w.seg_offsets)
    inv = np.empty(w.n, dtype=np.int64)
    inv[perm] = np.arange(w.n)
    ro = w.run_offsets.astype(np.int64)
    brk = np.zeros(w.n - 1, dtype=bool)
    brk[ro[1:-1][(ro[1:-1] > 0) & (ro[1:-1] < w.n)] - 1] = True
    assert (np.diff(inv)[~brk] > 0).all()


def test_sort_ties_and_extremes(oracle_lib):
    rng = np.random.default_rng(3)
    n = 5000
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["t_ps"] = rng.integers(0, 40, size=n)  # heavy ties
    h["pmt_id"] = rng.integers(0, 84, size=n)
    h["pad"] = np.arange(n) & 0xFFFF
    seg = np.array([0, 1234, 1234, n], dtype=np.uint32)  # includes an empty segment
    out, perm = oracle.sort(h, seg)
    _check_invariants(h, seg, out, perm)
    h["t_ps"] = rng.integers(-2**62, 2**62, size=n)  # negative and > 2^40 timestamps (R1)
    h["t_ps"][:4] = [-2**63, 2**63 - 1, 0, -1]
    out, perm = oracle.sort(h, seg)
    _check_invariants(h, seg, out, perm)
    for m in (0, 1):
        out, perm = oracle.sort(h[:m], np.array([0, m], dtype=np.uint32))
        assert len(out) == m and (perm == np.arange(m)).all()
