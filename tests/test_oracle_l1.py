"""Pins P4 / P5 for the L1 part of oracle_trigger."""
import numpy as np

import oracle
from oracle import brute
from paper_1411_3968_b200 import workload as W
from util import geo_args


def _dense_small(seed, n, span_ps, P=12, ppf=4, n_seg=2):
    rng = np.random.default_rng(seed)
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, P, size=n)
    h["floor"] = h["pmt_id"] // ppf
    h["charge"] = rng.integers(250, 350, size=n)
    cut = n // 3
    seg = np.array([0, cut, n], dtype=np.uint32) if n_seg == 2 else np.array([0, n], dtype=np.uint32)
    h["t_ps"] = rng.integers(0, span_ps, size=n)
    srt, _ = oracle.sort(h, seg)
    return srt, seg


def test_l1_brute_force_p4(oracle_lib):
    geo = W.make_geometry("nemo")
    for seed, n, span in ((1, 700, 3_000_000), (2, 500, 1_000_000), (3, 300, 30_000_000)):
        srt, seg = _dense_small(seed, n, span)
        tr = oracle.trigger(srt, seg, **geo_args(geo), l2_multiplicity=4)
        ref = brute.l1_flags(srt, seg, 300, 20_000)
        assert ((tr.flags & 7) == ref).all()
        assert 0 < (ref & 2).astype(bool).mean() < 1  # the case exercises both outcomes


def test_l1_poisson_closed_form_p5(oracle_lib):
    """Two PMTs on one floor at R = 1 MHz for T = 1 s, LC = 20 ns: hits on PMT 0 with a partner on
    PMT 1 within +-LC number R*T*(1 - exp(-2*R*LC)) = 39 211 (the flagged-hit form of north_star's
    random-coincidence rate 2*R1*R2*dt = 40 000 /s)."""
    geo = W.make_geometry("nemo")
    R, T = 1e6, 1_000_000_000_000
    rates = np.zeros(32)
    rates[[0, 1]] = R
    h, _, _ = W.make_segment(geo, rates, 0, T, 1, 0, 99)
    h["charge"] = 100  # no Q bits
    seg = np.array([0, len(h)], dtype=np.uint32)
    srt, _ = oracle.sort(h, seg)
    tr = oracle.trigger(srt, seg, **geo_args(geo), l2_multiplicity=4)
    n0 = int(((tr.flags & 2) != 0)[srt["pmt_id"] == 0].sum())
    expect = R * 1.0 * (1 - np.exp(-2 * R * 20e-9))
    assert abs(expect - 39211) < 1
    assert abs(n0 - expect) < 5 * np.sqrt(expect)
    # pair-count form: sum over PMT-0 hits of partners within +-LC = 2*R1*R2*dt*T = 40 000
    t0 = srt["t_ps"][srt["pmt_id"] == 0]
    t1 = srt["t_ps"][srt["pmt_id"] == 1]
    pairs = int((np.searchsorted(t1, t0 + 20_000, "right") - np.searchsorted(t1, t0 - 20_000, "left")).sum())
    assert abs(pairs - 40000) < 5 * 200
    # a hit with no partner is not flagged, one with a partner is: exact agreement with the pair count
    has = (np.searchsorted(t1, t0 + 20_000, "right") - np.searchsorted(t1, t0 - 20_000, "left")) > 0
    assert n0 == int(has.sum())


def test_l1_same_pmt_and_other_floor_do_not_count(oracle_lib):
    geo = W.make_geometry("nemo")
    # only PMT 0 firing at 5 MHz: no LC possible (R5); PMT 0 + PMT 4 (other floor): none either (R6)
    for pm in ([0], [0, 4]):
        rates = np.zeros(32)
        rates[pm] = 5e6
        h, _, _ = W.make_segment(geo, rates, 0, 2_000_000_000, 1, 0, 5)
        h["charge"] = 100
        seg = np.array([0, len(h)], dtype=np.uint32)
        srt, _ = oracle.sort(h, seg)
        tr = oracle.trigger(srt, seg, **geo_args(geo), l2_multiplicity=4)
        assert len(h) > 5000 and not tr.flags.any()
