"""Pins of oracle.prepare (NEXT-3, the paper's CPU preparation; reading R24).

P26  round trip: the generator's PMT-major records came first; workload.make_raw turns them into an arrival-order raw
     stream with waveforms; prepare must give back the records and run offsets byte for byte.
P27  run offsets = per-(slice, PMT) counts (numpy bincount), records of a run in arrival order (numpy stable argsort).
P28  hand-written case: saturating charge, zero-length waveform, a waveform cut off by the end of the sample section,
     pmt_id out of range, an empty slice.
P29  the paper's sizes: 28 bytes per raw hit on average, 16-byte fixed records."""
import numpy as np

import oracle
from paper_1411_3968_b200 import workload as W


def test_round_trip_configs(oracle_lib):  # P26
    for cfg, ts, ss in ((0, 0.1, 1), (1, 0.05, 1), (2, 0.002, 1), (3, 0.01, 4 / 64), (4, 0.001, 1)):
        w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
        raw, samples, slice_off = W.make_raw(w)
        assert not np.array_equal(raw["pmt_id"], w.hits["pmt_id"]), "the raw stream must not be PMT-major already"
        out, runs, st = oracle.prepare(raw, samples, slice_off, w.geometry.n_pmt)
        assert st == 0
        assert out.tobytes() == np.ascontiguousarray(w.hits).tobytes()
        assert (runs == w.run_offsets).all()


def test_counts_and_stable_order(oracle_lib):  # P27
    rng = np.random.default_rng(5)
    n, P, S = 20_000, 37, 3
    raw = np.zeros(n, dtype=W.RAW_DTYPE)
    raw["t_ps"] = rng.integers(-10**12, 10**12, size=n)
    raw["pmt_id"] = rng.integers(0, P, size=n)
    raw["floor"] = raw["pmt_id"] // 4
    raw["n_samples"] = rng.integers(0, 9, size=n)
    raw["pad"] = np.arange(n) & 0xFFFF
    samples = rng.integers(0, 400, size=int(raw["n_samples"].sum())).astype(np.uint16)
    slice_off = np.array([0, 7000, 7000 + 4000, n], dtype=np.uint32)
    out, runs, st = oracle.prepare(raw, samples, slice_off, P)
    assert st == 0
    sl = np.searchsorted(slice_off, np.arange(n), side="right") - 1
    key = sl * P + raw["pmt_id"].astype(np.int64)
    assert (np.diff(runs.astype(np.int64)) == np.bincount(key, minlength=S * P)).all() and runs[0] == 0 and runs[-1] == n
    order = np.argsort(key, kind="stable")
    assert (out["pad"] == raw["pad"][order]).all() and (out["t_ps"] == raw["t_ps"][order]).all()
    woff = np.concatenate([[0], np.cumsum(raw["n_samples"].astype(np.int64))])
    charge = np.array([min(65535, int(samples[woff[k]:woff[k + 1]].sum())) for k in order])
    assert (out["charge"] == charge).all()


def test_hand_case(oracle_lib):  # P28
    raw = np.zeros(6, dtype=W.RAW_DTYPE)
    #            t     pmt floor n_samples pad
    raw[0] = (500, 2, 0, 3, 10)   # slice 0
    raw[1] = (100, 0, 0, 0, 11)   # no waveform: charge 0
    raw[2] = (700, 9, 1, 1, 12)   # pmt 9 >= n_pmt 3: filed under pmt 2, status 8
    raw[3] = (600, 2, 0, 2, 13)
    # slice 1 is empty; slice 2:
    raw[4] = (-5, 1, 0, 2, 14)    # saturates: 40000 + 40000
    raw[5] = (7, 1, 0, 4, 15)     # only 2 of its 4 samples exist: status 32
    samples = np.array([1, 2, 3, 50, 7, 8, 40000, 40000, 5, 6], dtype=np.uint16)
    out, runs, st = oracle.prepare(raw, samples, np.array([0, 4, 4, 6], dtype=np.uint32), 3)
    assert st == (8 | 32)
    assert runs.tolist() == [0, 1, 1, 4, 4, 4, 4, 4, 6, 6]
    assert [tuple(int(x) for x in r) for r in out] == [
        (100, 0, 0, 0, 11), (500, 2, 0, 6, 10), (700, 9, 1, 50, 12), (600, 2, 0, 15, 13),
        (-5, 1, 0, 65535, 14), (7, 1, 0, 11, 15)]


def test_paper_sizes(oracle_lib):  # P29
    w = W.make_config(1, time_scale=0.2)
    raw, samples, _ = W.make_raw(w)
    mean_bytes = (raw.nbytes + samples.nbytes) / len(raw)
    assert abs(mean_bytes - 28.0) < 0.2, mean_bytes  # PAPER.md:21 "The PMT hit size is 28 bytes in average"
    assert W.RAW_DTYPE.itemsize == 16 and W.HIT_DTYPE.itemsize == 16
