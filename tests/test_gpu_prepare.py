"""GPU parity of tt_prepare_slice (NEXT-3; R24) against oracle.prepare: every record byte,
every run offset, the status word; then prepare -> sort + trigger equals the chain on the generator's own records."""
import numpy as np
import pytest
import torch

import oracle
from paper_1411_3968_b200 import workload as W
from util import oracle_chain

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1411_3968_b200 import binding

    binding.load()
    return binding


@pytest.mark.parametrize("cfg,ts,ss", [(0, 0.25, 1), (1, 0.1, 1), (2, 0.004, 1), (3, 0.02, 8 / 64), (4, 0.002, 1), (1, 1.0, 1)])
def test_prepare_configs(cfg, ts, ss, B, oracle_lib):
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    raw, samples, slice_off = W.make_raw(w)
    o_out, o_runs, o_st = oracle.prepare(raw, samples, slice_off, w.geometry.n_pmt)
    out, runs, st = B.prepare_slice(raw, samples, slice_off, w.geometry.n_pmt)
    assert st == o_st == 0
    assert out.tobytes() == o_out.tobytes()
    assert (runs == o_runs).all()
    assert out.tobytes() == np.ascontiguousarray(w.hits).tobytes()  # and both equal the generator's records


def test_prepare_edge_cases(B, oracle_lib):
    rng = np.random.default_rng(8)
    # the hand case of the oracle's pins: saturation, empty waveform, truncated section, bad PMT, empty slice
    raw = np.zeros(6, dtype=W.RAW_DTYPE)
    raw[0] = (500, 2, 0, 3, 10); raw[1] = (100, 0, 0, 0, 11); raw[2] = (700, 9, 1, 1, 12); raw[3] = (600, 2, 0, 2, 13)
    raw[4] = (-5, 1, 0, 2, 14); raw[5] = (7, 1, 0, 4, 15)
    samples = np.array([1, 2, 3, 50, 7, 8, 40000, 40000, 5, 6], dtype=np.uint16)
    so = np.array([0, 4, 4, 6], dtype=np.uint32)
    o = oracle.prepare(raw, samples, so, 3)
    g = B.prepare_slice(raw, samples, so, 3)
    assert g[2] == o[2] == (B.TT_S_BAD_PMT | B.TT_S_RAW_TRUNCATED)
    assert g[0].tobytes() == o[0].tobytes() and (g[1] == o[1]).all()
    # n = 0
    g = B.prepare_slice(raw[:0], samples[:0], np.array([0, 0], dtype=np.uint32), 5)
    assert len(g[0]) == 0 and (g[1] == 0).all() and g[2] == 0
    # random: many slices, many PMTs (three key digits), ragged sizes, extreme times, long waveforms
    for n, P, S in ((1, 1, 1), (2049, 7, 3), (100_000, 300, 70), (250_000, 3000, 40)):
        raw = np.zeros(n, dtype=W.RAW_DTYPE)
        raw["t_ps"] = rng.integers(-2**62, 2**62, size=n)
        raw["pmt_id"] = rng.integers(0, P, size=n)
        raw["floor"] = rng.integers(0, 65536, size=n)
        raw["n_samples"] = rng.integers(0, 40, size=n)
        raw["pad"] = np.arange(n) & 0xFFFF
        samples = rng.integers(0, 5000, size=int(raw["n_samples"].sum())).astype(np.uint16)
        cuts = np.sort(rng.integers(0, n + 1, size=S - 1)) if S > 1 else np.zeros(0, dtype=np.int64)
        so = np.concatenate([[0], cuts, [n]]).astype(np.uint32)
        o = oracle.prepare(raw, samples, so, P)
        g = B.prepare_slice(raw, samples, so, P)
        assert g[2] == o[2] == 0
        assert g[0].tobytes() == o[0].tobytes() and (g[1] == o[1]).all()


def test_prepare_then_sort_trigger(B, oracle_lib):
    """Raw stream -> tt_prepare_slice -> tt_sort_trigger_slice -> tt_extract_events = the oracle chain on the records."""
    w = W.make_config(2, time_scale=0.004)
    raw, samples, slice_off = W.make_raw(w)
    out, runs, st = B.prepare_slice(raw, samples, slice_off, w.geometry.n_pmt)
    assert st == 0
    g, p = w.geometry, w.params
    geo = B.Geometry(g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks)
    prm = B.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps)
    r = B.process_slice(out, w.seg_offsets, runs, geo, prm, fused=True)
    o = oracle_chain(w.hits, w.seg_offsets, g, p)
    assert r.sorted.tobytes() == o["sorted"].tobytes() and (r.flags == o["flags"]).all()
    assert (r.seeds == o["seeds"]).all() and r.events.tobytes() == o["events"].tobytes() and r.status == 0
