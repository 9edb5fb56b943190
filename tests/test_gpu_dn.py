"""GPU parity of tt_l0_dntw (distinct-PMT level-0 trigger) against oracle.l0_dntw, byte for byte."""
import numpy as np
import pytest
import torch

import oracle
from paper_1411_3968_b200 import workload as W
from util import mk_hits

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1411_3968_b200 import binding

    binding.load()
    return binding


def _check(B, srt, seg, N, tw):
    ref, ref_ns = oracle.l0_dntw(srt, seg, multiplicity=N, window_ps=tw)
    got, ns = B.l0_dntw(srt, seg, N, tw)
    bad = np.nonzero(got != ref)[0]
    assert len(bad) == 0, f"N={N} TW={tw}: {len(bad)} bytes differ, first at {bad[:5]}: gpu {got[bad[:5]]} oracle {ref[bad[:5]]}"
    assert ns == ref_ns
    return ref, ref_ns


def test_directed_cases(B, oracle_lib):
    one = lambda n: np.array([0, n], dtype=np.uint32)
    h = mk_hits([(0, 0, 0, 0), (10, 0, 0, 0), (20, 1, 0, 0)])
    assert _check(B, h, one(3), 2, 100)[0].tolist() == [3, 3, 2]
    h = mk_hits([(0, 0, 0, 0), (100, 1, 0, 0)])
    assert _check(B, h, one(2), 2, 100)[1] == 0
    assert _check(B, h, one(2), 2, 101)[0].tolist() == [3, 2]
    h7 = mk_hits([(i, 3, 0, 0) for i in range(7)])
    assert _check(B, h7, one(7), 2, 10**9)[1] == 0
    h = mk_hits([(0, 0, 0, 0), (10, 1, 0, 0)])
    assert _check(B, h, np.array([0, 1, 2], dtype=np.uint32), 2, 100)[1] == 0
    assert _check(B, h, one(2), 1, 1)[0].tolist() == [3, 3]
    assert _check(B, h, one(2), 2, 0)[1] == 0 and _check(B, h, one(2), 2, -7)[1] == 0
    assert _check(B, h[:0], one(0), 2, 10)[1] == 0
    big = mk_hits([(-2**63, 0, 0, 0), (2**63 - 1, 1, 0, 0)])
    assert _check(B, big, one(2), 2, 2**63 - 1)[1] == 0


@pytest.mark.parametrize("cfg,ts,ss,N,tw", [
    (0, 0.25, 1, 7, 1_000_000),      # DN7TW1000 on the NEMO tower
    (1, 0.1, 1, 7, 500_000),
    (2, 0.004, 1, 7, 200_000),       # burst: the 1 MHz PMTs repeat inside a window (the case DN is for)
    (3, 0.02, 8 / 64, 7, 500_000),   # 8 segments
    (4, 0.002, 1, 7, 12_000),        # 100 towers
    (2, 0.004, 1, 16, 600_000), (1, 0.1, 1, 2, 30_000), (1, 0.1, 1, 1, 1),
])
def test_configs_scaled(cfg, ts, ss, N, tw, B, oracle_lib):
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ref, ns = _check(B, srt, w.seg_offsets, N, tw)
    if N > 1:
        assert 0 < int((ref & 2).astype(bool).sum()) < w.n


def test_windows_longer_than_the_stage(B, oracle_lib):
    """Few PMTs and long windows: a window holds thousands of hits before the N-th different PMT shows up (or never
    does), far past the 256-hit halo and across many tiles -- the global-memory continuation and the cross-tile member
    marks decide."""
    rng = np.random.default_rng(8)
    n = 6 * 1024 + 100
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    # long stretches of one PMT, a different one every ~700 hits
    h["pmt_id"] = (np.arange(n) // 700) % 5
    h["pmt_id"][rng.integers(0, n, size=12)] = 9
    h["t_ps"] = np.sort(rng.integers(0, 50_000_000, size=n))
    for seg in (np.array([0, n], dtype=np.uint32), np.array([0, 1500, 1500, 4000, n], dtype=np.uint32)):
        srt, _ = oracle.sort(h, seg)
        for N, tw in [(2, 4_000_000), (3, 12_000_000), (4, 60_000_000), (6, 10**12)]:
            _check(B, srt, seg, N, tw)


def test_unaligned_output_and_argument_errors(B, oracle_lib):
    w = W.make_config(2, time_scale=0.002)
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ref, _ = oracle.l0_dntw(srt, w.seg_offsets, multiplicity=7, window_ps=200_000)
    d = B.hits_to_device(srt)
    seg = B.Offsets(w.seg_offsets)
    buf = torch.full((w.n + 64,), 0xEE, dtype=torch.uint8, device="cuda")
    B.tt_l0_dntw(d, seg, 7, 200_000, buf[3:3 + w.n], None)
    torch.cuda.synchronize()
    out = buf.cpu().numpy()
    assert (out[3:3 + w.n] == ref).all() and (out[:3] == 0xEE).all() and (out[3 + w.n:] == 0xEE).all()
    for N in (0, 17):
        with pytest.raises(B.TTError):
            B.tt_l0_dntw(d, seg, N, 1000, buf)


@pytest.mark.parametrize("cfg,N,tw", [(1, 7, 500_000), (2, 7, 200_000)])
def test_full_size(cfg, N, tw, B, oracle_lib):
    w = W.make_config(cfg)
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ref, ns = _check(B, srt, w.seg_offsets, N, tw)
    assert ns > 0
