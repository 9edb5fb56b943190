"""GPU parity of tt_l0_ntw (level-0 N-in-TW trigger) against oracle.l0_ntw, byte for byte.
The oracle's input is always the oracle's own sort of the seeded input, never the CUDA output."""
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
    ref, ref_ns = oracle.l0_ntw(srt, seg, multiplicity=N, window_ps=tw)
    got, ns = B.l0_ntw(srt, seg, N, tw)
    assert got.shape == ref.shape
    bad = np.nonzero(got != ref)[0]
    assert len(bad) == 0, f"N={N} TW={tw}: {len(bad)} bytes differ, first at {bad[:5]}: gpu {got[bad[:5]]} oracle {ref[bad[:5]]}"
    assert ns == ref_ns
    return ref, ref_ns


def test_directed_boundaries(B, oracle_lib):
    """The hand-written cases of P15 (strict '<', segments, ties, N = 1, N > n, empty, extreme timestamps)."""
    one = lambda n: np.array([0, n], dtype=np.uint32)
    h3a = mk_hits([(0, 0, 0, 0), (40, 1, 0, 0), (99, 2, 0, 0)])
    h3b = mk_hits([(0, 0, 0, 0), (40, 1, 0, 0), (100, 2, 0, 0)])
    assert _check(B, h3a, one(3), 3, 100)[0].tolist() == [3, 2, 2]
    assert _check(B, h3b, one(3), 3, 100)[0].tolist() == [0, 0, 0]
    h5 = mk_hits([(0, 0, 0, 0), (10, 0, 0, 0), (20, 0, 0, 0), (105, 0, 0, 0), (300, 0, 0, 0)])
    assert _check(B, h5, one(5), 3, 100)[0].tolist() == [3, 3, 2, 2, 0]
    assert _check(B, h5, np.array([0, 2, 5], dtype=np.uint32), 3, 100)[0].tolist() == [0] * 5
    h4 = mk_hits([(7, 0, 0, 0)] * 4)
    assert _check(B, h4, one(4), 4, 1)[0].tolist() == [3, 2, 2, 2]
    assert _check(B, h4, one(4), 5, 10)[1] == 0
    assert _check(B, h4, one(4), 1, 1)[0].tolist() == [3] * 4
    assert _check(B, h4, one(4), 2, 0)[1] == 0 and _check(B, h4, one(4), 2, -5)[1] == 0
    assert _check(B, h4[:0], one(0), 3, 10)[1] == 0
    big = mk_hits([(-2**63, 0, 0, 0), (2**63 - 1, 0, 0, 0)])
    assert _check(B, big, one(2), 2, 2**63 - 1)[1] == 0
    near = mk_hits([(2**63 - 10, 0, 0, 0), (2**63 - 1, 0, 0, 0)])
    assert _check(B, near, one(2), 2, 10)[0].tolist() == [3, 2]


@pytest.mark.parametrize("cfg,ts,ss,N,tw", [
    (0, 0.25, 1, 7, 1_000_000),        # NEMO tower, N7TW1000: 88 k hits, 22 tiles, ragged tail
    (1, 0.1, 1, 7, 500_000),           # KM3NeT-It tower, N7TW500
    (2, 0.004, 1, 7, 200_000),         # burst
    (3, 0.02, 8 / 64, 7, 500_000),     # 8 segments: windows never cross a segment
    (4, 0.002, 1, 7, 12_000),          # 100 towers superimposed: 0.46 hits/ns
    (1, 0.1, 1, 2, 30_000), (1, 0.1, 1, 1, 1),
    # long windows (halo up to 255 hits): TW near (N - 1) / 4.62 hits per us so that both outcomes occur
    (1, 0.1, 1, 33, 6_500_000), (1, 0.1, 1, 64, 13_500_000), (1, 0.1, 1, 256, 55_000_000),
])
def test_configs_scaled(cfg, ts, ss, N, tw, B, oracle_lib):
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ref, ns = _check(B, srt, w.seg_offsets, N, tw)
    if N > 1:
        assert 0 < int((ref & 2).astype(bool).sum()) < w.n  # both outcomes occur
    assert (ref[(ref & 1) != 0] & 2).all()  # a firing start is a member of its own window


def test_many_small_segments_and_ties(B, oracle_lib):
    """Segments shorter than N, segments ending inside a tile and its halo, a dozen distinct timestamps."""
    rng = np.random.default_rng(5)
    n = 3 * 4096 + 777
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["t_ps"] = rng.integers(0, 12, size=n) * 1000 - 4000
    cuts = np.unique(np.concatenate([[0, n], rng.integers(0, n, size=400), [4096, 4097, 4100, 8191, 8192]]))
    seg = cuts.astype(np.uint32)
    seg = np.insert(seg, 5, seg[5])  # an empty segment
    srt, _ = oracle.sort(h, seg)
    for N, tw in [(7, 3001), (3, 1), (2, 1001), (40, 12_000)]:
        _check(B, srt, seg, N, tw)


def test_unaligned_output_and_count_optional(B, oracle_lib):
    w = W.make_config(1, time_scale=0.02)
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ref, _ = oracle.l0_ntw(srt, w.seg_offsets, multiplicity=7, window_ps=500_000)
    d = B.hits_to_device(srt)
    seg = B.Offsets(w.seg_offsets)
    buf = torch.full((w.n + 64,), 0xEE, dtype=torch.uint8, device="cuda")
    B.tt_l0_ntw(d, seg, 7, 500_000, buf[3:3 + w.n], None)  # byte-store path, no count
    torch.cuda.synchronize()
    out = buf.cpu().numpy()
    assert (out[3:3 + w.n] == ref).all()
    assert (out[:3] == 0xEE).all() and (out[3 + w.n:] == 0xEE).all()  # nothing written outside [0, n)


def test_argument_errors(B):
    d = torch.zeros((8, 2), dtype=torch.int64, device="cuda")
    l0 = torch.zeros(8, dtype=torch.uint8, device="cuda")
    seg = B.Offsets(np.array([0, 8], dtype=np.uint32))
    for N in (0, 257):
        with pytest.raises(B.TTError):
            B.tt_l0_ntw(d, seg, N, 1000, l0)


@pytest.mark.parametrize("cfg,N,tw", [(1, 7, 500_000), (4, 7, 12_000)])
def test_full_size(cfg, N, tw, B, oracle_lib):
    """BASELINE.json's full sizes, every byte compared (the oracle is O(n N))."""
    w = W.make_config(cfg)
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ref, ns = _check(B, srt, w.seg_offsets, N, tw)
    assert ns > 0
