"""GPU parity of tt_pair_seeds (SC / FC / AFC) and tt_l0_combine against the
oracle, byte for byte.  The oracle's input is the oracle's own sort of the seeded input, never the CUDA output."""
import numpy as np
import pytest
import torch

import oracle
from paper_1411_3968_b200 import workload as W
from util import mk_hits

pytestmark = pytest.mark.gpu

SC, FC, AFC, CAND_A, CAND_B = 1, 2, 4, 8, 16


@pytest.fixture(scope="module")
def B():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1411_3968_b200 import binding

    binding.load()
    return binding


def _diff(name, got, ref):
    bad = np.nonzero(got != ref)[0]
    assert len(bad) == 0, f"{name}: {len(bad)} bytes differ, first at {bad[:5]}: gpu {got[bad[:5]]} oracle {ref[bad[:5]]}"


def _check(B, srt, seg, ppt, adj, N=7, tw=500_000, win=(20_000, 100_000, 250_000)):
    ref_l0, ref_ns = oracle.l0_ntw(srt, seg, multiplicity=N, window_ps=tw)
    ref_pb = oracle.pair_seeds(srt, seg, ppt, adj, sc_window_ps=win[0], fc_window_ps=win[1], afc_window_ps=win[2])
    ref_cd = oracle.l0_combine(ref_l0, ref_pb, N)
    l0, pb, cd, cnt = B.paper_trigger(srt, seg, ppt, adj, N, tw, *win)
    _diff("l0", l0, ref_l0)
    _diff("pair bits", pb, ref_pb)
    _diff("candidates", cd, ref_cd)
    assert cnt == (ref_ns, int(((ref_cd & CAND_A) != 0).sum()), int(((ref_cd & CAND_B) != 0).sum()))
    return ref_pb, ref_cd


def test_directed_cases(B, oracle_lib):
    """The hand-written cases of P19 (window edges, same PMT, tower boundaries, segments) through the CUDA path."""
    geo = W.make_geometry("km3", nx=2)
    adj, ppt = geo.adjacency(), geo.pmts_per_tower
    one = lambda n: np.array([0, n], dtype=np.uint32)
    cases = [
        ([(0, 0, 0, 0), (20_000, 1, 0, 0)], None, [SC | FC, SC | FC]),
        ([(0, 0, 0, 0), (20_001, 1, 0, 0)], None, [FC, FC]),
        ([(0, 0, 0, 0), (100_000, 1, 0, 0)], None, [FC, FC]),
        ([(0, 0, 0, 0), (100_001, 1, 0, 0)], None, [0, 0]),
        ([(0, 0, 0, 0), (5_000, 2, 0, 0)], None, [FC, FC]),
        ([(0, 0, 0, 0), (5_000, 0, 0, 0)], None, [0, 0]),
        ([(0, 0, 0, 0), (250_000, 6, 1, 0)], None, [AFC, AFC]),
        ([(0, 0, 0, 0), (250_001, 6, 1, 0)], None, [0, 0]),
        ([(0, 0, 0, 0), (1_000, 12, 2, 0)], None, [0, 0]),
        ([(0, 78, 13, 0), (1_000, 84, 14, 0)], None, [0, 0]),
        ([(0, 0, 0, 0), (1_000, 85, 14, 0)], None, [0, 0]),
        ([(0, 0, 0, 0), (1_000, 1, 0, 0)], np.array([0, 1, 2], dtype=np.uint32), [0, 0]),
        ([(0, 0, 0, 0), (10, 30, 5, 0), (250_000, 7, 1, 0)], None, [AFC, 0, AFC]),
        ([(-2**63, 0, 0, 0), (2**63 - 1, 1, 0, 0)], None, [0, 0]),
    ]
    for rows, seg, want in cases:
        h = mk_hits(rows)
        ref, _ = _check(B, h, seg if seg is not None else one(len(rows)), ppt, adj, N=2, tw=300_000)
        assert ref.tolist() == want
    _check(B, mk_hits([])[:0], one(0), ppt, adj)


@pytest.mark.parametrize("cfg,ts,ss,N,tw", [
    (0, 0.25, 1, 7, 1_000_000),      # NEMO tower, N7TW1000 + SC / FC / AFC: the paper's 32-PMT run
    (1, 0.1, 1, 7, 500_000),         # KM3NeT-It tower, N7TW500
    (2, 0.004, 1, 7, 200_000),       # burst: ~8 hits inside 250 ns
    (3, 0.02, 8 / 64, 7, 500_000),   # 8 segments
    (4, 0.0005, 1, 7, 12_000),       # 100 towers: ~116 hits inside 250 ns, same-tower tests matter
])
def test_configs_scaled(cfg, ts, ss, N, tw, B, oracle_lib):
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    g = w.geometry
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    pb, cd = _check(B, srt, w.seg_offsets, g.pmts_per_tower, g.adjacency(), N, tw)
    assert int(np.bitwise_or.reduce(pb)) == SC | FC | AFC   # every rule fires somewhere
    assert (cd != 0).any() and (cd == 0).any()


def test_windows_beyond_the_halo_and_zero_windows(B, oracle_lib):
    """Windows of 100-400 us at 4.6 hits/us reach 500-1800 hits, past the 256-hit halo: the exact global scans decide."""
    w = W.make_config(1, time_scale=0.03)
    g = w.geometry
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    for win in [(100_000_000, 20_000, 250_000), (20_000, 400_000_000, 250_000), (20_000, 100_000, 150_000_000),
                (0, 0, 0), (2**62, 0, 0)]:
        _check(B, srt, w.seg_offsets, g.pmts_per_tower, g.adjacency(), win=win)


def test_sparse_tiles_and_small_segments(B, oracle_lib):
    """>= 2^32 ps across a tile (the 32-bit staging cannot be used), many short segments, equal timestamps."""
    geo = W.make_geometry("km3")
    adj, ppt = geo.adjacency(), geo.pmts_per_tower
    rng = np.random.default_rng(11)
    n = 3 * 2048 + 333
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, 84, size=n)
    h["floor"] = geo.floor[h["pmt_id"]]
    # pairs 30 ns apart, the pairs 10 ms apart: 2048 hits span 10 s >> 2^32 ps
    h["t_ps"] = np.repeat(np.arange((n + 1) // 2, dtype=np.int64) * 10_000_000_000, 2)[:n] + rng.integers(0, 30_000, size=n)
    srt, _ = oracle.sort(h, np.array([0, n], dtype=np.uint32))
    pb, _ = _check(B, srt, np.array([0, n], dtype=np.uint32), ppt, adj, N=2, tw=40_000)
    assert pb.any()
    # dense, tied timestamps cut into ~300 segments (some empty, some ending inside the halo of a tile)
    h["t_ps"] = rng.integers(0, 40, size=n) * 5_000
    cuts = np.unique(np.concatenate([[0, n], rng.integers(0, n, size=300), [2048, 2049, 2303, 2304, 4095, 4096]]))
    seg = np.insert(cuts.astype(np.uint32), 7, cuts[7])
    srt, _ = oracle.sort(h, seg)
    _check(B, srt, seg, ppt, adj, N=3, tw=10_001)


def test_large_tower_table_in_global_memory(B, oracle_lib):
    """More than 128 PMTs per tower: the adjacency table is read from global memory."""
    ppt = 150
    rng = np.random.default_rng(2)
    adj = (rng.random((ppt, ppt)) < 0.2).astype(np.uint8)
    adj = adj | adj.T
    n = 5000
    h = np.zeros(n, dtype=W.HIT_DTYPE)
    h["pmt_id"] = rng.integers(0, 2 * ppt, size=n)
    h["floor"] = h["pmt_id"] // 10
    h["t_ps"] = rng.integers(0, 20_000_000, size=n)
    seg = np.array([0, n], dtype=np.uint32)
    srt, _ = oracle.sort(h, seg)
    pb, _ = _check(B, srt, seg, ppt, adj)
    assert int(np.bitwise_or.reduce(pb)) == SC | FC | AFC


def test_unaligned_output_and_argument_errors(B, oracle_lib):
    w = W.make_config(1, time_scale=0.02)
    g = w.geometry
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    ref = oracle.pair_seeds(srt, w.seg_offsets, g.pmts_per_tower, g.adjacency())
    d = B.hits_to_device(srt)
    seg = B.Offsets(w.seg_offsets)
    d_adj = torch.from_numpy(g.adjacency().reshape(-1).copy()).cuda()
    buf = torch.full((w.n + 64,), 0xEE, dtype=torch.uint8, device="cuda")
    B.tt_pair_seeds(d, seg, d_adj, g.pmts_per_tower, buf[5:5 + w.n])
    torch.cuda.synchronize()
    out = buf.cpu().numpy()
    assert (out[5:5 + w.n] == ref).all() and (out[:5] == 0xEE).all() and (out[5 + w.n:] == 0xEE).all()
    with pytest.raises(B.TTError):
        B.tt_pair_seeds(d, seg, d_adj, g.pmts_per_tower, buf[: w.n], sc_window_ps=-1)
    with pytest.raises(B.TTError):
        B.tt_l0_combine(buf, buf, w.n, 0, buf)


@pytest.mark.parametrize("cfg,N,tw", [(1, 7, 500_000), (2, 7, 200_000)])
def test_full_size(cfg, N, tw, B, oracle_lib):
    """BASELINE.json's full sizes (0.92 M and 30.8 M hits), every byte compared."""
    w = W.make_config(cfg)
    g = w.geometry
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    pb, cd = _check(B, srt, w.seg_offsets, g.pmts_per_tower, g.adjacency(), N, tw)
    assert (cd != 0).any()
