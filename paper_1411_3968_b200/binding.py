"""Thin ctypes binding of libtt.so (include/tt.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.

There is no CPU fallback: importing works without a GPU (so the ABI can be inspected), but every
compute call needs the library and a CUDA device and raises otherwise.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np
import torch

from . import _build

c_u32, c_i32, c_vp, c_sz = ctypes.c_uint32, ctypes.c_int32, ctypes.c_void_p, ctypes.c_size_t

TT_Q, TT_LC, TT_L1, TT_L2STAR, TT_L2, TT_INEVT = 1, 2, 4, 8, 16, 32
TT_OK, TT_E_INVAL, TT_E_CUDA, TT_E_WORKSPACE = 0, -1, -2, -3
TT_E_LIMIT = -4
TT_NOALLOC_WS_BYTES = 4 << 20
TT_S_SEED_OVERFLOW, TT_S_EVENT_OVERFLOW, TT_S_RUN_UNSORTED, TT_S_BAD_PMT, TT_S_DENSITY = 1, 2, 4, 8, 16
TT_S_RAW_TRUNCATED = 32
TT_S_L1_OVERFLOW = 64

EXPORTS = ["tt_version", "tt_geometry_create", "tt_geometry_destroy", "tt_sort_slice", "tt_trigger_slice",
           "tt_extract_events", "tt_host_ctx_create", "tt_host_ctx_destroy", "tt_process_host", "tt_launch_count",
           "tt_prof_enable", "tt_prof_read", "tt_l0_ntw", "tt_pair_seeds", "tt_l0_combine",
           "tt_l0_dntw", "tt_sort_trigger_slice", "tt_prepare_slice", "tt_host_submit",
           "tt_host_wait", "tt_sort_l1_slice", "tt_l1_export", "tt_l2_merged", "tt_l2_apply", "tt_tag_windows",
           "tt_extract_events_noalloc"]

HIT_DTYPE = np.dtype([("t_ps", "<i8"), ("pmt_id", "<u2"), ("floor", "<u2"), ("charge", "<u2"), ("pad", "<u2")])
EVENT_DTYPE = np.dtype([("t_start", "<i8"), ("t_end", "<i8"), ("hit_begin", "<u4"), ("hit_end", "<u4"),
                        ("seed_begin", "<u4"), ("n_seeds", "<u4")])


class TTParams(ctypes.Structure):
    """Mirror of tt_params (40 bytes)."""
    _fields_ = [("lc_window_ps", ctypes.c_int64), ("l2_window_ps", ctypes.c_int64),
                ("event_half_ps", ctypes.c_int64), ("l2_multiplicity", c_u32), ("l2_mode", c_u32),
                ("q_thresh", c_u32), ("l1_capacity", c_u32)]


assert ctypes.sizeof(TTParams) == 40


class TTError(RuntimeError):
    pass


_lib = None


def lib_path() -> str:
    return _build.LIB


def load(build: bool = True):
    """Load libtt.so (building it if stale).  Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build() if build else _build.LIB
        if not os.path.exists(path):
            raise TTError(f"{path} is missing: run __graft_entry__.build()")
        L = ctypes.CDLL(path)
        L.tt_version.restype = ctypes.c_char_p
        for name in EXPORTS[1:]:
            getattr(L, name).restype = ctypes.c_int
        L.tt_launch_count.restype = ctypes.c_uint64
        _lib = L
    return _lib


def launch_count() -> int:
    return int(load().tt_launch_count())


def prof_enable(on: bool):
    load().tt_prof_enable(c_i32(1 if on else 0))


def prof_read() -> dict[str, tuple[float, int]]:
    """{stage: (total ms, count)} since prof_enable(True); synchronise first."""
    buf = ctypes.create_string_buffer(1 << 16)
    nb = load().tt_prof_read(buf, c_sz(len(buf)))
    if nb < 0:
        raise TTError("tt_prof_read failed")
    out = {}
    for line in buf.raw[:nb].decode().splitlines():
        name, ms, cnt = line.split()
        out[name] = (float(ms), int(cnt))
    return out


def _check(rc: int, what: str):
    if rc != TT_OK:
        raise TTError(f"{what} failed: {({-1: 'TT_E_INVAL', -2: 'TT_E_CUDA', -3: 'TT_E_WORKSPACE'}).get(rc, rc)}")


def _need_cuda():
    if not torch.cuda.is_available():
        raise TTError("no CUDA device: the tower-trigger path has no CPU fallback")


def _dp(t: torch.Tensor | None):
    return c_vp(t.data_ptr()) if t is not None else c_vp(0)


def _hp(a: np.ndarray | None):
    return a.ctypes.data_as(c_vp) if a is not None else c_vp(0)


def _stream() -> c_vp:
    return c_vp(torch.cuda.current_stream().cuda_stream)


def make_params(q_thresh=300, lc_window_ps=20_000, l2_window_ps=3_000_000, l2_multiplicity=5, l2_mode=0,
                event_half_ps=3_000_000, l1_capacity=0) -> TTParams:
    return TTParams(int(lc_window_ps), int(l2_window_ps), int(event_half_ps), int(l2_multiplicity), int(l2_mode),
                    int(q_thresh), int(l1_capacity))


class Geometry:
    """Owns a tt_geometry handle (device copy of the block-sparse causality table)."""

    def __init__(self, n_pmt: int, n_tower: int, pmts_per_tower: int, pair_block: np.ndarray, blocks: np.ndarray):
        _need_cuda()
        L = load()
        pb = np.ascontiguousarray(pair_block, dtype=np.int32)
        bl = np.ascontiguousarray(blocks, dtype=np.int32)
        self.n_pmt, self.n_tower, self.ppt = int(n_pmt), int(n_tower), int(pmts_per_tower)
        self._h = c_vp(0)
        torch.cuda.init()
        torch.zeros(1, device="cuda")  # make sure the primary context exists
        rc = L.tt_geometry_create(ctypes.byref(self._h), c_u32(n_pmt), c_u32(n_tower), c_u32(pmts_per_tower), _hp(pb),
                                  _hp(bl), c_u32(bl.shape[0]))
        _check(rc, "tt_geometry_create")

    @property
    def handle(self):
        return self._h

    def close(self):
        if self._h:
            load().tt_geometry_destroy(self._h)
            self._h = c_vp(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def hits_to_device(hits: np.ndarray) -> torch.Tensor:
    """(n,) HIT_DTYPE numpy -> (n, 2) int64 CUDA tensor (16-byte records)."""
    _need_cuda()
    h = np.ascontiguousarray(hits, dtype=HIT_DTYPE)
    return torch.from_numpy(h.view(np.int64).reshape(-1, 2).copy()).cuda()


def hits_to_host(t: torch.Tensor) -> np.ndarray:
    return t.cpu().numpy().reshape(-1).view(HIT_DTYPE).copy()


def _offsets(o) -> tuple[np.ndarray, torch.Tensor]:
    h = np.ascontiguousarray(o, dtype=np.uint32)
    d = torch.from_numpy(h.view(np.int32).copy()).cuda()
    return h, d


class Offsets:
    """Host + device copies of an offsets array (uint32[k+1])."""

    def __init__(self, o):
        self.h, self.d = _offsets(o)
        self.count = len(self.h) - 1


def _ws(query, what) -> torch.Tensor:
    need = c_sz(0)
    _check(query(c_vp(0), ctypes.byref(need)), what + " (workspace query)")
    return torch.empty(max(int(need.value), 256), dtype=torch.uint8, device="cuda")


def tt_sort_slice(d_in: torch.Tensor, d_out: torch.Tensor, d_perm: torch.Tensor | None, seg: Offsets,
                  runs: Offsets | None, d_status: torch.Tensor, ws: torch.Tensor | None = None) -> torch.Tensor:
    """Enqueue tt_sort_slice on the current stream.  Returns the workspace tensor used (reusable)."""
    _need_cuda()
    L = load()
    n = d_in.shape[0]

    def call(wsp, nbytes):
        return L.tt_sort_slice(_dp(d_in), _dp(d_out), _dp(d_perm), c_u32(n), _dp(seg.d), _hp(seg.h), c_u32(seg.count),
                               _dp(runs.d) if runs else c_vp(0), _hp(runs.h) if runs else c_vp(0),
                               c_u32(runs.count if runs else 0), wsp, nbytes, _dp(d_status), _stream())

    if ws is None:
        ws = _ws(call, "tt_sort_slice")
    nb = c_sz(ws.numel())
    _check(call(_dp(ws), ctypes.byref(nb)), "tt_sort_slice")
    return ws


def tt_trigger_slice(d_sorted: torch.Tensor, seg: Offsets, geo: Geometry, params: TTParams, d_flags: torch.Tensor,
                     d_seeds: torch.Tensor, d_n_seeds: torch.Tensor, d_status: torch.Tensor,
                     ws: torch.Tensor | None = None) -> torch.Tensor:
    _need_cuda()
    L = load()
    n = d_sorted.shape[0]

    def call(wsp, nbytes):
        return L.tt_trigger_slice(_dp(d_sorted), c_u32(n), _dp(seg.d), _hp(seg.h), c_u32(seg.count), geo.handle,
                                  ctypes.byref(params), _dp(d_flags), _dp(d_seeds), c_u32(d_seeds.numel()),
                                  _dp(d_n_seeds), wsp, nbytes, _dp(d_status), _stream())

    if ws is None:
        ws = _ws(call, "tt_trigger_slice")
    nb = c_sz(ws.numel())
    _check(call(_dp(ws), ctypes.byref(nb)), "tt_trigger_slice")
    return ws


def tt_sort_trigger_slice(d_in: torch.Tensor, d_out: torch.Tensor, d_perm: torch.Tensor | None, seg: Offsets,
                          runs: Offsets | None, geo: Geometry, params: TTParams, d_flags: torch.Tensor,
                          d_seeds: torch.Tensor, d_n_seeds: torch.Tensor, d_status: torch.Tensor,
                          ws: torch.Tensor | None = None) -> torch.Tensor:
    """Enqueue tt_sort_trigger_slice (tt_sort_slice + tt_trigger_slice in one call, L1 fused into the last merge
    level) on the current stream.  Returns the workspace tensor used (reusable)."""
    _need_cuda()
    L = load()
    n = d_in.shape[0]

    def call(wsp, nbytes):
        return L.tt_sort_trigger_slice(_dp(d_in), _dp(d_out), _dp(d_perm), c_u32(n), _dp(seg.d), _hp(seg.h),
                                       c_u32(seg.count), _dp(runs.d) if runs else c_vp(0),
                                       _hp(runs.h) if runs else c_vp(0), c_u32(runs.count if runs else 0), geo.handle,
                                       ctypes.byref(params), _dp(d_flags), _dp(d_seeds), c_u32(d_seeds.numel()),
                                       _dp(d_n_seeds), wsp, nbytes, _dp(d_status), _stream())

    if ws is None:
        ws = _ws(call, "tt_sort_trigger_slice")
    nb = c_sz(ws.numel())
    _check(call(_dp(ws), ctypes.byref(nb)), "tt_sort_trigger_slice")
    return ws


def tt_extract_events(d_sorted: torch.Tensor, seg: Offsets, d_seeds: torch.Tensor, d_n_seeds: torch.Tensor,
                      params: TTParams, d_events: torch.Tensor, d_n_events: torch.Tensor,
                      d_flags: torch.Tensor | None, d_gather: torch.Tensor | None, d_n_gathered: torch.Tensor | None,
                      d_status: torch.Tensor, ws: torch.Tensor | None = None) -> torch.Tensor:
    _need_cuda()
    L = load()
    n = d_sorted.shape[0]

    def call(wsp, nbytes):
        return L.tt_extract_events(_dp(d_sorted), c_u32(n), _dp(seg.d), _hp(seg.h), c_u32(seg.count), _dp(d_seeds),
                                   _dp(d_n_seeds), c_u32(d_seeds.numel()), ctypes.byref(params), _dp(d_events),
                                   c_u32(d_events.shape[0]), _dp(d_n_events), _dp(d_flags), _dp(d_gather),
                                   _dp(d_n_gathered), wsp, nbytes, _dp(d_status), _stream())

    if ws is None:
        ws = _ws(call, "tt_extract_events")
    nb = c_sz(ws.numel())
    _check(call(_dp(ws), ctypes.byref(nb)), "tt_extract_events")
    return ws


def tt_extract_events_noalloc(d_sorted: torch.Tensor, seg: Offsets, d_seeds: torch.Tensor, d_n_seeds: torch.Tensor,
                              params: TTParams, d_events: torch.Tensor, d_n_events: torch.Tensor,
                              d_flags: torch.Tensor | None, d_gather: torch.Tensor | None,
                              d_n_gathered: torch.Tensor | None, d_status: torch.Tensor) -> int:
    """tt_extract_events with the scratch in the library's static device array: no workspace, nothing allocated.
    Returns the call's code (TT_OK or TT_E_LIMIT when seed_cap / event_cap need more than TT_NOALLOC_WS_BYTES);
    raises on any other error."""
    _need_cuda()
    L = load()
    rc = L.tt_extract_events_noalloc(_dp(d_sorted), c_u32(d_sorted.shape[0]), _dp(seg.d), _hp(seg.h), c_u32(seg.count),
                                     _dp(d_seeds), _dp(d_n_seeds), c_u32(d_seeds.numel()), ctypes.byref(params),
                                     _dp(d_events), c_u32(d_events.shape[0]), _dp(d_n_events), _dp(d_flags),
                                     _dp(d_gather), _dp(d_n_gathered), _dp(d_status), _stream())
    if rc != TT_E_LIMIT:
        _check(rc, "tt_extract_events_noalloc")
    return rc


RAW_DTYPE = np.dtype([("t_ps", "<i8"), ("pmt_id", "<u2"), ("floor", "<u2"), ("n_samples", "<u2"), ("pad", "<u2")])
L1HIT_DTYPE = np.dtype([("t_ps", "<i8"), ("idx", "<u4"), ("pmt_id", "<u2"), ("src", "<u2")])


# ---- the by-tower sharded trigger (include/tt.h: NEXT-4).  Records are (m, 2) int64 CUDA tensors (16 bytes each).
def _ws_call(call, what, ws):
    if ws is None:
        ws = _ws(call, what)
    nb = c_sz(ws.numel())
    _check(call(_dp(ws), ctypes.byref(nb)), what)
    return ws


def tt_sort_l1_slice(d_in, d_out, d_perm, seg: Offsets, runs: Offsets, params: TTParams, d_flags, d_status, ws=None):
    _need_cuda()
    L, n = load(), d_in.shape[0]
    return _ws_call(lambda w, nb: L.tt_sort_l1_slice(_dp(d_in), _dp(d_out), _dp(d_perm), c_u32(n), _dp(seg.d), _hp(seg.h),
                                                     c_u32(seg.count), _dp(runs.d), _hp(runs.h), c_u32(runs.count),
                                                     ctypes.byref(params), _dp(d_flags), w, nb, _dp(d_status), _stream()),
                    "tt_sort_l1_slice", ws)


def tt_l1_export(d_sorted, d_flags, src: int, d_l1, d_n_l1, d_status, ws=None):
    _need_cuda()
    L, n = load(), d_sorted.shape[0]
    return _ws_call(lambda w, nb: L.tt_l1_export(_dp(d_sorted), c_u32(n), _dp(d_flags), c_u32(int(src)), _dp(d_l1),
                                                 c_u32(d_l1.shape[0]), _dp(d_n_l1), w, nb, _dp(d_status), _stream()),
                    "tt_l1_export", ws)


def tt_l2_merged(d_l1, geo: Geometry, params: TTParams, d_bits, d_seeds, d_n_seeds, d_status, ws=None):
    _need_cuda()
    L, m = load(), d_l1.shape[0]
    return _ws_call(lambda w, nb: L.tt_l2_merged(_dp(d_l1), c_u32(m), geo.handle, ctypes.byref(params), _dp(d_bits),
                                                 _dp(d_seeds), c_u32(d_seeds.numel()), _dp(d_n_seeds), w, nb,
                                                 _dp(d_status), _stream()), "tt_l2_merged", ws)


def tt_l2_apply(d_l1, d_bits, src: int, d_flags, n: int, d_seeds, d_n_seeds, d_status, ws=None):
    _need_cuda()
    L, m = load(), d_l1.shape[0]
    return _ws_call(lambda w, nb: L.tt_l2_apply(_dp(d_l1), _dp(d_bits), c_u32(m), c_u32(int(src)), _dp(d_flags), c_u32(n),
                                                _dp(d_seeds), c_u32(d_seeds.numel()), _dp(d_n_seeds), w, nb, _dp(d_status),
                                                _stream()), "tt_l2_apply", ws)


def tt_tag_windows(d_sorted, d_events, d_n_events, params: TTParams, d_flags):
    _need_cuda()
    _check(load().tt_tag_windows(_dp(d_sorted), c_u32(d_sorted.shape[0]), _dp(d_events), _dp(d_n_events),
                                 c_u32(d_events.shape[0]), ctypes.byref(params), _dp(d_flags), _stream()), "tt_tag_windows")


def tt_prepare_slice(d_raw: torch.Tensor, d_samples: torch.Tensor, slices: Offsets, n_pmt: int, d_out: torch.Tensor,
                     d_run_offsets: torch.Tensor, d_status: torch.Tensor, ws: torch.Tensor | None = None) -> torch.Tensor:
    """Enqueue tt_prepare_slice: raw headers (n, 2) int64 + waveform samples (int16 storage of uint16)
    -> d_out (n, 2) int64 PMT-major records and d_run_offsets int32[n_slices * n_pmt + 1]."""
    _need_cuda()
    L = load()
    n = d_raw.shape[0]
    assert d_samples.dtype in (torch.int16, torch.uint16) and d_run_offsets.numel() >= slices.count * n_pmt + 1

    def call(wsp, nbytes):
        return L.tt_prepare_slice(_dp(d_raw), _dp(d_samples), c_u32(n), c_u32(d_samples.numel()), _dp(slices.d),
                                  _hp(slices.h), c_u32(slices.count), c_u32(int(n_pmt)), _dp(d_out), c_u32(d_out.shape[0]),
                                  _dp(d_run_offsets), wsp, nbytes, _dp(d_status), _stream())

    if ws is None:
        ws = _ws(call, "tt_prepare_slice")
    nb = c_sz(ws.numel())
    _check(call(_dp(ws), ctypes.byref(nb)), "tt_prepare_slice")
    return ws


def prepare_slice(raw: np.ndarray, samples: np.ndarray, slice_offsets, n_pmt: int):
    """Host-array convenience around tt_prepare_slice -> (records, run offsets, status)."""
    _need_cuda()
    r = np.ascontiguousarray(raw, dtype=RAW_DTYPE)
    n = len(r)
    d_raw = torch.from_numpy(r.view(np.int64).reshape(-1, 2).copy()).cuda()
    d_samples = torch.from_numpy(np.ascontiguousarray(samples, dtype=np.uint16).view(np.int16).copy()).cuda()
    sl = Offsets(slice_offsets)
    d_out = torch.full((max(n, 1), 2), -1, dtype=torch.int64, device="cuda")[:n]
    d_runs = torch.full((sl.count * n_pmt + 1,), -1, dtype=torch.int32, device="cuda")
    d_st = torch.zeros(1, dtype=torch.int32, device="cuda")
    tt_prepare_slice(d_raw, d_samples, sl, n_pmt, d_out, d_runs, d_st)
    torch.cuda.synchronize()
    return hits_to_host(d_out) if n else np.zeros(0, dtype=HIT_DTYPE), d_runs.cpu().numpy().view(np.uint32), int(d_st.item())


TT_L0_START, TT_L0_MEMBER = 1, 2


def tt_l0_ntw(d_sorted: torch.Tensor, seg: Offsets, multiplicity: int, window_ps: int, d_l0: torch.Tensor,
              d_n_start: torch.Tensor | None = None) -> None:
    """Enqueue tt_l0_ntw (level-0 N-in-TW trigger) on the current stream: d_l0[n] uint8 receives
    TT_L0_START | TT_L0_MEMBER, d_n_start (int32[1], optional) the number of firing window starts."""
    _need_cuda()
    L = load()
    n = d_sorted.shape[0]
    assert d_l0.dtype == torch.uint8 and d_l0.numel() >= n
    _check(L.tt_l0_ntw(_dp(d_sorted), c_u32(n), _dp(seg.d), c_u32(seg.count), c_u32(int(multiplicity)),
                       ctypes.c_int64(int(window_ps)), _dp(d_l0), _dp(d_n_start), _stream()), "tt_l0_ntw")


def l0_ntw(sorted_hits: np.ndarray, seg_offsets, multiplicity: int, window_ps: int):
    """Host-array convenience around tt_l0_ntw -> (l0 bytes [n], number of firing starts)."""
    _need_cuda()
    d_sorted = hits_to_device(sorted_hits)
    seg = Offsets(seg_offsets)
    n = d_sorted.shape[0]
    d_l0 = torch.zeros(max(n, 1), dtype=torch.uint8, device="cuda")
    d_ns = torch.zeros(1, dtype=torch.int32, device="cuda")
    tt_l0_ntw(d_sorted, seg, multiplicity, window_ps, d_l0, d_ns)
    torch.cuda.synchronize()
    return d_l0[:n].cpu().numpy(), int(d_ns.cpu().numpy().view(np.uint32)[0])


def tt_l0_dntw(d_sorted: torch.Tensor, seg: Offsets, multiplicity: int, window_ps: int, d_l0: torch.Tensor,
               d_n_start: torch.Tensor | None = None) -> None:
    """Enqueue tt_l0_dntw (distinct-PMT level-0 trigger) on the current stream."""
    _need_cuda()
    n = d_sorted.shape[0]
    assert d_l0.dtype == torch.uint8 and d_l0.numel() >= n
    _check(load().tt_l0_dntw(_dp(d_sorted), c_u32(n), _dp(seg.d), c_u32(seg.count), c_u32(int(multiplicity)),
                             ctypes.c_int64(int(window_ps)), _dp(d_l0), _dp(d_n_start), _stream()), "tt_l0_dntw")


def l0_dntw(sorted_hits: np.ndarray, seg_offsets, multiplicity: int, window_ps: int):
    """Host-array convenience around tt_l0_dntw -> (l0 bytes [n], number of firing starts)."""
    _need_cuda()
    d_sorted = hits_to_device(sorted_hits)
    seg = Offsets(seg_offsets)
    n = d_sorted.shape[0]
    d_l0 = torch.full((max(n, 1),), 0xEE, dtype=torch.uint8, device="cuda")  # the call zeroes it itself
    d_ns = torch.zeros(1, dtype=torch.int32, device="cuda")
    tt_l0_dntw(d_sorted, seg, multiplicity, window_ps, d_l0, d_ns)
    torch.cuda.synchronize()
    return d_l0[:n].cpu().numpy(), int(d_ns.cpu().numpy().view(np.uint32)[0])


TT_P_SC, TT_P_FC, TT_P_AFC, TT_P_CAND_A, TT_P_CAND_B = 1, 2, 4, 8, 16


def tt_pair_seeds(d_sorted: torch.Tensor, seg: Offsets, d_adj: torch.Tensor, ppt: int, d_bits: torch.Tensor,
                  sc_window_ps=20_000, fc_window_ps=100_000, afc_window_ps=250_000) -> None:
    """Enqueue tt_pair_seeds (SC / FC / AFC): d_bits[n] uint8 receives TT_P_SC | TT_P_FC | TT_P_AFC."""
    _need_cuda()
    n = d_sorted.shape[0]
    assert d_bits.dtype == torch.uint8 and d_bits.numel() >= n
    assert d_adj.dtype == torch.uint8 and d_adj.numel() == ppt * ppt and d_adj.is_contiguous()
    _check(load().tt_pair_seeds(_dp(d_sorted), c_u32(n), _dp(seg.d), c_u32(seg.count), _dp(d_adj), c_u32(int(ppt)),
                                ctypes.c_int64(int(sc_window_ps)), ctypes.c_int64(int(fc_window_ps)),
                                ctypes.c_int64(int(afc_window_ps)), _dp(d_bits), _stream()), "tt_pair_seeds")


def tt_l0_combine(d_l0: torch.Tensor, d_pair_bits: torch.Tensor, n: int, multiplicity: int, d_cand: torch.Tensor,
                  d_n_cand: torch.Tensor | None = None) -> None:
    """Enqueue tt_l0_combine: d_cand[n] uint8 receives TT_P_CAND_A | TT_P_CAND_B on firing starts."""
    _need_cuda()
    assert d_cand.dtype == torch.uint8 and d_cand.numel() >= n
    _check(load().tt_l0_combine(_dp(d_l0), _dp(d_pair_bits), c_u32(n), c_u32(int(multiplicity)), _dp(d_cand),
                                _dp(d_n_cand), _stream()), "tt_l0_combine")


def paper_trigger(sorted_hits: np.ndarray, seg_offsets, ppt: int, adj: np.ndarray, multiplicity: int, window_ps: int,
                  sc_window_ps=20_000, fc_window_ps=100_000, afc_window_ps=250_000):
    """Host-array convenience: tt_l0_ntw -> tt_pair_seeds -> tt_l0_combine.
    Returns (l0 bytes, pair bits, candidate bytes, (n_start, n_cand_a, n_cand_b))."""
    _need_cuda()
    d_sorted = hits_to_device(sorted_hits)
    seg = Offsets(seg_offsets)
    n = d_sorted.shape[0]
    d_adj = torch.from_numpy(np.ascontiguousarray(adj, dtype=np.uint8).reshape(-1).copy()).cuda()
    d_l0, d_pb, d_cd = (torch.zeros(max(n, 1), dtype=torch.uint8, device="cuda") for _ in range(3))
    d_cnt = torch.zeros(3, dtype=torch.int32, device="cuda")
    tt_l0_ntw(d_sorted, seg, multiplicity, window_ps, d_l0, d_cnt[0:1])
    tt_pair_seeds(d_sorted, seg, d_adj, ppt, d_pb, sc_window_ps, fc_window_ps, afc_window_ps)
    tt_l0_combine(d_l0, d_pb, n, multiplicity, d_cd, d_cnt[1:3])
    torch.cuda.synchronize()
    cnt = d_cnt.cpu().numpy().view(np.uint32)
    return d_l0[:n].cpu().numpy(), d_pb[:n].cpu().numpy(), d_cd[:n].cpu().numpy(), tuple(int(x) for x in cnt)


@dataclass
class SliceResult:
    sorted: np.ndarray
    perm: np.ndarray
    flags: np.ndarray
    seeds: np.ndarray
    n_seeds: int
    events: np.ndarray
    n_events: int
    status: int
    gathered: np.ndarray | None = None


def process_slice(hits: np.ndarray, seg_offsets, run_offsets, geo: Geometry, params: TTParams, seed_cap=None,
                  event_cap=None, gather=False, fused=False) -> SliceResult:
    """Convenience for tests: upload, run the three calls (fused: tt_sort_trigger_slice + tt_extract_events),
    download everything."""
    _need_cuda()
    n = len(hits)
    seg = Offsets(seg_offsets)
    runs = Offsets(run_offsets) if run_offsets is not None else None
    d_in = hits_to_device(hits)
    d_out = torch.empty_like(d_in)
    d_perm = torch.empty(max(n, 1), dtype=torch.int32, device="cuda")
    d_status = torch.zeros(1, dtype=torch.int32, device="cuda")
    seed_cap = n if seed_cap is None else seed_cap
    event_cap = n if event_cap is None else event_cap
    d_flags = torch.full((max(n, 1),), 0xEE if fused else 0, dtype=torch.uint8, device="cuda")  # every byte is written
    d_seeds = torch.zeros(max(seed_cap, 1), dtype=torch.int32, device="cuda")[:seed_cap]
    d_ns = torch.zeros(1, dtype=torch.int32, device="cuda")
    d_ev = torch.zeros((max(event_cap, 1), 4), dtype=torch.int64, device="cuda")[:event_cap]
    d_ne = torch.zeros(1, dtype=torch.int32, device="cuda")
    d_g = torch.zeros((max(n, 1), 2), dtype=torch.int64, device="cuda") if gather else None
    d_ng = torch.zeros(1, dtype=torch.int32, device="cuda") if gather else None
    if fused:
        tt_sort_trigger_slice(d_in, d_out, d_perm, seg, runs, geo, params, d_flags, d_seeds, d_ns, d_status)
    else:
        tt_sort_slice(d_in, d_out, d_perm, seg, runs, d_status)
        tt_trigger_slice(d_out, seg, geo, params, d_flags, d_seeds, d_ns, d_status)
    tt_extract_events(d_out, seg, d_seeds, d_ns, params, d_ev, d_ne, d_flags, d_g, d_ng, d_status)
    torch.cuda.synchronize()
    ns, ne = int(d_ns.item()) & 0xFFFFFFFF, int(d_ne.item()) & 0xFFFFFFFF
    res = SliceResult(
        sorted=hits_to_host(d_out), perm=d_perm.cpu().numpy().view(np.uint32)[:n].copy(),
        flags=d_flags.cpu().numpy()[:n].copy(), seeds=d_seeds.cpu().numpy().view(np.uint32)[: min(ns, seed_cap)].copy(),
        n_seeds=ns, events=d_ev.cpu().numpy().reshape(-1).view(EVENT_DTYPE)[: min(ne, event_cap)].copy(), n_events=ne,
        status=int(d_status.item()))
    if gather:
        ng = int(d_ng.item()) & 0xFFFFFFFF
        res.gathered = hits_to_host(d_g)[:ng]
    return res
