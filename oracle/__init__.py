"""CPU oracle of the sort + trigger path -- TEST INFRASTRUCTURE, not product code.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_1411_3968_b200's CUDA binding and shares no code
with it; the numpy record dtypes below are re-declared from the paper's description of the
fixed-size hit structure and BASELINE.json configs[0].

`build()` compiles oracle/tt_oracle.cpp with g++ into oracle/liboracle.so.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tt_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

HIT = np.dtype([("t_ps", "<i8"), ("pmt_id", "<u2"), ("floor", "<u2"), ("charge", "<u2"), ("pad", "<u2")])
EVENT = np.dtype([("t_start", "<i8"), ("t_end", "<i8"), ("hit_begin", "<u4"), ("hit_end", "<u4"),
                  ("seed_begin", "<u4"), ("n_seeds", "<u4")])
F_Q, F_LC, F_L1, F_L2STAR, F_L2, F_INEVT = 1, 2, 4, 8, 16, 32


class _Params(ctypes.Structure):
    _fields_ = [("lc_window_ps", ctypes.c_int64), ("l2_window_ps", ctypes.c_int64),
                ("event_half_ps", ctypes.c_int64), ("l2_multiplicity", ctypes.c_uint32),
                ("l2_mode", ctypes.c_uint32), ("q_thresh", ctypes.c_uint32), ("reserved", ctypes.c_uint32)]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p) if a is not None else None


def _mk_params(q_thresh, lc_window_ps, l2_window_ps, l2_multiplicity, l2_mode, event_half_ps):
    return _Params(int(lc_window_ps), int(l2_window_ps), int(event_half_ps), int(l2_multiplicity),
                   int(l2_mode), int(q_thresh), 0)


def sort(hits: np.ndarray, seg_offsets: np.ndarray):
    """-> (sorted hits, perm)"""
    hits = np.ascontiguousarray(hits, dtype=HIT)
    seg = np.ascontiguousarray(seg_offsets, dtype=np.uint32)
    n = hits.shape[0]
    out = np.empty_like(hits)
    perm = np.empty(n, dtype=np.uint32)
    rc = lib().oracle_sort(_p(hits), _p(out), _p(perm), ctypes.c_uint32(n), _p(seg), ctypes.c_uint32(len(seg) - 1))
    assert rc == 0
    return out, perm


@dataclass
class TriggerResult:
    flags: np.ndarray
    seeds: np.ndarray
    status: int


def trigger(sorted_hits: np.ndarray, seg_offsets: np.ndarray, n_pmt: int, n_tower: int, ppt: int,
            pair_block: np.ndarray, blocks: np.ndarray, *, q_thresh=300, lc_window_ps=20_000,
            l2_window_ps=3_000_000, l2_multiplicity=5, l2_mode=0, event_half_ps=3_000_000) -> TriggerResult:
    h = np.ascontiguousarray(sorted_hits, dtype=HIT)
    seg = np.ascontiguousarray(seg_offsets, dtype=np.uint32)
    pb = np.ascontiguousarray(pair_block, dtype=np.int32)
    bl = np.ascontiguousarray(blocks, dtype=np.int32)
    n = h.shape[0]
    flags = np.zeros(n, dtype=np.uint8)
    seeds = np.zeros(max(n, 1), dtype=np.uint32)
    ns = ctypes.c_uint32(0)
    st = ctypes.c_int32(0)
    prm = _mk_params(q_thresh, lc_window_ps, l2_window_ps, l2_multiplicity, l2_mode, event_half_ps)
    rc = lib().oracle_trigger(_p(h), ctypes.c_uint32(n), _p(seg), ctypes.c_uint32(len(seg) - 1),
                              ctypes.c_uint32(n_pmt), ctypes.c_uint32(n_tower), ctypes.c_uint32(ppt),
                              _p(pb), _p(bl), ctypes.byref(prm), _p(flags), _p(seeds), ctypes.byref(ns),
                              ctypes.byref(st))
    if rc != 0:
        raise ValueError("oracle_trigger: invalid parameters")
    return TriggerResult(flags, seeds[: ns.value].copy(), st.value)


def events(sorted_hits: np.ndarray, seg_offsets: np.ndarray, seeds: np.ndarray, *, event_half_ps=3_000_000,
           flags: np.ndarray | None = None):
    """-> events array (EVENT dtype); ORs F_INEVT into flags in place when given."""
    h = np.ascontiguousarray(sorted_hits, dtype=HIT)
    seg = np.ascontiguousarray(seg_offsets, dtype=np.uint32)
    sd = np.ascontiguousarray(seeds, dtype=np.uint32)
    ev = np.zeros(max(len(sd), 1), dtype=EVENT)
    ne = ctypes.c_uint32(0)
    prm = _mk_params(0, 0, 0, 1, 0, event_half_ps)
    if flags is not None:
        assert flags.dtype == np.uint8 and flags.flags.c_contiguous
    rc = lib().oracle_events(_p(h), ctypes.c_uint32(h.shape[0]), _p(seg), ctypes.c_uint32(len(seg) - 1), _p(sd),
                             ctypes.c_uint32(len(sd)), ctypes.byref(prm), _p(ev), ctypes.byref(ne), _p(flags))
    if rc != 0:
        raise ValueError("oracle_events: invalid parameters")
    return ev[: ne.value].copy()


L0_START, L0_MEMBER = 1, 2


def l0_ntw(sorted_hits: np.ndarray, seg_offsets: np.ndarray, *, multiplicity: int, window_ps: int):
    """Level-0 N-in-TW trigger -> (l0 bytes [n], number of firing window starts)."""
    h = np.ascontiguousarray(sorted_hits, dtype=HIT)
    seg = np.ascontiguousarray(seg_offsets, dtype=np.uint32)
    n = h.shape[0]
    l0 = np.zeros(n, dtype=np.uint8)
    ns = ctypes.c_uint32(0)
    rc = lib().oracle_l0_ntw(_p(h), ctypes.c_uint32(n), _p(seg), ctypes.c_uint32(len(seg) - 1),
                             ctypes.c_uint32(int(multiplicity)), ctypes.c_int64(int(window_ps)), _p(l0),
                             ctypes.byref(ns))
    if rc != 0:
        raise ValueError("oracle_l0_ntw: invalid parameters")
    return l0, ns.value


P_SC, P_FC, P_AFC, P_CAND_A, P_CAND_B = 1, 2, 4, 8, 16


def pair_seeds(sorted_hits: np.ndarray, seg_offsets: np.ndarray, ppt: int, adj: np.ndarray, *, sc_window_ps=20_000,
               fc_window_ps=100_000, afc_window_ps=250_000) -> np.ndarray:
    """SC / FC / AFC bits per hit.  adj: (ppt, ppt) uint8, nonzero = adjacent PMTs of one tower."""
    h = np.ascontiguousarray(sorted_hits, dtype=HIT)
    seg = np.ascontiguousarray(seg_offsets, dtype=np.uint32)
    a = np.ascontiguousarray(adj, dtype=np.uint8)
    assert a.shape == (ppt, ppt)
    bits = np.zeros(h.shape[0], dtype=np.uint8)
    rc = lib().oracle_pair_seeds(_p(h), ctypes.c_uint32(h.shape[0]), _p(seg), ctypes.c_uint32(len(seg) - 1),
                                 ctypes.c_uint32(int(ppt)), _p(a), ctypes.c_int64(int(sc_window_ps)),
                                 ctypes.c_int64(int(fc_window_ps)), ctypes.c_int64(int(afc_window_ps)), _p(bits))
    if rc != 0:
        raise ValueError("oracle_pair_seeds: invalid parameters")
    return bits


def l0_combine(l0: np.ndarray, pair_bits: np.ndarray, multiplicity: int) -> np.ndarray:
    """Candidate bits (8 = N-in-TW with [SC and AFC], 16 = with [FC and AFC]) on firing window starts."""
    a = np.ascontiguousarray(l0, dtype=np.uint8)
    b = np.ascontiguousarray(pair_bits, dtype=np.uint8)
    assert a.shape == b.shape
    out = np.zeros_like(a)
    rc = lib().oracle_l0_combine(_p(a), _p(b), ctypes.c_uint32(a.shape[0]), ctypes.c_uint32(int(multiplicity)), _p(out))
    if rc != 0:
        raise ValueError("oracle_l0_combine: invalid input")
    return out


def l0_dntw(sorted_hits: np.ndarray, seg_offsets: np.ndarray, *, multiplicity: int, window_ps: int):
    """Distinct-PMT level-0 trigger DNnTW -> (l0 bytes [n], number of firing window starts)."""
    h = np.ascontiguousarray(sorted_hits, dtype=HIT)
    seg = np.ascontiguousarray(seg_offsets, dtype=np.uint32)
    n = h.shape[0]
    l0 = np.zeros(n, dtype=np.uint8)
    ns = ctypes.c_uint32(0)
    rc = lib().oracle_l0_dntw(_p(h), ctypes.c_uint32(n), _p(seg), ctypes.c_uint32(len(seg) - 1),
                              ctypes.c_uint32(int(multiplicity)), ctypes.c_int64(int(window_ps)), _p(l0),
                              ctypes.byref(ns))
    if rc != 0:
        raise ValueError("oracle_l0_dntw: invalid parameters")
    return l0, ns.value


RAW = np.dtype([("t_ps", "<i8"), ("pmt_id", "<u2"), ("floor", "<u2"), ("n_samples", "<u2"), ("pad", "<u2")])


def prepare(raw: np.ndarray, samples: np.ndarray, slice_offsets: np.ndarray, n_pmt: int):
    """The paper's CPU preparation (R24): raw headers + concatenated waveforms ->
    (fixed-size hit records slice-major / PMT-major, run offsets [n_slices * n_pmt + 1], status)."""
    r = np.ascontiguousarray(raw, dtype=RAW)
    sm = np.ascontiguousarray(samples, dtype=np.uint16)
    so = np.ascontiguousarray(slice_offsets, dtype=np.uint32)
    n, ns = r.shape[0], len(so) - 1
    out = np.zeros(n, dtype=HIT)
    runs = np.zeros(ns * int(n_pmt) + 1, dtype=np.uint32)
    st = ctypes.c_int32(0)
    rc = lib().oracle_prepare(_p(r), _p(sm), ctypes.c_uint32(n), ctypes.c_uint32(len(sm)), _p(so), ctypes.c_uint32(ns),
                              ctypes.c_uint32(int(n_pmt)), _p(out), _p(runs), ctypes.byref(st))
    if rc != 0:
        raise ValueError("oracle_prepare: invalid parameters")
    return out, runs, st.value
