"""Seeded synthetic workloads shaped like the paper's tower data (input generator only).

This module serves both the oracle (``oracle/``) and the CUDA path; it holds none of the
method's arithmetic (no sorting of the mixed stream, no L1/L2/event logic).  It produces

* the PMT geometry of the two towers the paper simulates -- NEMO Phase II, 8 floors x 4 PMTs,
  40 m floor spacing, 6 m floor (sect. 2) and the KM3NeT-It tower, 14 floors x 6 PMTs,
  20 m spacing (sect. 5) -- and the 100-tower block of BASELINE.json configs[4];
* the integer causality table ``dtmax[i][j] = llround((d_ij * n / c + 20 ns) * 1e12)`` ps
  (BASELINE.json configs[0]), dense per tower-offset block;
* per-PMT time-ordered hit streams ("our data ... is time-ordered for single PMT",
  PAPER.md:53 sect. 4.2): Poisson background at 50-55 kHz per PMT plus injected
  straight muon tracks with Cherenkov-timed hits (sect. 3), concatenated PMT-major.

The paper's simulated NEMO data are not available; these inputs stand in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

HIT_DTYPE = np.dtype(
    [("t_ps", "<i8"), ("pmt_id", "<u2"), ("floor", "<u2"), ("charge", "<u2"), ("pad", "<u2")]
)
assert HIT_DTYPE.itemsize == 16

C_LIGHT = 299_792_458.0  # m/s
N_WATER = 1.35
LC_SLACK_S = 20e-9
TOWER_RANGE_M = 300.0
BASE_SEED = 14113968


@dataclass
class Geometry:
    name: str
    pos: np.ndarray  # (P,3) float64 metres
    tower: np.ndarray  # (P,) int32 tower index
    floor: np.ndarray  # (P,) uint16 global floor id = tower*floors + f
    n_tower: int
    pmts_per_tower: int
    pair_block: np.ndarray  # (n_tower*n_tower,) int32 block id or -1
    blocks: np.ndarray  # (n_blocks, ppt, ppt) int32 ps

    @property
    def n_pmt(self) -> int:
        return int(self.pos.shape[0])

    def adjacency(self) -> np.ndarray:
        """(ppt, ppt) uint8, 1 = "adjacent PMTs" (SC) of one tower -- DESIGN.md reading R21: two PMTs of
        the same floor at that floor's smallest inter-PMT distance (cross arm: the two at 3*sqrt(2) m; bar: the
        neighbours at 1.2 m).  Input data for tt_pair_seeds, like the causality table."""
        ppt = self.pmts_per_tower
        pos, fl = self.pos[:ppt], self.floor[:ppt]
        d = np.linalg.norm(pos[:, None, :] - pos[None, :, :], axis=2)
        same = (fl[:, None] == fl[None, :]) & ~np.eye(ppt, dtype=bool)
        out = np.zeros((ppt, ppt), dtype=np.uint8)
        for f in np.unique(fl):
            m = same & (fl[:, None] == f)
            if m.any():
                out[m & (d <= d[m].min() + 1e-9)] = 1
        return out

    def dense_table(self) -> np.ndarray:
        """(P,P) int32 table, -1 where the tower pair is unconnected (small geometries only)."""
        P, ppt = self.n_pmt, self.pmts_per_tower
        out = np.full((P, P), -1, dtype=np.int32)
        for ta in range(self.n_tower):
            for tb in range(self.n_tower):
                b = int(self.pair_block[ta * self.n_tower + tb])
                if b >= 0:
                    out[ta * ppt:(ta + 1) * ppt, tb * ppt:(tb + 1) * ppt] = self.blocks[b]
        return out


def dtmax_ps(d_m: np.ndarray) -> np.ndarray:
    """Causality bound for a PMT pair at distance d (R16): llround((d*n/c + 20 ns) * 1e12)."""
    return np.rint((np.asarray(d_m, dtype=np.float64) * N_WATER / C_LIGHT + LC_SLACK_S) * 1e12).astype(np.int64)


def _tower_local_positions(kind: str) -> tuple[np.ndarray, int, int]:
    """PMT positions of one tower about its axis."""
    if kind == "nemo":
        floors, dz = 8, 40.0
        xy = [(3.0, 0.0), (-3.0, 0.0), (0.0, 3.0), (0.0, -3.0)]  # ends of a 6 m cross arm
    elif kind == "km3":
        floors, dz = 14, 20.0
        xy = [(-3.0 + 1.2 * k, 0.0) for k in range(6)]  # 6 PMTs on a 6 m bar
    else:
        raise ValueError(kind)
    pos = np.array([(x, y, f * dz) for f in range(floors) for (x, y) in xy], dtype=np.float64)
    return pos, floors, len(xy)


def make_geometry(kind: str, nx: int = 1, ny: int = 1, pitch: float = 90.0) -> Geometry:
    """kind in {'nemo','km3'}; nx*ny towers on a square grid of the given pitch."""
    local, floors, ppf = _tower_local_positions(kind)
    ppt = local.shape[0]
    n_tower = nx * ny
    origins = np.array([(ix * pitch, iy * pitch, 0.0) for ix in range(nx) for iy in range(ny)], dtype=np.float64)
    pos = (origins[:, None, :] + local[None, :, :]).reshape(-1, 3)
    tower = np.repeat(np.arange(n_tower, dtype=np.int32), ppt)
    floor_local = np.repeat(np.arange(floors), ppf)
    floor = (tower.astype(np.int64) * floors + np.tile(floor_local, n_tower)).astype(np.uint16)
    # one dense block per distinct tower offset within range
    offsets: dict[tuple[int, int], int] = {}
    blocks: list[np.ndarray] = []
    pair_block = np.full(n_tower * n_tower, -1, dtype=np.int32)
    for ax in range(nx):
        for ay in range(ny):
            for bx in range(nx):
                for by in range(ny):
                    dx, dy = bx - ax, by - ay
                    if pitch * math.hypot(dx, dy) > TOWER_RANGE_M:
                        continue
                    key = (dx, dy)
                    if key not in offsets:
                        shift = np.array([dx * pitch, dy * pitch, 0.0])
                        d = np.linalg.norm(local[:, None, :] - (local[None, :, :] + shift), axis=2)
                        offsets[key] = len(blocks)
                        blocks.append(dtmax_ps(d).astype(np.int32))
                    pair_block[(ax * ny + ay) * n_tower + (bx * ny + by)] = offsets[key]
    name = f"{kind}{'' if n_tower == 1 else f'x{n_tower}'}"
    return Geometry(name, pos, tower, floor, n_tower, ppt, pair_block, np.stack(blocks))


@dataclass
class Params:
    """Trigger parameters (BASELINE.json configs[0]); mirrors tt_params in include/tt.h."""
    q_thresh: int = 300  # 0.01 p.e.
    lc_window_ps: int = 20_000
    l2_window_ps: int = 3_000_000
    l2_multiplicity: int = 5
    l2_mode: int = 0  # 0 clique, 1 star
    event_half_ps: int = 3_000_000


@dataclass
class Workload:
    name: str
    hits: np.ndarray  # HIT_DTYPE, PMT-major runs
    seg_offsets: np.ndarray  # uint32 [n_seg+1]
    run_offsets: np.ndarray  # uint32 [n_runs+1]
    geometry: Geometry
    params: Params
    track_id: np.ndarray  # int32 [n], -1 = background (truth; never given to the library)
    slice_ms: float = 200.0
    n_slices: int = 1  # number of 200 ms slices the workload represents
    meta: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.hits.shape[0])


def draw_charges(rng: np.random.Generator, n: int) -> np.ndarray:
    """0.95 Gaussian(1.0, 0.35) p.e. + 0.05 Exponential(mean 2 p.e.), clipped, in 0.01 p.e. (u16)."""
    q = rng.normal(1.0, 0.35, size=n)
    tail = rng.random(n) < 0.05
    nt = int(tail.sum())
    q[tail] = rng.exponential(2.0, size=nt)
    return np.rint(np.clip(q, 0.05, 655.35) * 100.0).astype(np.uint16)


def _track_hits(rng: np.random.Generator, geo: Geometry, n_tracks: int, t_lo: int, t_hi: int):
    """Straight muon tracks. Returns (pmt, t_ps, charge, track) arrays."""
    pos = geo.pos
    lo = pos.min(axis=0) - 50.0
    hi = pos.max(axis=0) + 50.0
    tan_c = math.sqrt(N_WATER * N_WATER - 1.0)  # tan(theta_c), cos(theta_c) = 1/n
    pm_l, t_l, q_l, k_l = [], [], [], []
    margin = min(5_000_000, max(0, (t_hi - t_lo) // 4))
    for k in range(n_tracks):
        p0 = lo + rng.random(3) * (hi - lo)
        cz = rng.uniform(-1.0, 1.0)
        ph = rng.uniform(0.0, 2.0 * math.pi)
        s = math.sqrt(max(0.0, 1.0 - cz * cz))
        u = np.array([s * math.cos(ph), s * math.sin(ph), cz])
        t0 = int(rng.integers(t_lo + margin, max(t_lo + margin + 1, t_hi - margin)))
        rel = pos - p0
        z = rel @ u
        rho = np.linalg.norm(rel - z[:, None] * u[None, :], axis=1)
        rho = np.maximum(rho, 0.1)
        mu = np.minimum(50.0, (40.0 / rho) * np.exp(-rho / 60.0))
        npe = rng.poisson(mu)
        sel = np.nonzero(npe >= 1)[0]
        if sel.size == 0:
            continue
        tt = t0 + np.rint(((z[sel] + rho[sel] * tan_c) / C_LIGHT) * 1e12 + rng.normal(0.0, 1000.0, size=sel.size)).astype(np.int64)
        kk = npe[sel].astype(np.float64)
        q = kk * rng.normal(1.0, 0.35 / np.sqrt(kk))
        qq = np.rint(np.clip(q, 0.05, 655.35) * 100.0).astype(np.uint16)
        ok = (tt >= t_lo) & (tt < t_hi)
        pm_l.append(sel[ok].astype(np.int64)); t_l.append(tt[ok]); q_l.append(qq[ok])
        k_l.append(np.full(int(ok.sum()), k, dtype=np.int32))
    if not pm_l:
        z = np.zeros(0, dtype=np.int64)
        return z, z.copy(), np.zeros(0, dtype=np.uint16), np.zeros(0, dtype=np.int32)
    return np.concatenate(pm_l), np.concatenate(t_l), np.concatenate(q_l), np.concatenate(k_l)


def make_segment(geo: Geometry, rates_hz: np.ndarray, t0_ps: int, T_ps: int, n_sub: int,
                 n_tracks: int, seed: int):
    """One independent segment: per-PMT streams over [t0, t0+T), cut into n_sub consecutive
    sub-slices (five 200 ms slices packed into one 1 s buffer); runs are
    sub-slice-major then PMT-major and each run is time-ordered.

    Returns (hits, run_lengths[n_sub*P], track_id)."""
    P = geo.n_pmt
    ss = np.random.SeedSequence(seed)
    r_time, r_charge, r_track = (np.random.default_rng(s) for s in ss.spawn(3))
    rates = np.broadcast_to(np.asarray(rates_hz, dtype=np.float64), (P,))
    counts = r_time.poisson(rates * (T_ps * 1e-12))
    n_bg = int(counts.sum())
    sub_ps = T_ps // n_sub
    assert sub_ps * n_sub == T_ps
    pm = np.repeat(np.arange(P, dtype=np.int64), counts)
    trel = r_time.integers(0, T_ps, size=n_bg, dtype=np.int64)
    # combined key = run * T + t_rel, run = sub*P + pmt: one global sort orders every run in time
    key = ((trel // sub_ps) * P + pm) * T_ps + trel
    del pm
    key.sort()
    q = draw_charges(r_charge, n_bg)
    trk = np.full(n_bg, -1, dtype=np.int32)
    if n_tracks > 0:
        tp, tt, tq, tk = _track_hits(r_track, geo, n_tracks, t0_ps, t0_ps + T_ps)
        if tp.size:
            trl = tt - t0_ps
            tkey = ((trl // sub_ps) * P + tp) * T_ps + trl
            o = np.argsort(tkey, kind="stable")
            tkey, tq, tk = tkey[o], tq[o], tk[o]
            at = np.searchsorted(key, tkey, side="right")
            key = np.insert(key, at, tkey)
            q = np.insert(q, at, tq)
            trk = np.insert(trk, at, tk)
    n = key.shape[0]
    run = key // T_ps
    trel = key - run * T_ps
    del key
    hits = np.zeros(n, dtype=HIT_DTYPE)
    hits["t_ps"] = trel + t0_ps
    pmt = (run % P)
    hits["pmt_id"] = pmt.astype(np.uint16)
    hits["floor"] = geo.floor[pmt]
    hits["charge"] = q
    run_len = np.bincount(run, minlength=n_sub * P).astype(np.int64)
    return hits, run_len, trk


# (geometry kind, nx, ny, rate spec, T_ms, n_sub, n_seg, tracks per segment, N)
CONFIGS = {
    0: dict(name="cfg0 NEMO Phase II tower, 32 PMTs, 55 kHz, 1 x 200 ms", kind="nemo", nx=1, ny=1,
            rate="55k", T_ms=200, n_sub=1, n_seg=1, tracks=20, N=4),
    1: dict(name="cfg1 KM3NeT-It tower, 84 PMTs, 55 kHz, 1 x 200 ms", kind="km3", nx=1, ny=1,
            rate="55k", T_ms=200, n_sub=1, n_seg=1, tracks=50, N=5),
    2: dict(name="cfg2 KM3NeT-It burst, 300 kHz + 10% PMTs at 1 MHz, 5 x 200 ms", kind="km3", nx=1, ny=1,
            rate="burst", T_ms=1000, n_sub=5, n_seg=1, tracks=200, N=5),
    3: dict(name="cfg3 64 independent KM3NeT-It slices, 55 kHz", kind="km3", nx=1, ny=1,
            rate="55k", T_ms=200, n_sub=1, n_seg=64, tracks=50, N=5),
    4: dict(name="cfg4 100 KM3NeT-It towers (8400 PMTs), 55 kHz, 1 x 200 ms", kind="km3", nx=10, ny=10,
            rate="55k", T_ms=200, n_sub=1, n_seg=1, tracks=1000, N=5),
    # not a BASELINE.json config: the "8 towers of KM3NeT-It" of the paper's proposed DAQ (one TGPU per
    # tower), the workload of the by-tower sharded path; a 4 x 2 grid at the same 90 m pitch
    5: dict(name="8 KM3NeT-It towers (672 PMTs, PAPER.md:81), 55 kHz, 1 x 200 ms", kind="km3", nx=4, ny=2,
            rate="55k", T_ms=200, n_sub=1, n_seg=1, tracks=100, N=5),
}


def make_config(cfg: int, time_scale: float = 1.0, seg_scale: float = 1.0, seed_offset: int = 0,
                t0_ps: int = 0) -> Workload:
    """Build BASELINE.json configs[cfg].  time_scale < 1 shortens the slice duration (and the
    track count) for oracle-speed parity cases; seg_scale < 1 reduces the number of segments."""
    c = CONFIGS[cfg]
    geo = make_geometry(c["kind"], c["nx"], c["ny"])
    P = geo.n_pmt
    T_ps = int(round(c["T_ms"] * 1e9 * time_scale))
    T_ps -= T_ps % c["n_sub"]
    n_seg = max(1, int(round(c["n_seg"] * seg_scale)))
    n_tracks = max(1, int(math.ceil(c["tracks"] * time_scale)))
    base = BASE_SEED + 1000 * cfg + seed_offset
    if c["rate"] == "55k":
        rates = np.full(P, 55e3)
    else:
        rates = np.full(P, 300e3)
        hot = np.random.default_rng(base + 500).permutation(P)[: P // 10]  # floor(10 %) of PMTs
        rates[hot] = 1e6
    hits_l, runlen_l, trk_l, seg_off = [], [], [], [0]
    for s in range(n_seg):
        h, rl, tk = make_segment(geo, rates, t0_ps, T_ps, c["n_sub"], n_tracks, base + s)
        hits_l.append(h); runlen_l.append(rl); trk_l.append(tk)
        seg_off.append(seg_off[-1] + h.shape[0])
    hits = hits_l[0] if n_seg == 1 else np.concatenate(hits_l)
    trk = trk_l[0] if n_seg == 1 else np.concatenate(trk_l)
    n = hits.shape[0]
    assert n < 2**32
    hits["pad"] = (np.arange(n, dtype=np.int64) & 0xFFFF).astype(np.uint16)  # tracer: low input-index bits
    run_off = np.zeros(sum(len(r) for r in runlen_l) + 1, dtype=np.int64)
    np.cumsum(np.concatenate(runlen_l), out=run_off[1:])
    params = Params(l2_multiplicity=c["N"])
    return Workload(c["name"], hits, np.asarray(seg_off, dtype=np.uint32), run_off.astype(np.uint32), geo, params,
                    trk, slice_ms=200.0, n_slices=max(1, int(round(c["T_ms"] * time_scale / 200.0))) * n_seg,
                    meta=dict(cfg=cfg, time_scale=time_scale, n_seg=n_seg, T_ps=T_ps, rates=rates))


def shuffled(w: Workload, seed: int = 7) -> tuple[np.ndarray, np.ndarray]:
    """A fully shuffled copy (within each segment) for the run_offsets = NULL path; returns
    (hits, permutation used)."""
    rng = np.random.default_rng(seed)
    out = w.hits.copy()
    perm = np.arange(w.n, dtype=np.int64)
    for s in range(len(w.seg_offsets) - 1):
        a, b = int(w.seg_offsets[s]), int(w.seg_offsets[s + 1])
        p = rng.permutation(b - a) + a
        out[a:b] = w.hits[p]
        perm[a:b] = p
    return out, perm


RAW_DTYPE = np.dtype([("t_ps", "<i8"), ("pmt_id", "<u2"), ("floor", "<u2"), ("n_samples", "<u2"), ("pad", "<u2")])


def make_raw(w: Workload, frame_ps: int = 100_000_000, seed: int = 11):
    """The workload as the RAW stream the paper's preparation step starts from ("a header with the GPS
    time and geometry information, followed by a sampled charge waveform with a variable size"; 28 bytes on average,
    PAPER.md:21).  Synthetic format (R24): 16-byte headers in ARRIVAL order + all waveforms concatenated in
    the same order.  Arrival order inside a slice: frame by frame (frame = t // frame_ps, the Hit Manager merging the
    PMT streams), PMT by PMT inside a frame, so every PMT's hits stay time-ordered but the stream is not
    PMT-major.  A slice = n_pmt consecutive runs of the workload (a 200 ms sub-slice of one tower or tower array).
    The waveform of a hit has 1 + Poisson(5) samples (16 + 2 * 6 = 28 bytes per hit on average) that sum to its charge.
    Returns (raw headers, samples uint16, slice_offsets uint32)."""
    P = w.geometry.n_pmt
    n_runs = len(w.run_offsets) - 1
    assert n_runs % P == 0, "runs are (slice, PMT)"
    n_slices = n_runs // P
    slice_off = np.asarray(w.run_offsets[::P], dtype=np.uint32)
    assert len(slice_off) == n_slices + 1
    h = w.hits
    n = w.n
    slice_id = np.repeat(np.arange(n_slices, dtype=np.int64), np.diff(slice_off.astype(np.int64)))
    frame = h["t_ps"] // frame_ps
    # stable: inside (slice, frame, pmt) the workload's order (= time order of that PMT) is kept
    order = np.lexsort((h["pmt_id"], frame, slice_id))
    ha = h[order]
    rng = np.random.default_rng(seed)
    ns = (1 + rng.poisson(5.0, size=n)).astype(np.uint16)
    raw = np.zeros(n, dtype=RAW_DTYPE)
    raw["t_ps"], raw["pmt_id"], raw["floor"], raw["pad"], raw["n_samples"] = ha["t_ps"], ha["pmt_id"], ha["floor"], ha["pad"], ns
    # pulse shape: sample j of a waveform of m samples gets floor(charge * wgt_j), wgt ~ a fixed falling shape; what
    # the floors lose goes to sample 0, so the samples sum to the charge exactly
    woff = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(ns, out=woff[1:])
    total = int(woff[-1])
    hit_of = np.repeat(np.arange(n, dtype=np.int64), ns)
    j = np.arange(total, dtype=np.int64) - woff[hit_of]
    m = ns[hit_of].astype(np.float64)
    wgt = (m - j) / (m * (m + 1) / 2.0)  # m, m-1, ..., 1 over their sum
    c = ha["charge"].astype(np.int64)
    samples = np.floor(c[hit_of] * wgt).astype(np.int64)
    lost = c - np.bincount(hit_of, weights=samples, minlength=n).astype(np.int64)
    samples[woff[:-1]] += lost
    assert samples.min() >= 0 and samples.max() <= 65535
    return raw, samples.astype(np.uint16), slice_off
