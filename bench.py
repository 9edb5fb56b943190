#!/usr/bin/env python
"""bench.py -- sort + trigger + event extraction throughput on B200 (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

One "step" = one pass of the whole hot path (tt_sort_slice -> tt_trigger_slice -> tt_extract_events
with INEVT tagging) over one synthetic workload already resident in HBM.  Default workload:
BASELINE.json configs[4] (100 KM3NeT-It towers, 8400 PMTs, one 200 ms slice, ~92.6 M hits, 1.48 GB --
larger than the 126 MB L2, so no flush is needed between steps).  N > 1: one process per GPU
(torchrun), each rank processes its own slice (different seed), no collective on the data path
("successive time slices are sent to different" trigger nodes): weak scaling.

Prints ONE JSON line (rank 0).  --impl reference times the CPU oracle (oracle/) on a bounded sample.
"""
from __future__ import annotations

import argparse
import ctypes
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "hits/s sorted+triggered on 1 B200 (ms per 200 ms slice) and % of HBM roofline"
ALG_BYTES_PIPELINE = 50  # sort 16 r + 16 w, trigger 16 r + ~2 w
ALG_BYTES = {"sort": 32, "trig": 18, "ev": 2}
# oracle sample per config (time_scale, seg_scale): the FULL config everywhere (cfg4: ~22 s of one host core)
ORACLE_SAMPLE = {0: (1.0, 1.0), 1: (1.0, 1.0), 2: (1.0, 1.0), 3: (1.0, 1.0), 4: (1.0, 1.0)}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region.  NVML is polled from a thread every ~0.5 ms (the timed
    region of the small configs lasts a few ms, shorter than one `nvidia-smi -lms 100` poll); `nvidia-smi` is the
    fallback when NVML cannot be loaded."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []
        self.nvml, self.handle, self.thread, self.run = None, None, None, False
        self.sm, self.mask, self.sm_max = [], 0, None

    def _nvml_open(self):
        import pynvml
        pynvml.nvmlInit()
        h = None
        try:  # the CUDA ordinal is not the NVML index under CUDA_VISIBLE_DEVICES: go through the UUID
            import torch
            h = pynvml.nvmlDeviceGetHandleByUUID("GPU-" + str(torch.cuda.get_device_properties(self.index).uuid))
        except Exception:
            h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
        self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
        pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)
        self.nvml, self.handle = pynvml, h

    def _poll(self):
        nv, h = self.nvml, self.handle
        while self.run:
            try:
                self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                self.mask |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
            except Exception:
                pass
            time.sleep(0.0005)

    def start(self):
        """Called right before the timed region: only samples taken from here on count."""
        try:
            self._nvml_open()
            self.run = True
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
            time.sleep(0.3)
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.nvml is not None:
            self.run = False
            self.thread.join(timeout=1.0)
            reasons = sorted(nm for bit, nm in self.REASONS.items() if self.mask & bit)
            return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": self.sm_max,
                    "reasons": reasons, "samples": len(self.sm), "source": "nvml"}
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "source": "nvidia-smi"}


def make_workload(cfg: int, rank: int, scale: float):
    from paper_1411_3968_b200 import workload as W

    if scale == 1.0:
        return W.make_config(cfg, seed_offset=rank)  # = sharding.workload_seed_offset(rank, 0, world)
    return W.make_config(cfg, time_scale=scale, seed_offset=rank)


def time_oracle(cfg: int, nthreads: int = 1):
    """The oracle as it stands, single thread, on a bounded sample of config `cfg`."""
    import oracle
    from paper_1411_3968_b200 import workload as W

    ts, ss = ORACLE_SAMPLE[cfg]
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    g, p = w.geometry, w.params
    oracle.build()
    t0 = time.perf_counter()
    srt, _ = oracle.sort(w.hits, w.seg_offsets)
    t1 = time.perf_counter()
    tr = oracle.trigger(srt, w.seg_offsets, g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks,
                        q_thresh=p.q_thresh, lc_window_ps=p.lc_window_ps, l2_window_ps=p.l2_window_ps,
                        l2_multiplicity=p.l2_multiplicity, l2_mode=p.l2_mode, event_half_ps=p.event_half_ps)
    t2 = time.perf_counter()
    fl = tr.flags.copy()
    oracle.events(srt, w.seg_offsets, tr.seeds, event_half_ps=p.event_half_ps, flags=fl)
    t3 = time.perf_counter()
    sample = (f"cfg{cfg} at time_scale={ts}, seg_scale={ss}: {w.n} hits; sort {1e3 * (t1 - t0):.0f} ms, "
              f"trigger {1e3 * (t2 - t1):.0f} ms, events {1e3 * (t3 - t2):.0f} ms")
    return w.n, t3 - t0, sample, w.name


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    for _ in range(args.warmup):
        pass  # the oracle has no warm state worth priming beyond the build
    times, n, sample, name = [], 0, "", ""
    for _ in range(max(1, args.steps)):
        n, dt, sample, name = time_oracle(args.config)
        times.append(dt)
        if sum(times) > 150:
            break
    dt = float(np.mean(times))
    v = n / dt
    slices = {0: 1, 1: 1, 2: 5, 3: 64, 4: 1}[args.config]
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": "hits/s", "n_gpus": args.gpus, "steps": len(times),
        "warmup": args.warmup, "ms_per_step": 1e3 * dt, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": name, "sample": sample, "slices_full_config": slices},
        "cpu_baseline": {"value": v, "unit": "hits/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "hits/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def time_oracle_all_cores(cfg: int):
    """the oracle on ALL host cores where the split is exact -- independent segments (cfg3), else time
    chunks with a 6.02 us halo (chunking invariance P12) -- each chunk through sort -> trigger -> events in its own
    thread (the C++ oracle releases the GIL).  Same bounded sample as the single-core figure."""
    import oracle
    from concurrent.futures import ThreadPoolExecutor
    from paper_1411_3968_b200 import workload as W

    ts, ss = ORACLE_SAMPLE[cfg]
    w = W.make_config(cfg, time_scale=ts, seg_scale=ss)
    g, p = w.geometry, w.params
    cores = os.cpu_count() or 1
    halo = p.event_half_ps + p.l2_window_ps + p.lc_window_ps
    seg = np.asarray(w.seg_offsets, dtype=np.int64)
    chunks = []
    if len(seg) - 1 >= cores:
        for s in range(len(seg) - 1):
            chunks.append(np.ascontiguousarray(w.hits[seg[s]:seg[s + 1]]))
        how = f"{len(chunks)} independent segments"
    else:
        t = w.hits["t_ps"]
        lo, hi = int(t.min()), int(t.max()) + 1
        nch = cores * 2
        edges = np.linspace(lo, hi, nch + 1).astype(np.int64)
        for k in range(nch):
            sel = (t >= edges[k] - halo) & (t < edges[k + 1] + halo)
            chunks.append(np.ascontiguousarray(w.hits[sel]))  # input order = run-major: the oracle's stable order
        how = f"{nch} time chunks with a {halo} ps halo each side (the halo hits are processed twice)"
    oracle.build()

    def work(h):
        so = np.array([0, len(h)], dtype=np.uint32)
        srt, _ = oracle.sort(h, so)
        tr = oracle.trigger(srt, so, g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks, q_thresh=p.q_thresh,
                            lc_window_ps=p.lc_window_ps, l2_window_ps=p.l2_window_ps, l2_multiplicity=p.l2_multiplicity,
                            l2_mode=p.l2_mode, event_half_ps=p.event_half_ps)
        fl = tr.flags.copy()
        oracle.events(srt, so, tr.seeds, event_half_ps=p.event_half_ps, flags=fl)
        return len(tr.seeds)

    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=cores) as ex:
        list(ex.map(work, chunks))
    dt = time.perf_counter() - t0
    return {"value": w.n / dt, "unit": "hits/s", "cores": cores, "kind": "oracle", "split": how,
            "sample": f"cfg{cfg} at time_scale={ts}, seg_scale={ss}: {w.n} hits in {1e3 * dt:.0f} ms"}


def _cuda_time(fn, reps):
    import torch

    fn()
    torch.cuda.synchronize()
    b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    b0.record()
    for _ in range(reps):
        fn()
    b1.record()
    torch.cuda.synchronize()
    return b0.elapsed_time(b1) / reps


def time_radix(B, run, peak):
    """tt_sort_slice with run_offsets = NULL (arbitrary input: the LSD radix path) on this run's hits."""
    import torch

    st = torch.zeros(1, dtype=torch.int32, device="cuda")
    ws = {}

    def go():
        ws["r"] = B.tt_sort_slice(run.d_in, run.d_out, None, run.seg, None, st, ws.get("r"))

    ms = _cuda_time(go, 3)
    return {"workload": run.w.name, "hits": run.n, "ms": ms, "hits_per_s": run.n / (ms * 1e-3),
            "alg_bytes_per_hit": 32, "frac": 32.0 * run.n / (ms * 1e-3) / 1e9 / peak,
            "note": "8-bit LSD passes over the varying key bits + one gather: ~5 passes x (12 B read + 24 B moved)"}


def time_library_sort(B, run):
    """Context, not a target and not on the product path: the library radix sort (torch.sort = CUB) of the int64 time keys of
    this run's hits (keys + index; the 16-byte records would still have to be gathered through the index) next to this
    repo's sort alone, tt_sort_slice with the permutation output, on the same device buffers."""
    import torch

    keys = run.d_in[:, 0].contiguous()
    ms_lib = _cuda_time(lambda: torch.sort(keys, stable=True), 3)
    del keys
    st = torch.zeros(1, dtype=torch.int32, device="cuda")
    perm = torch.empty(run.n, dtype=torch.int32, device="cuda")
    ws = {}

    def go():
        ws["s"] = B.tt_sort_slice(run.d_in, run.d_out, perm, run.seg, run.runs, st, ws.get("s"))

    ms_ours = _cuda_time(go, 3)
    return {"workload": run.w.name, "hits": run.n, "library_sort_keys_and_index_ms": ms_lib,
            "tt_sort_slice_records_and_perm_ms": ms_ours,
            "note": "torch.sort(int64 keys, stable) ignores the per-PMT order of the input (PAPER.md:51-53 uses it) and "
                    "moves 8-byte keys + 8-byte indices; tt_sort_slice moves the 16-byte records and a 4-byte permutation"}


def time_streams(B, run, steps):
    """BASELINE.json configs[3]: "64 independent slices processed concurrently on one GPU through CUDA streams".  The
    same work as run.step(), but one call chain per segment (n_seg = 1) on its own stream, against the single
    segmented call the timed step uses (compare the two).  Direct launches both ways."""
    import torch

    w = run.w
    seg = np.asarray(w.seg_offsets, dtype=np.int64)
    ro = np.asarray(w.run_offsets, dtype=np.int64)
    n_seg = len(seg) - 1
    streams = [torch.cuda.Stream() for _ in range(n_seg)]
    parts = []
    for s in range(n_seg):
        a, b = int(seg[s]), int(seg[s + 1])
        r0, r1 = int(np.searchsorted(ro, a, side="left")), int(np.searchsorted(ro, b, side="left"))
        cap = max((b - a) // 4, 1024)
        parts.append(dict(a=a, b=b, seg=B.Offsets(np.array([0, b - a], dtype=np.uint32)),
                          runs=B.Offsets((ro[r0:r1 + 1] - a).astype(np.uint32)),
                          seeds=torch.zeros(cap, dtype=torch.int32, device="cuda"),
                          ev=torch.zeros((cap, 4), dtype=torch.int64, device="cuda"),
                          cnt=torch.zeros(4, dtype=torch.int32, device="cuda"), ws={}))

    def step():
        start = torch.cuda.Event()
        start.record()
        for st, pt in zip(streams, parts):
            st.wait_event(start)
            with torch.cuda.stream(st):
                a, b, c, ws = pt["a"], pt["b"], pt["cnt"], pt["ws"]
                c.zero_()
                ws["f"] = B.tt_sort_trigger_slice(run.d_in[a:b], run.d_out[a:b], None, pt["seg"], pt["runs"], run.geo, run.prm,
                                                  run.d_flags[a:b], pt["seeds"], c[0:1], c[2:3], ws.get("f"))
                ws["e"] = B.tt_extract_events(run.d_out[a:b], pt["seg"], pt["seeds"], c[0:1], run.prm, pt["ev"], c[1:2],
                                              run.d_flags[a:b], None, None, c[2:3], ws.get("e"))
        for st in streams:
            torch.cuda.current_stream().wait_stream(st)

    for _ in range(2):
        step()
    torch.cuda.synchronize()
    ns = sum(int(pt["cnt"][0].item()) for pt in parts)
    ms_streams = _cuda_time(step, max(2, min(steps, 5)))
    B.prof_enable(False)
    ms_one = _cuda_time(run.step, max(2, min(steps, 5)))
    return {"segments": n_seg, "ms_per_step_one_stream_per_segment": ms_streams, "ms_per_step_one_segmented_call": ms_one,
            "n_seeds_streams": ns,
            "note": "direct launches both ways (no CUDA graph); the default timed step is the segmented call replayed as a graph"}


def time_tower_shard(B, w, geo, prm, ranks):
    """NEXT-4: ONE cfg4 slice sharded by tower over `ranks` GPUs with one exchange of L1 hits.  This box has
    one GPU, so the ranks are EMULATED one after the other (no kernel waits on another rank): what is reported is the
    per-rank device time of the two phases and the bytes a rank would all-gather -- not a multi-GPU measurement."""
    import torch

    from paper_1411_3968_b200 import sharding

    g = w.geometry
    parts = sharding.split_runs_by_tower(w.run_offsets, g.pmts_per_tower, g.n_tower, ranks)
    d_parts = [(B.hits_to_device(np.ascontiguousarray(w.hits[a:b])), B.Offsets(ro)) for a, b, ro in parts]

    def ev_pair():
        return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def phase1():
        out, tms = [], []
        for r, (d_h, ro) in enumerate(d_parts):
            e0, e1 = ev_pair()
            e0.record()
            out.append(sharding.tower_local(B, r, d_h, ro, prm))  # ends with the read-back of the rank's L1 count
            e1.record()
            torch.cuda.synchronize()
            tms.append(e0.elapsed_time(e1))
        return out, tms

    phase1()  # warm-up (allocator, plans)
    states, t_local = phase1()
    gathered = torch.cat([s["l1"] for s in states], dim=0)
    offs = [0]
    for s in states:
        offs.append(offs[-1] + int(s["l1"].shape[0]))
    t_global, seeds = [], 0
    for rep in range(3):
        for s in states[:2]:  # the global phase does the same work on every rank: two of them are timed
            e0, e1 = ev_pair()
            e0.record()
            res = sharding.tower_global(B, s, gathered, offs, geo, prm, download=False)
            e1.record()
            torch.cuda.synchronize()
            if rep:
                t_global.append(e0.elapsed_time(e1))
            seeds = int(res["d_counts"].cpu().numpy().view(np.uint32)[0])
    return {"ranks_emulated": ranks, "hits": w.n, "l1_records_total": int(gathered.shape[0]),
            "all_gather_bytes_per_rank": int(16 * gathered.shape[0]),
            "local_phase_ms_max_over_ranks": max(t_local), "global_phase_ms": max(t_global), "global_seeds": seeds,
            "note": "ranks emulated sequentially on one GPU, device-resident input and output (CUDA events; buffer "
                    "allocation inside); a step of the sharded path = local phase + all-gather + global phase; "
                    "tests/test_gpu_towers.py checks the result against the oracle on the whole detector"}


def time_prepare(B, peak):
    """tt_prepare_slice (NEXT-3) on the raw stream of a cfg2-shaped burst: five 200 ms sub-slices at
    half the duration (15 M raw hits, 28 B each on average) -> PMT-major 16-byte records + run offsets."""
    import torch

    from paper_1411_3968_b200 import workload as W

    w = W.make_config(2, time_scale=0.5)
    raw, samples, slice_off = W.make_raw(w)
    n = len(raw)
    d_raw = torch.from_numpy(raw.view(np.int64).reshape(-1, 2).copy()).cuda()
    d_samples = torch.from_numpy(samples.view(np.int16).copy()).cuda()
    sl = B.Offsets(slice_off)
    d_out = torch.empty((n, 2), dtype=torch.int64, device="cuda")
    d_runs = torch.zeros(sl.count * w.geometry.n_pmt + 1, dtype=torch.int32, device="cuda")
    st = torch.zeros(1, dtype=torch.int32, device="cuda")
    ws = {}

    def go():
        ws["p"] = B.tt_prepare_slice(d_raw, d_samples, sl, w.geometry.n_pmt, d_out, d_runs, st, ws.get("p"))

    ms = _cuda_time(go, 5)
    assert B.hits_to_host(d_out).tobytes() == np.ascontiguousarray(w.hits).tobytes(), "prepare differs from the generator"
    byt = raw.nbytes + samples.nbytes + 16 * n
    return {"workload": w.name + " x 0.5", "raw_hits": n, "raw_bytes_per_hit": (raw.nbytes + samples.nbytes) / n,
            "ms": ms, "hits_per_s": n / (ms * 1e-3), "alg_bytes": byt, "frac": byt / (ms * 1e-3) / 1e9 / peak,
            "paper": "200-300 ms of CPU time per second of data, transfer included (PAPER.md:71)"}


class Run:
    """One workload on the device with its buffers; step() = one pass of the whole hot path."""

    def __init__(self, B, cfg, rank, scale, fused):
        import torch

        self.B, self.fused = B, fused
        self.w = w = make_workload(cfg, rank, scale)
        self.n = n = w.n
        g = w.geometry
        self.geo = B.Geometry(g.n_pmt, g.n_tower, g.pmts_per_tower, g.pair_block, g.blocks)
        p = w.params
        self.prm = B.make_params(p.q_thresh, p.lc_window_ps, p.l2_window_ps, p.l2_multiplicity, p.l2_mode, p.event_half_ps)
        self.seg, self.runs = B.Offsets(w.seg_offsets), B.Offsets(w.run_offsets)
        self.d_in = B.hits_to_device(w.hits)
        self.d_out = torch.empty_like(self.d_in)
        self.seed_cap = self.event_cap = max(n // 4, 1024)
        self.d_flags = torch.zeros(n, dtype=torch.uint8, device="cuda")
        self.d_seeds = torch.zeros(self.seed_cap, dtype=torch.int32, device="cuda")
        self.d_ev = torch.zeros((self.event_cap, 4), dtype=torch.int64, device="cuda")
        self.d_cnt = torch.zeros(4, dtype=torch.int32, device="cuda")  # n_seeds, n_events, status, spare
        self.ws = {}

    def step(self):
        B, ws, c = self.B, self.ws, self.d_cnt
        d_ns, d_ne, d_st = c[0:1], c[1:2], c[2:3]
        c.zero_()
        if self.fused:
            ws["f"] = B.tt_sort_trigger_slice(self.d_in, self.d_out, None, self.seg, self.runs, self.geo, self.prm,
                                              self.d_flags, self.d_seeds, d_ns, d_st, ws.get("f"))
        else:
            ws["s"] = B.tt_sort_slice(self.d_in, self.d_out, None, self.seg, self.runs, d_st, ws.get("s"))
            ws["t"] = B.tt_trigger_slice(self.d_out, self.seg, self.geo, self.prm, self.d_flags, self.d_seeds, d_ns, d_st,
                                         ws.get("t"))
        ws["e"] = B.tt_extract_events(self.d_out, self.seg, self.d_seeds, d_ns, self.prm, self.d_ev, d_ne, self.d_flags,
                                      None, None, d_st, ws.get("e"))

    def counts(self):
        c = self.d_cnt.cpu().numpy().view(np.uint32)
        return int(c[0]), int(c[1]), int(c[2])


def timed_steps(B, run, steps, warmup, graph_mode, barrier, sampler=None):
    """W warm-up steps, then exactly `steps` timed steps (CUDA events on the launching stream) -- replayed as a CUDA
    graph when it can be captured -- then a separate profiled pass of direct launches for the per-stage times."""
    import torch

    for _ in range(max(warmup, 3)):
        run.step()
    barrier()
    n_seeds, n_events, status = run.counts()
    graph, graph_note, launches_per_replay = None, None, 0
    if graph_mode in ("on", "auto"):
        try:
            cg = torch.cuda.CUDAGraph()
            lc = B.launch_count()
            with torch.cuda.graph(cg):
                run.step()
            launches_per_replay = B.launch_count() - lc
            cg.replay()
            torch.cuda.synchronize()
            assert run.counts() == (n_seeds, n_events, status), "graph replay differs"
            graph = cg
        except Exception as ex:  # capture not possible here: time the direct launches
            graph, graph_note = None, f"capture failed: {type(ex).__name__}"
            torch.cuda.synchronize()
    go = graph.replay if graph is not None else run.step
    if graph is None:
        B.prof_enable(True)
    l0 = B.launch_count()
    barrier()
    if sampler is not None:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        go()
    e1.record()
    barrier()
    clocks = sampler.stop() if sampler is not None else None
    launches = B.launch_count() - l0 if graph is None else launches_per_replay * steps
    ms_total = e0.elapsed_time(e1)
    if graph is not None:  # stage breakdown from direct launches, outside the timed region
        B.prof_enable(True)
        run.step()         # first profiled step creates the event pool and the pinned counter buffers: not measured
        barrier()
        B.prof_enable(True)  # clears the marks
        for _ in range(steps):
            run.step()
        barrier()
    stages = B.prof_read()
    B.prof_enable(False)
    counters = {k[4:]: v[0] / max(v[1], 1) for k, v in stages.items() if k.startswith("ctr.")}
    stages = {k: v for k, v in stages.items() if not k.startswith("ctr.")}
    per_stage = {k: v[0] / steps for k, v in stages.items()}  # ms per step
    per_launches = {k: v[1] / steps for k, v in stages.items()}
    return dict(ms_step=ms_total / steps, per_stage=per_stage, per_launches=per_launches, counters=counters,
                launches=int(launches), clocks=clocks, graph=graph is not None, graph_note=graph_note,
                n_seeds=n_seeds, n_events=n_events, status=status)


def stage_fracs(per_stage, n, peak):
    """Stage-level roofline fractions: the stage's algorithmic bytes ONCE (sort 32 B/hit whatever the
    number of merge levels, trigger 18 B/hit, events ~2 B/hit) over the summed time of all its kernels."""
    out = {}
    for fam, byt in ALG_BYTES.items():
        ms = sum(v for k, v in per_stage.items() if k.split(".")[0] == fam)
        if ms > 0:
            out[fam] = {"alg_bytes_per_hit": byt, "ms": ms, "achieved": byt * n / (ms * 1e-3) / 1e9,
                        "frac": byt * n / (ms * 1e-3) / 1e9 / peak}
    return out


def run_ours(args):
    import torch

    from paper_1411_3968_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.load()
    fused = args.fused == "on"
    run = Run(B, args.config, rank, args.scale, fused)
    w, n, geo, prm, seg, runs = run.w, run.n, run.geo, run.prm, run.seg, run.runs
    d_out, seed_cap, event_cap = run.d_out, run.seed_cap, run.event_cap

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    m = timed_steps(B, run, args.steps, args.warmup, args.graph, barrier, sampler)
    n_seeds, n_events, status = m["n_seeds"], m["n_events"], m["status"]
    l1_frac = float((run.d_flags & 4).ne(0).float().mean().item())
    inevt_frac = float((run.d_flags & 32).ne(0).float().mean().item())
    clocks, launches, per_stage, counters = m["clocks"], m["launches"], m["per_stage"], m["counters"]
    ms_step_local = m["ms_step"]
    from paper_1411_3968_b200 import sharding

    ms_step, n_total = sharding.reduce_timing(ms_step_local, n, "cuda")  # max over ranks, whole-job hits
    value = n_total / (ms_step * 1e-3)

    # ---- roofline of the dominant kernel (device time from the stage events of the profiled steps) ----
    peak, peak_src = peaks()
    dom = max(per_stage, key=per_stage.get) if per_stage else None
    roof = None
    if dom:
        launches_dom = m["per_launches"][dom]
        fam = dom.split(".")[0]
        # one launch of a merge-level tile kernel moves every hit once: 16 B read + 16 B written (+ 1 flag byte when L1
        # is fused into it).  NOTE: with two merge levels EACH level is credited these bytes here; the stage-level
        # figure below (`stage_frac`) counts the sort's 32 B/hit once, whatever the number of levels.
        alg = ALG_BYTES[fam] * n
        dur_ms = per_stage[dom]
        ach = alg / (dur_ms * 1e-3) / 1e9
        traffic = None  # dram__bytes_read + write per launch from the committed ncu --set full summary of THIS build
        tp = os.path.join(ROOT, "profiles", "traffic.csv")
        if os.path.exists(tp):
            for ln in open(tp).read().splitlines()[1:]:
                f = ln.split(",")
                if len(f) >= 3 and f[0] == f"cfg{args.config}" and f[1] == dom:
                    traffic = float(f[2])
        sf = stage_fracs(per_stage, n, peak)
        roof = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": traffic, "traffic_source": "profiles/traffic.csv: ncu --set full capture of this build (not "
                "measured inside this run; ncu cannot run in the timed process)", "peak_source": peak_src,
                "alg_bytes_per_launch": alg / max(launches_dom, 1), "launches_per_step": launches_dom,
                "kernel_ms_per_step": dur_ms, "share_of_step": dur_ms / ms_step_local,
                "stage_note": "with --fused on the L1 step runs INSIDE the last sort.merge_tile kernel, so its time is "
                              "in the sort family and the trig family holds the edge pass, compaction, L2 and seeds",
                "stage_frac": sf.get(fam, {}).get("frac"), "stages": sf}
    pipe_ach = ALG_BYTES_PIPELINE * n / (ms_step_local * 1e-3) / 1e9  # this rank

    # ---- level-0 N-in-TW trigger (tt_l0_ntw) on the sorted hits of this workload: timed on its
    # own, NOT part of the step above.  N7TW1000 for the 32-PMT tower, N7TW500 otherwise.
    # Algorithmic bytes: 16 B read (AoS record, only the time is used) + 1 B written per hit.
    l0 = None
    if rank == 0:
        l0_n, l0_tw = 7, (1_000_000 if args.config == 0 else 500_000)
        g_multi = w.geometry.n_tower > 1
        l0_src, l0_seg, l0_scope = d_out, seg, "the sorted slice"
        ppt_ = w.geometry.pmts_per_tower
        if g_multi and (len(w.run_offsets) - 1) % ppt_ == 0:
            # The paper applies N7TW500, SC, FC and AFC PER TOWER.  On the time-merged stream of 100
            # towers every window fires and a hit walks the hits of 99 foreign towers, so these legs run on the
            # per-tower streams instead: the same input sorted with one segment per (slice, tower) -- the runs are
            # tower-major, so a tower's 84 runs are contiguous -- and windows / pairs never cross a segment.
            l0_seg = B.Offsets(np.ascontiguousarray(w.run_offsets[::ppt_], dtype=np.uint32))
            l0_src = torch.empty_like(run.d_in)
            st_ = torch.zeros(1, dtype=torch.int32, device="cuda")
            B.tt_sort_slice(run.d_in, l0_src, None, l0_seg, runs, st_)
            torch.cuda.synchronize()
            assert int(st_.item()) == 0
            l0_scope = f"per-tower streams: {l0_seg.count} segments of one (slice, tower) each, sorted by tt_sort_slice"
        d_l0 = torch.empty(n, dtype=torch.uint8, device="cuda")
        d_l0n = torch.zeros(1, dtype=torch.int32, device="cuda")
        for _ in range(3):
            B.tt_l0_ntw(l0_src, l0_seg, l0_n, l0_tw, d_l0, d_l0n)
        torch.cuda.synchronize()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record()
        for _ in range(args.steps):
            B.tt_l0_ntw(l0_src, l0_seg, l0_n, l0_tw, d_l0, d_l0n)
        a1.record()
        torch.cuda.synchronize()
        l0_ms = a0.elapsed_time(a1) / args.steps
        l0_ach = 17.0 * n / (l0_ms * 1e-3) / 1e9
        l0 = {"kernel": "l0_ntw_kernel", "multiplicity": l0_n, "window_ps": l0_tw, "ms": l0_ms,
              "hits_per_s": n / (l0_ms * 1e-3), "alg_bytes_per_hit": 17, "achieved": l0_ach, "peak": peak,
              "unit": "GB/s", "frac": l0_ach / peak, "n_start": int(d_l0n.cpu().numpy().view(np.uint32)[0]),
              "scope": l0_scope,
              "note": "level-0 / DN / pair / combine legs: separate calls, outside the timed step"}
        # the paper's pair seeds (SC / FC / AFC) and its combination with the level-0 windows
        # (PAPER.md:65, 73): tt_pair_seeds 16 B read + 1 B written per hit, tt_l0_combine 2 B read + 1 B written
        gw = w.geometry
        d_adj = torch.from_numpy(gw.adjacency().reshape(-1).copy()).cuda()
        d_pb = torch.empty(n, dtype=torch.uint8, device="cuda")
        d_cd = torch.empty(n, dtype=torch.uint8, device="cuda")
        d_nc = torch.zeros(2, dtype=torch.int32, device="cuda")

        def timed(fn, reps):
            fn()
            torch.cuda.synchronize()
            b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            b0.record()
            for _ in range(reps):
                fn()
            b1.record()
            torch.cuda.synchronize()
            return b0.elapsed_time(b1) / reps

        reps = max(2, min(args.steps, 5))
        ps_ms = timed(lambda: B.tt_pair_seeds(l0_src, l0_seg, d_adj, gw.pmts_per_tower, d_pb), reps)
        cb_ms = timed(lambda: B.tt_l0_combine(d_l0, d_pb, n, l0_n, d_cd, d_nc), reps)
        nc = d_nc.cpu().numpy().view(np.uint32)
        l0["pair_seeds"] = {"kernel": "pair_seeds_kernel", "windows_ps": [20_000, 100_000, 250_000], "ms": ps_ms,
                            "alg_bytes_per_hit": 17, "achieved": 17.0 * n / (ps_ms * 1e-3) / 1e9, "peak": peak,
                            "unit": "GB/s", "frac": 17.0 * n / (ps_ms * 1e-3) / 1e9 / peak}
        l0["combine"] = {"kernel": "l0_combine_kernel", "ms": cb_ms, "alg_bytes_per_hit": 3,
                         "achieved": 3.0 * n / (cb_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                         "frac": 3.0 * n / (cb_ms * 1e-3) / 1e9 / peak, "n_cand_a": int(nc[0]), "n_cand_b": int(nc[1])}
        # distinct-PMT variant DN7: 16 B read + 1 B zeroed + 1 B written per hit
        d_dn = torch.empty(n, dtype=torch.uint8, device="cuda")
        d_dnn = torch.zeros(1, dtype=torch.int32, device="cuda")
        dn_ms = timed(lambda: B.tt_l0_dntw(l0_src, l0_seg, l0_n, l0_tw, d_dn, d_dnn), reps)
        l0["dn"] = {"kernel": "l0_dntw_kernel", "multiplicity": l0_n, "window_ps": l0_tw, "ms": dn_ms,
                    "alg_bytes_per_hit": 18, "achieved": 18.0 * n / (dn_ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                    "frac": 18.0 * n / (dn_ms * 1e-3) / 1e9 / peak,
                    "n_start": int(d_dnn.cpu().numpy().view(np.uint32)[0])}
        del d_l0, d_pb, d_cd, d_dn, l0_src

    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region ----
    e2e = None
    if not args.no_e2e:
        L = B.load()
        ctx = ctypes.c_void_p(0)
        rc = L.tt_host_ctx_create(ctypes.byref(ctx), ctypes.c_uint32(n), ctypes.c_uint32(seg.count),
                                  ctypes.c_uint32(runs.count), ctypes.c_uint32(seed_cap), ctypes.c_uint32(event_cap))
        if rc != 0:
            raise SystemExit(f"tt_host_ctx_create failed: {rc}")
        h_in = torch.from_numpy(w.hits.view(np.int64).reshape(-1, 2)).pin_memory()
        h_flags = torch.empty(n, dtype=torch.uint8).pin_memory()
        h_seeds = torch.empty(seed_cap, dtype=torch.int32).pin_memory()
        h_ev = torch.empty((event_cap, 4), dtype=torch.int64).pin_memory()
        h_cnt = np.zeros(4, dtype=np.uint32)
        vp = ctypes.c_void_p

        def host_args(cnt):
            return (ctx, vp(h_in.data_ptr()), vp(0), vp(h_flags.data_ptr()), ctypes.c_uint32(n),
                    seg.h.ctypes.data_as(vp), ctypes.c_uint32(seg.count), runs.h.ctypes.data_as(vp),
                    ctypes.c_uint32(runs.count), geo.handle, ctypes.byref(prm), vp(h_seeds.data_ptr()),
                    vp(h_ev.data_ptr()), cnt.ctypes.data_as(vp))

        def host_step():  # the synchronous call: upload, compute, read back, return
            rc = L.tt_process_host(*host_args(h_cnt))
            if rc != 0:
                raise SystemExit(f"tt_process_host failed: {rc}")

        host_step()
        barrier()
        k2 = max(2, min(args.steps, 6))
        t0 = time.perf_counter()
        for _ in range(k2):
            host_step()
        dt_sync = (time.perf_counter() - t0) / k2
        assert int(h_cnt[0]) == n_seeds and int(h_cnt[1]) == n_events, "host path disagrees with device path"
        # successive slices back to back: tt_host_submit / tt_host_wait, two slices in flight -- the upload
        # of slice k + 1 overlaps the compute of slice k and the read-back of slice k - 1.  Every slice is uploaded,
        # computed and read back inside the timed region; the time is per slice at steady state.
        cnts = [np.zeros(4, dtype=np.uint32) for _ in range(2)]
        barrier()
        t0 = time.perf_counter()
        for k in range(k2):
            rc = L.tt_host_submit(*host_args(cnts[k & 1]))
            if rc != 0:
                raise SystemExit(f"tt_host_submit failed: {rc}")
            if k >= 1 and L.tt_host_wait(ctx) != 0:
                raise SystemExit("tt_host_wait failed")
        if L.tt_host_wait(ctx) != 0:
            raise SystemExit("tt_host_wait failed")
        dt = (time.perf_counter() - t0) / k2
        for c2 in cnts:
            assert int(c2[0]) == n_seeds and int(c2[1]) == n_events, "pipelined host path disagrees with device path"
        dt, _ = sharding.reduce_timing(dt, n, "cuda")
        ns, ne = int(min(h_cnt[0], seed_cap)), int(min(h_cnt[1], event_cap))
        h2d = int(16 * n + 4 * (seg.count + 1) + 4 * (runs.count + 1))
        d2h = int(n + 4 * ns + 32 * ne + 12)
        # PCIe floor of one slice: its upload at the H2D rate measured right here on a plain pinned copy of the same size
        d_tmp = torch.empty_like(run.d_in)
        d_tmp.copy_(h_in, non_blocking=True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        d_tmp.copy_(h_in, non_blocking=True)
        torch.cuda.synchronize()
        floor_ms = 1e3 * (time.perf_counter() - t0)
        del d_tmp
        e2e = {"value": n_total / dt, "unit": "hits/s", "ms_per_step": 1e3 * dt,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "pcie_floor_ms": floor_ms, "vs_pcie_floor": 1e3 * dt / floor_ms,
               "ms_per_step_synchronous_call": 1e3 * dt_sync,
               "api": "tt_host_submit / tt_host_wait, two slices in flight (pinned host buffers; every slice uploaded, "
                      "computed, flags + seeds + events read back); ms_per_step_synchronous_call = tt_process_host"}
        L.tt_host_ctx_destroy(ctx)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        on, odt, sample, _ = time_oracle(args.config)
        cpu = {"value": on / odt, "unit": "hits/s", "cores": 1, "kind": "oracle", "sample": sample}
        try:
            cpu["all_cores"] = time_oracle_all_cores(args.config)
        except Exception as ex:  # the reported baseline must not take the bench line down
            cpu["all_cores"] = {"error": type(ex).__name__}

    # ---- the other configs (short runs; the driver's record then covers all five), the unsorted-input radix path and
    # the preparation step (tt_prepare_slice), each timed on its own, none part of the step above
    extra = None
    if rank == 0 and world == 1 and not args.no_extra:
        extra = {"configs": {}}
        if w.geometry.n_tower >= 8:
            n_seeds_step = n_seeds
            extra["tower_shard"] = time_tower_shard(B, w, geo, prm, 8)
            assert extra["tower_shard"]["global_seeds"] == n_seeds_step, "by-tower path disagrees with the single-GPU path"
        try:
            extra["library_sort"] = time_library_sort(B, run)
        except Exception as ex:  # context only: never takes the bench line down
            extra["library_sort"] = {"error": type(ex).__name__}
        torch.cuda.empty_cache()
        del run
        torch.cuda.empty_cache()
        for c2 in [c for c in (0, 1, 2, 3, 4) if c != args.config]:
            r2 = Run(B, c2, 0, 1.0, fused)
            m2 = timed_steps(B, r2, max(3, min(args.steps, 10)), 3, args.graph, barrier)
            extra["configs"][f"cfg{c2}"] = {
                "workload": r2.w.name, "hits": r2.n, "ms_per_step": m2["ms_step"],
                "ms_per_200ms_slice": m2["ms_step"] / r2.w.n_slices, "hits_per_s": r2.n / (m2["ms_step"] * 1e-3),
                "pipeline_frac": ALG_BYTES_PIPELINE * r2.n / (m2["ms_step"] * 1e-3) / 1e9 / peak,
                "stages": {k: v["frac"] for k, v in stage_fracs(m2["per_stage"], r2.n, peak).items()},
                "n_seeds": m2["n_seeds"], "n_events": m2["n_events"], "status": m2["status"]}
            if c2 == 3:
                extra["cfg3_streams_vs_segmented"] = time_streams(B, r2, args.steps)
                assert extra["cfg3_streams_vs_segmented"]["n_seeds_streams"] == m2["n_seeds"], "per-stream path disagrees"
            if c2 == 1:
                extra["radix_unsorted_input"] = time_radix(B, r2, peak)
            if c2 == 2:
                extra["prepare"] = time_prepare(B, peak)
            del r2
            torch.cuda.empty_cache()

    if rank == 0:
        slices = w.n_slices
        out = {
            "metric": METRIC, "value": value, "unit": "hits/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int64", "data": "synthetic",
            "config": {"workload": w.name, "hits_per_rank": n, "slices_per_step": slices,
                       "timed_step": ("tt_sort_trigger_slice (sort + L1 fused + L2 + seeds)" if fused else
                                      "tt_sort_slice + tt_trigger_slice") + " + tt_extract_events with INEVT tagging "
                                     "(SURVEY.md 8(d) times the events separately: they are INSIDE this step, "
                                     "ev.* in stages_ms_per_step)",
                       "ms_per_200ms_slice": ms_step / slices, "l2_flush": "inputs larger than L2 (16 B x n)"
                       if 16 * n > 130e6 else "inputs fit in L2: not flushed (launch-bound config)",
                       "n_seeds": n_seeds, "n_events": n_events, "status": status, "l1_fraction": l1_frac,
                       "inevt_fraction": inevt_frac, "parallelism": f"slice-per-gpu x{world}",
                       "cuda_graph": m["graph"], "cuda_graph_note": m["graph_note"]},
            "clocks": clocks, "gpu_launches": int(launches),
            "roofline": roof,
            "pipeline_roofline": {"alg_bytes_per_hit": ALG_BYTES_PIPELINE, "achieved": pipe_ach, "peak": peak,
                                  "unit": "GB/s", "frac": pipe_ach / peak},
            "stages_ms_per_step": {k: round(v, 5) for k, v in sorted(per_stage.items())},
            "counters": counters,
            "l0_ntw": l0,
            "e2e": e2e, "cpu_baseline": cpu, "extra": extra,
        }
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--scale", type=float, default=1.0, help="time_scale < 1 shrinks the workload (debugging only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--graph", default="auto", choices=["auto", "on", "off"],
                    help="replay the step as a CUDA graph in the timed region (auto: yes, direct launches if capture fails)")
    ap.add_argument("--fused", default="on", choices=["on", "off"],
                    help="on: tt_sort_trigger_slice (L1 fused into the last merge level); off: the three separate calls")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the short runs of the other configs / radix / prepare")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
