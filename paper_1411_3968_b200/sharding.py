"""Host-side logic of the N > 1 path (one process per GPU, multi-GPU).

Two ways to shard.  (i) By time slice -- the default of bench.py: "successive time slices are sent to different" trigger nodes, every
rank sorts and triggers whole slices of its own, and no step of the data path exchanges anything -- so there is no
collective here beyond the two scalars of the timing protocol (max of the step time, sum of the hits).  Works on any
torch.distributed backend (nccl on the GPUs, gloo in the CPU tests).  (ii) By tower (NEXT-4): every rank
owns a contiguous range of towers of ONE slice, sorts and L1-tags its hits, and the ranks all-gather their L1 hits
(~2 % of the hits) once before the inter-tower L2: `tower_local` -> `all_gather_records` -> `tower_global` below; the
arithmetic of every step runs in the CUDA kernels behind the C ABI (include/tt.h), this module only moves buffers."""
from __future__ import annotations

import torch


def slice_owner(slice_index: int, world: int) -> int:
    """Round-robin: consecutive 200 ms slices go to consecutive ranks."""
    return slice_index % world


def my_slices(n_slices: int, rank: int, world: int) -> list[int]:
    return [s for s in range(n_slices) if slice_owner(s, world) == rank]


def workload_seed_offset(rank: int, round_index: int, world: int) -> int:
    """Seed offset of the slice rank `rank` processes in round `round_index` (= its global slice index)."""
    return round_index * world + rank


def reduce_timing(ms_local: float, units_local: int, device: torch.device | str = "cpu") -> tuple[float, int]:
    """(max over ranks of the step time, sum over ranks of the units processed).  No-op without a process group."""
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), int(units_local)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([int(units_local)], dtype=torch.int64, device=device)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


# ---- (ii) by tower -----------------------------------------------------------------------------------------------
def tower_ranges(n_tower: int, world: int) -> list[tuple[int, int]]:
    """Contiguous tower ranges, as even as possible: rank r owns towers [lo, hi)."""
    base, rem = divmod(n_tower, world)
    out, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < rem else 0)
        out.append((lo, hi))
        lo = hi
    return out


def split_runs_by_tower(run_offsets, pmts_per_tower: int, n_tower: int, world: int):
    """For a single-slice, tower-major / PMT-major input (run p = PMT p): per rank (first hit, end hit, its run offsets
    rebased to 0).  The rank's input is a contiguous range of the global input, in the global order."""
    import numpy as np

    ro = np.asarray(run_offsets, dtype=np.int64)
    assert len(ro) - 1 == pmts_per_tower * n_tower, "one run per PMT, one slice"
    out = []
    for lo, hi in tower_ranges(n_tower, world):
        a, b = lo * pmts_per_tower, hi * pmts_per_tower
        out.append((int(ro[a]), int(ro[b]), (ro[a:b + 1] - ro[a]).astype(np.uint32)))
    return out


def all_gather_records(rec: torch.Tensor) -> tuple[torch.Tensor, list[int]]:
    """All-gather variable-length (m_r, 2) int64 record lists: returns their concatenation in rank order and the
    offsets [0, m_0, m_0 + m_1, ...].  Without a process group: the list itself."""
    import torch.distributed as dist

    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return rec, [0, int(rec.shape[0])]
    world = dist.get_world_size()
    dev = rec.device
    if rec.is_cuda and dist.get_backend() == "gloo":  # gloo moves host memory: stage through the host and come back
        cat, offs = all_gather_records(rec.cpu())
        return cat.to(dev), offs
    cnt = torch.tensor([rec.shape[0]], dtype=torch.int64, device=rec.device)
    cnts = [torch.zeros_like(cnt) for _ in range(world)]
    dist.all_gather(cnts, cnt)
    ms = [int(c.item()) for c in cnts]
    mmax = max(max(ms), 1)
    pad = torch.zeros((mmax, 2), dtype=torch.int64, device=rec.device)
    pad[: rec.shape[0]] = rec
    bufs = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(bufs, pad)
    offs = [0]
    for m in ms:
        offs.append(offs[-1] + m)
    return torch.cat([b[:m] for b, m in zip(bufs, ms)], dim=0), offs


def tower_local(B, rank: int, hits, run_offsets, params):
    """Phase 1 on rank `rank`: its towers' hits (numpy, PMT-major runs) -> sorted + L1 flags on the device, and its L1
    records.  Returns the state `tower_global` continues from."""
    import numpy as np

    d_in = hits if isinstance(hits, torch.Tensor) else B.hits_to_device(hits)  # (n, 2) int64 on the device, or numpy hits
    n = int(d_in.shape[0])
    seg = B.Offsets(np.array([0, n], dtype=np.uint32))
    runs = run_offsets if isinstance(run_offsets, B.Offsets) else B.Offsets(run_offsets)
    d_out = torch.empty_like(d_in)
    d_flags = torch.full((max(n, 1),), 0xEE, dtype=torch.uint8, device="cuda")
    d_st = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.tt_sort_l1_slice(d_in, d_out, None, seg, runs, params, d_flags, d_st)
    d_l1 = torch.empty((max(n, 1), 2), dtype=torch.int64, device="cuda")
    d_m = torch.zeros(1, dtype=torch.int32, device="cuda")
    B.tt_l1_export(d_out, d_flags, rank, d_l1, d_m, d_st)
    m = int(d_m.item())
    return dict(rank=rank, n=n, d_sorted=d_out, d_flags=d_flags, d_status=d_st, l1=d_l1[:m].contiguous())


def tower_global(B, state, gathered: torch.Tensor, offsets: list[int], geo, params, download: bool = True):
    """Phase 2: merge the gathered L1 records in time, inter-tower L2 on the merged list, global event windows, then
    this rank's flag bits, seeds and INEVT tags.  Returns numpy arrays: flags, seeds (local indices), events
    (download=False: leaves everything on the device and returns the device tensors)."""
    import numpy as np

    m = int(gathered.shape[0])
    seg = B.Offsets(np.array([0, m], dtype=np.uint32))
    runs = B.Offsets(np.asarray(offsets, dtype=np.uint32))
    d_st = state["d_status"]
    d_l1m = torch.empty_like(gathered)
    if m:
        B.tt_sort_slice(gathered.contiguous(), d_l1m, None, seg, runs, d_st)  # a record starts with its time, like a hit
    d_bits = torch.zeros(max(m, 1), dtype=torch.uint8, device="cuda")
    d_gseeds = torch.zeros(max(m, 1), dtype=torch.int32, device="cuda")
    d_cnt = torch.zeros(4, dtype=torch.int32, device="cuda")  # global seeds, events, local seeds
    B.tt_l2_merged(d_l1m, geo, params, d_bits, d_gseeds, d_cnt[0:1], d_st)
    d_ev = torch.zeros((max(m, 1), 4), dtype=torch.int64, device="cuda")
    B.tt_extract_events(d_l1m, seg, d_gseeds, d_cnt[0:1], params, d_ev, d_cnt[1:2], None, None, None, d_st)
    n = state["n"]
    d_seeds = torch.zeros(max(n, 1), dtype=torch.int32, device="cuda")
    B.tt_l2_apply(d_l1m, d_bits, state["rank"], state["d_flags"], n, d_seeds, d_cnt[2:3], d_st)
    B.tt_tag_windows(state["d_sorted"], d_ev, d_cnt[1:2], params, state["d_flags"])
    if not download:
        return dict(d_flags=state["d_flags"], d_seeds=d_seeds, d_events=d_ev, d_counts=d_cnt)
    torch.cuda.synchronize()
    cnt = d_cnt.cpu().numpy().view(np.uint32)
    return dict(sorted=B.hits_to_host(state["d_sorted"]), flags=state["d_flags"].cpu().numpy()[:n].copy(),
                seeds=d_seeds[: int(cnt[2])].cpu().numpy().view(np.uint32).copy(), n_global_seeds=int(cnt[0]),
                events=d_ev[: int(cnt[1])].cpu().numpy().reshape(-1).view(B.EVENT_DTYPE).copy(), status=int(d_st.item()))
