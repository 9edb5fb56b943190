"""Host-side logic of the N > 1 path (one process per GPU, multi-GPU).

The path shards by time slice: "successive time slices are sent to different" trigger nodes, every
rank sorts and triggers whole slices of its own, and no step of the data path exchanges anything -- so there is no
collective here beyond the two scalars of the timing protocol (max of the step time, sum of the hits).  Works on any
torch.distributed backend (nccl on the GPUs, gloo in the CPU tests)."""
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
