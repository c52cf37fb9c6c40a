"""Energy sharding over ranks (energies are independent,
"embarrassingly parallel", one GPU per energy chunk, morphology replicated).

Host-side logic only -- which energies a rank owns and how the per-rank image stacks are
put back in energy order on one rank.  There is no data-path collective: every rank runs
`cyrsoxs_run` on its own slice of the energy list with the full morphology; the only
communication is the optional gather of the finished images (Ny*Nx floats per energy).
`torch.distributed` is the plumbing (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import List, Optional, Tuple


def energy_slices(n_energy: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous, balanced [start, stop) energy ranges, one per rank; the first
    n_energy % world ranks own one energy more.  Ranks beyond n_energy own an empty range."""
    if n_energy < 0 or world < 1:
        raise ValueError("n_energy must be >= 0 and world >= 1")
    base, extra = divmod(n_energy, world)
    out, start = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((start, start + n))
        start += n
    return out


def shard_workload(workload, rank: int, world: int):
    """The rank's share of a `workloads.Workload`: same morphology and angles, its slice of
    the energies and of the optical-constant tables.  Returns (workload_or_None, (start, stop))."""
    start, stop = energy_slices(workload.n_energy, world)[rank]
    if stop == start:
        return None, (start, stop)
    return workload.restrict_energies(range(start, stop)), (start, stop)


def gather_images(local, n_energy: int, dst: int = 0, group=None):
    """Collects the per-rank image stacks [n_local][Ny][Nx] (torch tensors, same device and
    dtype on every rank) into one [n_energy][Ny][Nx] tensor on rank `dst`, in energy order.
    Returns the full stack on `dst`, None elsewhere.  Uses all_gather on a stack padded to the
    largest slice (works on both nccl and gloo)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    slices = energy_slices(n_energy, world)
    n_max = max(b - a for a, b in slices)
    a, b = slices[rank]
    if local.shape[0] != b - a:
        raise ValueError(f"rank {rank} holds {local.shape[0]} energies, its slice is [{a}, {b})")
    padded = torch.zeros((n_max,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    padded[: b - a] = local
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded, group=group)
    if rank != dst:
        return None
    return torch.cat([parts[r][: slices[r][1] - slices[r][0]] for r in range(world)], 0)


def simulate_sharded(workload, algorithm: int = 0, device: Optional[str] = None, gather: bool = True, group=None):
    """Runs the rank's slice of `workload` through the C-ABI library on this rank's GPU and
    (optionally) gathers the images on rank 0.  Requires an initialised process group."""
    import torch
    import torch.distributed as dist
    from . import binding
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    dev = device or f"cuda:{torch.cuda.current_device()}"
    mine, (a, b) = shard_workload(workload, rank, world)
    if mine is None:
        local = torch.zeros((0, workload.Ny, workload.Nx), dtype=torch.float32, device=dev)
    else:
        local = binding.simulate(mine, algorithm=algorithm, device=dev)[0]
    if not gather:
        return local
    return gather_images(local, workload.n_energy, 0, group)
