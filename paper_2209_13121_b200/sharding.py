"""Sharding over ranks.  Two partitions:

* energies -- no data-path collective, every rank holds the full morphology;
* the energy-independent spectra of SPECTRAL_BASIS over MATERIALS (`material_parts`, `exchange_spectra`,
  `simulate_strong`): after reduction R4 almost all device time of a large run is the transform of the basis fields,
  which energy sharding would repeat on every rank.  Rank r transforms the fields of material group r, the pruned
  spectra (the Ewald windows: 0.77 GB at CFG3, 3.6 GB at CFG5) are exchanged once per run over NVLink (one broadcast per
  group), then every rank does its slice of the energies.

Energy sharding over ranks (energies are independent,
"embarrassingly parallel", one GPU per energy chunk, morphology replicated).

Host-side logic only -- which energies a rank owns and how the per-rank image stacks are
put back in energy order on one rank.  There is no data-path collective: every rank runs
`cyrsoxs_run` on its own slice of the energy list with the full morphology; the only
communication is the optional gather of the finished images (Ny*Nx floats per energy).
`torch.distributed` is the plumbing (nccl on GPUs, gloo in the CPU tests).
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple


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


# ----------------------------------------------------------------------------- spectra shards (strong scaling)

def material_parts(aligned: Sequence[bool], n_parts: int) -> List[Tuple[int, int]]:
    """Contiguous material ranges [m0, m1), one per part, of about equal basis-field count (7 fields per aligned
    material, 1 per isotropic one), every part at least one material.  The same rule as the library's
    (cyrsoxs_set_spectra_shard; `Context.spectra_part` reports the library's pack ranges)."""
    n_mat = len(aligned)
    if not 1 <= n_parts <= n_mat:
        raise ValueError("1 <= n_parts <= number of materials")
    w = [7 if a else 1 for a in aligned]
    total = sum(w)
    out, m, cum = [], 0, 0
    for q in range(n_parts):
        m0 = m
        must_leave = n_parts - 1 - q
        target = total * (q + 1)                                   # cumulative field count this part should end at, times n_parts
        while True:
            cum += w[m]
            m += 1
            if m >= n_mat - must_leave:
                break
            # take the next material too if that ends closer to the target (the last part takes everything left)
            if q < n_parts - 1 and abs((cum + w[m]) * n_parts - target) >= abs(cum * n_parts - target):
                break
        out.append((m0, m))
    return out


def pack_ranges(aligned: Sequence[bool], n_parts: int) -> List[Tuple[int, int]]:
    """(first pack, number of packs) of every part: the fields of a part are paired among themselves, an odd count
    is padded (n_parts = 1: all fields in one sequence)."""
    out, first = [], 0
    for m0, m1 in material_parts(aligned, n_parts):
        fields = sum(7 if a else 1 for a in aligned[m0:m1])
        n = (fields + 1) // 2
        out.append((first, n))
        first += n
    return out


def owner_of_part(part: int, world: int) -> int:
    """The rank whose transform of `part` is the one that is broadcast (ranks beyond the number of parts repeat a
    part concurrently and only receive)."""
    return part % world


def exchange_spectra(spectra, ranges: Sequence[Tuple[int, int]], group=None):
    """spectra: [n_pack, ...] tensor, on every rank the block of its own part filled in.  One broadcast per part
    from its owner; afterwards every rank holds all blocks.  Returns the bytes this rank received."""
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    received = 0
    for part, (first, n) in enumerate(ranges):
        if n == 0:
            continue
        block = spectra[first:first + n]
        src = owner_of_part(part, world)
        dist.broadcast(block, src=src if group is None else dist.get_global_rank(group, src), group=group)
        if rank != src:
            received += block.numel() * block.element_size()
    return received


class _DevicePtr:
    """CUDA array interface over a raw device pointer (the library owns the memory)."""
    def __init__(self, ptr: int, nbytes: int):
        self.__cuda_array_interface__ = {"shape": (nbytes,), "typestr": "|u1", "data": (ptr, False), "version": 2}


def spectra_tensor(ctx, device=None):
    """The context-owned spectra buffer as a [n_pack, pack_bytes] uint8 CUDA tensor (no copy).  `device`: index of the
    GPU the context was created on (default: torch's current device -- pass it when that may differ)."""
    import torch
    ptr, pack_bytes, n_pack = ctx.spectra()
    dev = torch.device("cuda", torch.cuda.current_device() if device is None else int(device))
    return torch.as_tensor(_DevicePtr(ptr, pack_bytes * n_pack), device=dev).view(n_pack, pack_bytes)


def run_strong(ctx, workload, out, stream_ptr: int, group=None, device=None):
    """One strong-scaling run on this rank: its part of the spectra, the exchange, its slice of the energies into
    `out` [n_local][Ny][Nx].  `ctx` has the full morphology, ALL energies of the workload, angles and Ewald mode set,
    its shard set to (rank % n_parts, n_parts) and, unless the rank's slice is empty, its energy range set to that slice.
    A rank with an empty slice (more ranks than energies) passes `out` with zero rows (or None): it still transforms and
    exchanges, and skips the energy phase.  `stream_ptr` is the cudaStream_t everything is ordered on: the broadcasts
    of the exchange are issued with that stream current (NCCL orders a collective after the current stream's work), so
    they sit between cyrsoxs_run_spectra and cyrsoxs_run_energies whatever stream the caller has current.  `device`:
    index of the context's GPU (default: torch's current device).  Returns bytes received.  Not yet run on more than one
    physical GPU."""
    import contextlib

    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    ctx.run_spectra(stream_ptr)
    received = 0
    if world > 1:
        aligned = [m[1] is not None for m in workload.materials]
        n_parts = min(world, len(aligned))
        dev = torch.cuda.current_device() if device is None else int(device)
        spec = spectra_tensor(ctx, dev)
        ranges = [ctx.spectra_part(q) for q in range(n_parts)]
        assert ranges == pack_ranges(aligned, n_parts), "library and host disagree on the pack layout"
        on_run_stream = contextlib.nullcontext()
        if torch.cuda.current_stream(dev).cuda_stream != int(stream_ptr or 0):
            on_run_stream = torch.cuda.stream(torch.cuda.ExternalStream(int(stream_ptr), device=dev))
        with on_run_stream:
            received = exchange_spectra(spec, ranges, group)
    if out is not None and out.shape[0] > 0:
        ctx.run_energies(out.data_ptr(), stream_ptr)
    return received
