"""Energy sharding over ranks: the host logic, exercised on CPU with the
gloo backend and world_size 2/3.  Each "rank" computes its slice with the oracle (this is a
test; the product path uses the CUDA library) and the gathered stack must equal the
single-process result energy by energy."""
import os
import socket

import numpy as np
import pytest

from paper_2209_13121_b200 import sharding, workloads as W


def test_energy_slices_cover_and_balance():
    for n in (0, 1, 2, 7, 10, 50, 100):
        for world in (1, 2, 3, 8, 16):
            sl = sharding.energy_slices(n, world)
            assert len(sl) == world and sl[0][0] == 0 and sl[-1][1] == n
            assert all(sl[i][1] == sl[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in sl]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        sharding.energy_slices(4, 0)


def test_shard_workload_tables_follow_the_slice():
    w = W.tiny(seed=5, nx=8, ny=8, nz=4, n_mat=3, n_energy=5)
    seen = []
    for r in range(3):
        part, (a, b) = sharding.shard_workload(w, r, 3)
        assert part.n_energy == b - a
        assert np.array_equal(part.energies, w.energies[a:b])
        for name in ("delta_par", "beta_par", "delta_perp", "beta_perp"):
            assert np.array_equal(getattr(part, name), getattr(w, name)[a:b])
        assert part.materials is w.materials and part.angles == w.angles
        seen += list(range(a, b))
    assert seen == list(range(5))
    assert sharding.shard_workload(w, 7, 8)[0] is None          # more ranks than energies


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_energy, q):
    import torch
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = W.tiny(seed=21, nx=16, ny=16, nz=4, n_mat=2, n_energy=n_energy, voxel_nm=2.0)
        part, (a, b) = sharding.shard_workload(w, rank, world)
        if part is None:
            local = torch.zeros((0, w.Ny, w.Nx), dtype=torch.float64)
        else:
            out, _ = oracle.run(part.materials, part.voxel_nm, part.energies, part.delta_par, part.beta_par,
                                part.delta_perp, part.beta_perp, part.angles, part.ewald)
            local = torch.from_numpy(out)
        full = sharding.gather_images(local, w.n_energy, dst=0)
        if rank == 0:
            q.put(full.numpy())
        else:
            assert full is None
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,n_energy", [(2, 5), (3, 2)])
def test_gloo_sharded_run_matches_single_process(world, n_energy):
    import torch.multiprocessing as mp
    import oracle
    oracle.build()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_energy, q)) for r in range(world)]
    for p in procs:
        p.start()
    full = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    w = W.tiny(seed=21, nx=16, ny=16, nz=4, n_mat=2, n_energy=n_energy, voxel_nm=2.0)
    ref, _ = oracle.run(w.materials, w.voxel_nm, w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp,
                        w.angles, w.ewald)
    assert full.shape == ref.shape
    assert np.array_equal(full, ref)


# ----------------------------------------------------------------------------- spectra shards (strong scaling)

def test_material_parts_cover_balance_and_pack_layout():
    cases = [([True, True], 2), ([True, True, False], 2), ([True, True, False, False], 3), ([False] * 5, 5),
             ([True, False, False, False, True], 2), ([False] * 5, 2), ([True] * 4 + [False] * 3, 3), ([True, True, False], 1)]
    for aligned, n_parts in cases:
        parts = sharding.material_parts(aligned, n_parts)
        assert len(parts) == n_parts and parts[0][0] == 0 and parts[-1][1] == len(aligned)
        assert all(parts[i][1] == parts[i + 1][0] for i in range(n_parts - 1)) and all(b > a for a, b in parts)
        fields = [sum(7 if x else 1 for x in aligned[a:b]) for a, b in parts]
        assert max(fields) - min(fields) <= 7, (aligned, parts)           # no part is off by more than one material's worth
        ranges = sharding.pack_ranges(aligned, n_parts)
        assert ranges[0][0] == 0 and all(ranges[i][0] + ranges[i][1] == ranges[i + 1][0] for i in range(n_parts - 1))
        assert [n for _, n in ranges] == [(f + 1) // 2 for f in fields]
    assert sharding.material_parts([True, True, False], 2) == [(0, 1), (1, 3)]   # 7 | 8 fields, not 14 | 1
    with pytest.raises(ValueError):
        sharding.material_parts([True], 2)


def _spectra_worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        aligned = [True, False, True, False, False]
        n_parts = min(world, len(aligned))
        ranges = sharding.pack_ranges(aligned, n_parts)
        n_pack = ranges[-1][0] + ranges[-1][1]
        spec = torch.full((n_pack, 6), -1.0)
        for part, (first, n) in enumerate(ranges):                   # what this rank "transformed": its own part(s)
            if part % world == rank:
                spec[first:first + n] = torch.arange(first, first + n, dtype=torch.float32)[:, None] * 10 + torch.arange(6.0)
        got = sharding.exchange_spectra(spec, ranges)
        q.put((rank, spec.numpy(), got))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_gloo_exchange_of_spectra_parts(world):
    """Every rank ends with every part's block (one broadcast per part from its owner) and counts its received bytes."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_spectra_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    aligned = [True, False, True, False, False]
    ranges = sharding.pack_ranges(aligned, min(world, len(aligned)))
    n_pack = ranges[-1][0] + ranges[-1][1]
    expect = np.arange(n_pack, dtype=np.float32)[:, None] * 10 + np.arange(6, dtype=np.float32)
    for rank, spec, got in res:
        assert np.array_equal(spec, expect), rank
        own = sum(n for part, (_, n) in enumerate(ranges) if part % world == rank)
        assert got == (n_pack - own) * 6 * 4
