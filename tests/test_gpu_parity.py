"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded
inputs, element by element, with the north_star gates (tests/parity.py)."""
import os

import numpy as np
import pytest

from paper_2209_13121_b200 import workloads as W
from tests.parity import compare, oracle_run

pytestmark = pytest.mark.gpu

ALGS = [1, 2]      # binding.ALG_PER_ENERGY, binding.ALG_SPECTRAL_BASIS


def _gpu(w, alg, images=False):
    from paper_2209_13121_b200 import binding
    res = binding.simulate(w, algorithm=alg, want_counts=True, want_images=images)
    out, cnt = res[0].cpu().numpy(), res[1].cpu().numpy()
    if images:
        return out, cnt, res[2].cpu().numpy(), res[-1]
    return out, cnt, res[-1]


@pytest.mark.parametrize("alg", ALGS)
@pytest.mark.parametrize("mode", [W.EWALD_NEAREST, W.EWALD_TRILINEAR])
@pytest.mark.parametrize("shape", [(8, 8, 4), (32, 16, 8), (16, 64, 2), (64, 32, 1), (4, 4, 16), (16, 512, 2), (8, 4, 512), (1024, 4, 1), (8, 128, 256), (4, 1024, 2), (16, 16, 7), (32, 16, 63), (8, 8, 12), (8, 4, 3), (8, 4, 500),
                                   (16, 2, 4), (2048, 4, 2), (4, 2048, 2), (8, 4, 2048), (2048, 2, 8)])
def test_tiny_random(shape, mode, alg):
    """Ragged and extreme shapes: Ny = 2, every axis at its maximum of 2048 inside a 3-D model, z axes that are not
    powers of two; a voxel size that is not representable in float32 (1.3 nm: the ABI takes a double, so the detector
    grid dq is the oracle's bit for bit)."""
    nx, ny, nz = shape
    w = W.tiny(seed=100 + nx + nz, nx=nx, ny=ny, nz=nz, n_mat=3, n_energy=3, voxel_nm=1.3 if nx in (16, 2048) else 2.0, ewald=mode)
    ref, rcnt = oracle_run(w)
    out, cnt, _ = _gpu(w, alg)
    compare(out, cnt, ref, rcnt, f"tiny{shape}")


@pytest.mark.parametrize("mode", [W.EWALD_NEAREST, W.EWALD_TRILINEAR])
@pytest.mark.parametrize("shape", [(96, 80, 12), (45, 27, 5), (12, 10, 3), (100, 64, 8), (64, 100, 1), (33, 2, 2), (640, 24, 3), (24, 600, 2)])
def test_lateral_sizes_that_are_not_powers_of_two(shape, mode):
    """SURVEY 8(f) NEXT-4 / DESIGN 3-A14: Nx, Ny of any length (pruned direct DFT along such an axis), AUTO algorithm
    (SPECTRAL_BASIS), both Ewald modes, odd and even sizes, one axis or both, rho = Nx / Ny not a power of two."""
    nx, ny, nz = shape
    w = W.tiny(seed=300 + nx + nz, nx=nx, ny=ny, nz=nz, n_mat=3, n_energy=2, voxel_nm=2.0, ewald=mode)
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, ctx = _gpu(w, 0)
    assert ctx.stats()["algorithm"] == 2
    compare(out, cnt, ref, rcnt, f"nonpow2{shape}")


def test_film_1000x600_not_a_power_of_two():
    """A 1000 x 600 x 1 film (the reduced cfg4 recipe cannot be cropped, so the random-everything generator): every
    row and column goes through the direct-DFT passes at a size where their summation order matters."""
    w = W.tiny(seed=41, nx=1000, ny=600, nz=1, n_mat=3, n_energy=2, voxel_nm=2.0, ewald=W.EWALD_NEAREST, angles=(0.0, 45.0, 135.0))
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, _ = _gpu(w, 0)
    print("film 1000x600", compare(out, cnt, ref, rcnt, "film1000x600"))


def test_per_energy_refuses_nx_that_is_not_a_power_of_two():
    from paper_2209_13121_b200 import binding
    w = W.tiny(seed=5, nx=12, ny=8, nz=2, n_mat=2, n_energy=1)
    with pytest.raises(binding.CyrsoxsError) as ei:
        binding.simulate(w, algorithm=binding.ALG_PER_ENERGY)
    assert ei.value.status == binding.ERR_NOT_IMPLEMENTED
    w2 = W.tiny(seed=5, nx=16, ny=12, nz=6, n_mat=2, n_energy=1)           # Ny, Nz of any length are fine for PER_ENERGY
    ref, rcnt = oracle_run(w2, linear=True)
    out, cnt, _ = _gpu(w2, binding.ALG_PER_ENERGY)
    compare(out, cnt, ref, rcnt, "per-energy 16x12x6")


@pytest.mark.parametrize("alg", ALGS)
def test_stage_images_match_oracle_linear_images(alg):
    w = W.tiny(seed=3, nx=32, ny=32, nz=16, n_mat=3, n_energy=2, voxel_nm=1.0, ewald=W.EWALD_TRILINEAR)
    ref, rcnt, (Ixx, Iyy, Ixy, valid) = oracle_run(w, linear=True, return_images=True)
    out, cnt, imgs, ctx = _gpu(w, alg, images=True)
    assert imgs.shape[0] == 2
    for e in range(2):
        assert (imgs[e, :, :, 3].astype(bool) == valid[e].astype(bool)).all()
        for j, r in enumerate((Ixx[e], Iyy[e], Ixy[e])):
            err = np.abs(imgs[e, :, :, j] - r).max() / np.abs(Ixx[e]).max()
            assert err < 5e-6, (e, j, err)


@pytest.mark.parametrize("alg", ALGS)
def test_cfg1_full(alg):
    w = W.cfg1()
    ref, rcnt = oracle_run(w)
    out, cnt, _ = _gpu(w, alg)
    r = compare(out, cnt, ref, rcnt, "cfg1")
    print("cfg1", r)


@pytest.mark.parametrize("alg", ALGS)
def test_cfg2_reduced_definition_mode(alg):
    w = W.cfg2(n=64, n_energy=3)
    ref, rcnt = oracle_run(w)
    out, cnt, _ = _gpu(w, alg)
    print("cfg2/64", compare(out, cnt, ref, rcnt, "cfg2/64"))


@pytest.mark.parametrize("alg", ALGS)
def test_cfg2_full_size(alg):
    """BASELINE configs[1] at full size (the bench workload), oracle in linear mode."""
    w = W.cfg2()
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, ctx = _gpu(w, alg)
    print("cfg2", compare(out, cnt, ref, rcnt, "cfg2"), ctx.stats())


@pytest.mark.parametrize("alg", ALGS)
def test_cfg3_reduced(alg):
    w = W.cfg3(nx=64, ny=64, nz=32, n_energy=4, grain=8.0)
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, _ = _gpu(w, alg)
    print("cfg3/64", compare(out, cnt, ref, rcnt, "cfg3/64"))


@pytest.mark.parametrize("alg", ALGS)
def test_cfg4_reduced(alg):
    w = W.cfg4(n=256, n_energy=3)
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, _ = _gpu(w, alg)
    print("cfg4/256", compare(out, cnt, ref, rcnt, "cfg4/256"))


def _full_size_sampled(w, energy_idx, label, chunk=1):
    """Full-size config through the launch configuration bench.py uses (AUTO algorithm, all
    energies in one run); the oracle (linear mode) recomputes the sampled energies one by one."""
    out, cnt, ctx = _gpu(w, 0)
    assert np.isfinite(out).all()
    st = ctx.stats()
    energy_idx = list(energy_idx)
    for i in range(0, len(energy_idx), chunk):
        idx = energy_idx[i:i + chunk]
        ref, rcnt = oracle_run(w.restrict_energies(idx), linear=True)
        r = compare(out[idx], cnt[idx], ref, rcnt, f"{label} e={idx}")
        print(label, "energies", idx, {k: float(np.max(v)) for k, v in r.items()}, "algorithm", st["algorithm"], "batch", st["energy_batch"])


def test_cfg3_full_size_11_of_50_energies():
    """BASELINE configs[2] at full size (512x512x256, 50 energies, trilinear): 11 energies spread over the grid,
    both ends included (the last has the largest k: the one that sizes the spectral windows), against the oracle --
    11 different Ewald geometries (node and validity decisions depend on k)."""
    w = W.cfg3()
    _full_size_sampled(w, [0, 5, 10, 15, 20, 24, 30, 35, 40, 45, 49], "cfg3")


def test_cfg4_full_size_all_100_energies():
    """BASELINE configs[3] at full size (2048x2048x1, 4 materials, 100 energies x 36 angles): every energy against
    the linear-mode oracle (2-D: cheap), i.e. 100 different Ewald disks cutting the detector."""
    w = W.cfg4()
    _full_size_sampled(w, range(w.n_energy), "cfg4", chunk=10)


def _host_ram_gb():
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable"):
                return int(line.split()[1]) / 1e6
    except OSError:
        pass
    return 0.0


def test_cfg5_quarter_depth_sampled_energies():
    """BASELINE configs[4] at full lateral size and a quarter of the depth (1024x1024x128, 1.3e8
    voxels; same generator, same energies, trilinear).  The full-depth run is the next test."""
    w = W.cfg5(nz=128)
    _full_size_sampled(w, [0, 10, 19], "cfg5/nz128")


@pytest.mark.skipif(_host_ram_gb() < 100.0 or os.environ.get("CYRSOXS_SKIP_FULL_CFG5") == "1",
                    reason="full CFG5 needs ~90 GB of host RAM for the generator and the oracle (about 80 s on the B200 box)")
def test_cfg5_full_size_five_energies():
    """BASELINE configs[4] at full size (1024x1024x512 = 5.4e8 voxels, 17 GB of morphology): 64-bit indexing, memory
    footprint, the largest windows (last energy), the low-k end (first energy) and three energies in between -- five
    Ewald geometries of the 20 on the configuration the bench line is quoted on (about 40 s of oracle time each)."""
    w = W.cfg5()
    _full_size_sampled(w, [0, 5, 10, 15, 19], "cfg5")


@pytest.mark.parametrize("alg", ALGS)
def test_edge_cases(alg):
    # single angle, 90 degrees (pixel permutation), all-isotropic materials, Nz = 2
    w = W.tiny(seed=9, nx=16, ny=16, nz=2, n_mat=2, n_energy=1, voxel_nm=3.0, ewald=W.EWALD_TRILINEAR,
               angles=(90.0, 0.0, 90.0))
    ref, rcnt = oracle_run(w)
    out, cnt, _ = _gpu(w, alg)
    compare(out, cnt, ref, rcnt, "single-angle-90")
    iso = [(m[0], None, None, None) for m in w.materials]
    w2 = W.Workload("iso", w.Nx, w.Ny, w.Nz, w.voxel_nm, iso, w.energies, w.delta_par, w.beta_par, w.delta_par,
                    w.beta_par, (0.0, 45.0, 315.0), W.EWALD_NEAREST)
    ref, rcnt = oracle_run(w2)
    out, cnt, _ = _gpu(w2, alg)
    compare(out, cnt, ref, rcnt, "all-isotropic")
    # a detector mostly off the Ewald sphere: tiny voxels -> large dq, few valid pixels
    w3 = W.tiny(seed=10, nx=32, ny=32, nz=8, n_mat=2, n_energy=2, voxel_nm=0.4, ewald=W.EWALD_NEAREST)
    ref, rcnt = oracle_run(w3)
    assert (rcnt == 0).mean() > 0.5
    out, cnt, _ = _gpu(w3, alg)
    compare(out, cnt, ref, rcnt, "mostly-invalid")


def test_errors_and_not_ready():
    import torch
    from paper_2209_13121_b200 import binding
    ctx = binding.Context(16, 16, 4, 1, 2.0)
    out = torch.empty((1, 16, 16), device="cuda")
    with pytest.raises(binding.CyrsoxsError) as ei:
        ctx.run(out.data_ptr())
    assert ei.value.status == binding.ERR_NOT_READY
    for bad in [(0.0, 0.0, 10.0), (10.0, 5.0, 0.0)]:
        with pytest.raises(binding.CyrsoxsError) as ei:
            ctx.set_angles(*bad)
        assert ei.value.status == binding.ERR_INVALID_ARG
    with pytest.raises(binding.CyrsoxsError):
        ctx.set_ewald(7)
    with pytest.raises(binding.CyrsoxsError):
        ctx.set_optical_constants([-1.0], [[0]], [[0]], [[0]], [[0]])
    phi = torch.ones((4, 16, 16), device="cuda")
    with pytest.raises(binding.CyrsoxsError):
        ctx.set_morphology([(phi, phi, None, None)])      # S without theta/psi
    ctx.close()


def test_host_output_and_host_morphology():
    """End-to-end entry: morphology from host arrays, images written to pinned host memory."""
    import torch
    from paper_2209_13121_b200 import binding
    w = W.tiny(seed=12, nx=32, ny=32, nz=8, n_mat=2, n_energy=5, voxel_nm=2.0)
    ref, rcnt = oracle_run(w)
    ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    s = torch.cuda.current_stream().cuda_stream
    ctx.set_morphology_host(w.materials, s)
    ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald); ctx.set_algorithm(ALGS[0])
    out = torch.empty((w.n_energy, w.Ny, w.Nx), dtype=torch.float32).pin_memory()
    ctx.run(out.data_ptr(), s)
    torch.cuda.synchronize()
    compare(out.numpy(), None, ref, rcnt, "host-io")


@pytest.mark.parametrize("shape,n_bins,width", [((64, 64, 1), 32, 20.0), ((128, 32, 4), 70, 10.0), ((32, 64, 2), 16, 45.0)])
def test_reductions_match_oracle(shape, n_bins, width):
    """cyrsoxs_reduce (NEXT-1: I(|q|), anisotropy, ISI) on the GPU path's own images against the
    oracle's reductions of the oracle's images: bins are integer decisions (compared through the
    means of a coordinate image, exactly), values within the image tolerance."""
    import torch
    import oracle
    from paper_2209_13121_b200 import binding
    nx, ny, nz = shape
    w = W.tiny(seed=31 + nx, nx=nx, ny=ny, nz=nz, n_mat=3, n_energy=3, voxel_nm=2.5, ewald=W.EWALD_NEAREST)
    ref, rcnt = oracle_run(w)
    out, cnt, ctx = binding.simulate(w, want_counts=True)[:3]
    I = torch.zeros((3, n_bins), device="cuda"); A = torch.zeros_like(I); isi = torch.zeros(3, device="cuda")
    ctx.reduce(out.data_ptr(), cnt.data_ptr(), 3, n_bins, width, I.data_ptr(), A.data_ptr(), isi.data_ptr(),
               torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    I, A, isi = I.cpu().numpy(), A.cpu().numpy(), isi.cpu().numpy()
    for e in range(3):
        rI, rA, rn, risi = oracle.reductions(ref[e], rcnt[e], w.voxel_nm, n_bins, width)
        scale = rI.max()
        assert np.abs(I[e] - rI).max() <= 2e-5 * scale, (e, np.abs(I[e] - rI).max() / scale)
        sig = rI > 1e-4 * scale                         # A is a ratio: compare where the bin carries signal
        assert np.abs(A[e] - rA)[sig].max() <= 1e-4, (e, np.abs(A[e] - rA)[sig].max())
        assert abs(isi[e] - risi) <= 2e-5 * abs(risi)
    # the binning itself, bit-exact: reduce an image whose value is its own pixel index
    # (sums of distinct integers < 2^24 identify the set of pixels of every bin and sector)
    idx = torch.arange(nx * ny, dtype=torch.float32, device="cuda").reshape(1, ny, nx).contiguous()
    I1 = torch.zeros((1, n_bins), device="cuda"); A1 = torch.zeros_like(I1); s1 = torch.zeros(1, device="cuda")
    ctx.reduce(idx.data_ptr(), None, 1, n_bins, width, I1.data_ptr(), A1.data_ptr(), s1.data_ptr(),
               torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    rI, rA, rn, risi = oracle.reductions(idx[0].cpu().numpy().astype(np.float64), None, w.voxel_nm, n_bins, width)
    assert np.allclose(I1[0].cpu().numpy(), rI, rtol=2e-7, atol=0)
    assert np.allclose(A1[0].cpu().numpy(), rA, rtol=0, atol=2e-7)
    assert np.isclose(float(s1[0]), risi, rtol=2e-7)


def test_reduce_rejects_bad_arguments():
    import torch
    from paper_2209_13121_b200 import binding
    ctx = binding.Context(16, 16, 1, 1, 2.0)
    img = torch.zeros((1, 16, 16), device="cuda"); I = torch.zeros((1, 8), device="cuda")
    for bins, width in [(0, 20.0), (5000, 20.0), (8, 0.0), (8, 60.0)]:
        with pytest.raises(binding.CyrsoxsError) as ei:
            ctx.reduce(img.data_ptr(), None, 1, bins, width, I.data_ptr())
        assert ei.value.status == binding.ERR_INVALID_ARG
    ctx.close()


def test_aos_morphology_matches_soa():
    """cyrsoxs_set_morphology_aos (the paper's Real4 layout): same images, bit for bit,
    as the structure-of-arrays entry; an S == 0 material is detected as isotropic."""
    import torch
    from paper_2209_13121_b200 import binding
    w = W.tiny(seed=41, nx=32, ny=16, nz=8, n_mat=3, n_energy=2, voxel_nm=2.0)
    ref = binding.simulate(w, want_counts=True)
    n = w.Nx * w.Ny * w.Nz
    aos = np.zeros((w.n_mat, n, 4), np.float32)
    for m, (phi, S, th, ps) in enumerate(w.materials):
        aos[m, :, 0] = phi.ravel()
        if S is not None:
            aos[m, :, 1] = S.ravel(); aos[m, :, 2] = ps.ravel(); aos[m, :, 3] = th.ravel()
    d = torch.from_numpy(aos).cuda()
    ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    s = torch.cuda.current_stream().cuda_stream
    ctx.set_morphology_aos(d.data_ptr(), s)
    ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald)
    out = torch.empty((w.n_energy, w.Ny, w.Nx), dtype=torch.float32, device="cuda")
    ctx.run(out.data_ptr(), s)
    torch.cuda.synchronize()
    assert torch.equal(out, ref[0])
    # ... and against the oracle, fed from the SoA arrays the Real4 array was packed from (not only against the SoA GPU run)
    oref, ocnt = oracle_run(w)
    compare(out.cpu().numpy(), None, oref, ocnt, "aos-vs-oracle")
    # the isotropic last material was detected: same transform count as the SoA run
    assert ctx.stats()["stage_bytes"]["xpass"] == ref[-1].stats()["stage_bytes"]["xpass"]
    with pytest.raises(binding.CyrsoxsError):
        ctx.set_morphology_aos(0, s)
    ctx.close()


@pytest.mark.parametrize("alg", ALGS)
def test_degenerate_and_extreme_cases(alg):
    from paper_2209_13121_b200 import binding
    # the longest supported axis along z
    w = W.tiny(seed=51, nx=4, ny=4, nz=2048, n_mat=2, n_energy=1, voxel_nm=1.0, ewald=W.EWALD_TRILINEAR)
    ref, rcnt = oracle_run(w)
    out, cnt, _ = _gpu(w, alg)
    compare(out, cnt, ref, rcnt, "nz2048")
    # the largest material count (32: 31 aligned + 1 isotropic = 218 basis fields)
    w = W.tiny(seed=52, nx=8, ny=8, nz=4, n_mat=32, n_energy=2, voxel_nm=3.0, ewald=W.EWALD_NEAREST)
    ref, rcnt = oracle_run(w)
    out, cnt, _ = _gpu(w, alg)
    compare(out, cnt, ref, rcnt, "32-materials")
    # more energies than one batch holds (batches of 256), 2-D
    w = W.tiny(seed=53, nx=16, ny=8, nz=1, n_mat=2, n_energy=300, voxel_nm=4.0, energies=np.linspace(270.0, 340.0, 300))
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, ctx = _gpu(w, alg)
    compare(out, cnt, ref, rcnt, "300-energies")
    # an empty model (phi == 0 everywhere): every image is exactly zero, counts are pure geometry
    z = [(np.zeros_like(m[0]), None if m[1] is None else np.zeros_like(m[1]), None if m[2] is None else np.zeros_like(m[2]),
          None if m[3] is None else np.zeros_like(m[3])) for m in W.tiny(seed=54, nx=16, ny=16, nz=4, n_mat=2).materials]
    w0 = W.tiny(seed=54, nx=16, ny=16, nz=4, n_mat=2)
    w0 = W.Workload("empty", 16, 16, 4, w0.voxel_nm, z, w0.energies, w0.delta_par, w0.beta_par, w0.delta_perp, w0.beta_perp,
                    w0.angles, w0.ewald)
    ref, rcnt = oracle_run(w0)
    out, cnt, _ = _gpu(w0, alg)
    assert (out == 0).all() and (ref == 0).all() and (cnt == rcnt).all()


@pytest.mark.parametrize("nx", [32, 40])
@pytest.mark.parametrize("group", [1, 2, 5])
def test_streamed_morphology_matches_oracle(group, nx):
    """cyrsoxs_set_morphology_streamed (NEXT-3, the paper's Algorithm 2/3 idea): materials pass through
    a double-buffered staging area group by group; images within the gates, counts equal, and repeated
    runs (staging slots reused across runs) give identical images.  nx = 40: the groups go through the
    direct-DFT x pass (k_xdft) with their own slice of the basis plan."""
    import torch
    from paper_2209_13121_b200 import binding
    w = W.tiny(seed=61, nx=nx, ny=32, nz=8, n_mat=4, n_energy=3, voxel_nm=2.0, ewald=W.EWALD_TRILINEAR)
    ref, rcnt = oracle_run(w)
    pinned = [tuple(None if a is None else torch.from_numpy(a).pin_memory() for a in m) for m in w.materials]
    ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    ctx.set_morphology_streamed(pinned, group)
    ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald)
    out = torch.empty((w.n_energy, w.Ny, w.Nx), dtype=torch.float32, device="cuda")
    cnt = torch.zeros((w.n_energy, w.Ny, w.Nx), dtype=torch.int32, device="cuda")
    ctx.set_counts_output(cnt.data_ptr())
    s = torch.cuda.current_stream().cuda_stream
    ctx.run(out.data_ptr(), s)
    torch.cuda.synchronize()
    first = out.clone()
    compare(out.cpu().numpy(), cnt.cpu().numpy(), ref, rcnt, f"streamed g={group}")
    for _ in range(3):
        ctx.run(out.data_ptr(), s)
    torch.cuda.synchronize()
    assert torch.equal(out, first)
    ctx.set_algorithm(binding.ALG_PER_ENERGY)
    with pytest.raises(binding.CyrsoxsError) as ei:
        ctx.run(out.data_ptr(), s)
    assert ei.value.status == binding.ERR_NOT_IMPLEMENTED
    # a spectra shard needs a resident morphology (cyrsoxs.h): refused, not silently ignored
    ctx.set_algorithm(binding.ALG_AUTO)
    ctx.set_spectra_shard(1, 2)
    with pytest.raises(binding.CyrsoxsError) as ei:
        ctx.run_spectra(s)
    assert ei.value.status == binding.ERR_NOT_IMPLEMENTED
    ctx.set_spectra_shard(0, 1)
    # back to a resident morphology on the same context
    ctx.set_morphology_host(w.materials, s)
    ctx.run(out.data_ptr(), s)
    torch.cuda.synchronize()
    compare(out.cpu().numpy(), cnt.cpu().numpy(), ref, rcnt, "resident after streamed")
    ctx.close()


def test_setters_between_runs_on_a_non_blocking_stream_without_sync():
    """Two runs on a non-blocking side stream with cyrsoxs_set_optical_constants and cyrsoxs_set_angles in between and
    no synchronisation: the setters only touch host tables, the device copies are refreshed at the next run on its
    stream (cyrsoxs.h), so the first run's kernels keep the tables they were launched with."""
    import torch
    from paper_2209_13121_b200 import binding
    w = W.tiny(seed=62, nx=64, ny=64, nz=16, n_mat=3, n_energy=4, voxel_nm=2.0, ewald=W.EWALD_TRILINEAR)
    w2 = W.tiny(seed=63, nx=64, ny=64, nz=16, n_mat=3, n_energy=4, voxel_nm=2.0, ewald=W.EWALD_TRILINEAR, angles=(10.0, 25.0, 160.0))
    w2.materials = w.materials                               # same morphology, other constants and angles
    ref1, rcnt1 = oracle_run(w, linear=True)
    ref2, rcnt2 = oracle_run(w2, linear=True)
    side = torch.cuda.Stream()                               # non-blocking: not ordered against the legacy stream
    mats = [tuple(None if a is None else torch.from_numpy(a).cuda() for a in m) for m in w.materials]
    out1 = torch.empty((4, 64, 64), dtype=torch.float32, device="cuda")
    out2 = torch.empty_like(out1)
    cnt1 = torch.zeros((4, 64, 64), dtype=torch.int32, device="cuda")
    cnt2 = torch.zeros_like(cnt1)
    torch.cuda.synchronize()
    ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    ctx.set_morphology(mats)
    for rep in range(3):
        ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
        ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald)
        ctx.set_counts_output(cnt1.data_ptr())
        ctx.run(out1.data_ptr(), side.cuda_stream)
        ctx.set_optical_constants(w2.energies, w2.delta_par, w2.beta_par, w2.delta_perp, w2.beta_perp)     # no sync
        ctx.set_angles(*w2.angles)
        ctx.set_counts_output(cnt2.data_ptr())
        ctx.run(out2.data_ptr(), side.cuda_stream)
    side.synchronize()
    compare(out1.cpu().numpy(), cnt1.cpu().numpy(), ref1, rcnt1, "first of two back-to-back runs")
    compare(out2.cpu().numpy(), cnt2.cpu().numpy(), ref2, rcnt2, "second of two back-to-back runs")
    ctx.close()


@pytest.mark.parametrize("alg", ALGS)
def test_thin_film_nz63(alg):
    """A z axis that is not a power of two, as in the paper's validation model (Nz = 63): 128 x 128 x 63
    voxels, three materials, trilinear Ewald; the z pass is the pruned direct DFT."""
    w = W.tiny(seed=71, nx=128, ny=128, nz=63, n_mat=3, n_energy=3, voxel_nm=1.0, ewald=W.EWALD_TRILINEAR,
               angles=(0.0, 15.0, 165.0))
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, _ = _gpu(w, alg)
    print("nz63", compare(out, cnt, ref, rcnt, "nz63"))


def test_host_output_across_several_energy_batches():
    """Pinned-host `out` with more energies than one batch holds (batches of 256): the double-buffered
    staging area and the copy stream's events are exercised over three batches, twice in a row."""
    import torch
    from paper_2209_13121_b200 import binding
    w = W.tiny(seed=81, nx=16, ny=16, nz=2, n_mat=2, n_energy=600, voxel_nm=3.0, energies=np.linspace(270.0, 340.0, 600))
    ref, rcnt = oracle_run(w, linear=True)
    ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    s = torch.cuda.current_stream().cuda_stream
    ctx.set_morphology_host(w.materials, s)
    ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald)
    out = torch.zeros((w.n_energy, w.Ny, w.Nx), dtype=torch.float32).pin_memory()
    for _ in range(2):
        out.zero_()
        ctx.run(out.data_ptr(), s)
        torch.cuda.synchronize()
        assert ctx.stats()["energy_batch"] == 256
        compare(out.numpy(), None, ref, rcnt, "host-io-3-batches")
    ctx.close()


def test_context_reconfiguration_sequence():
    """One context driven through a sequence of reconfigurations (energies, angles, Ewald mode, algorithm,
    morphology); every run is compared with the oracle, so cached plans, tables and buffers must follow."""
    import torch
    from paper_2209_13121_b200 import binding
    base = W.tiny(seed=91, nx=32, ny=16, nz=8, n_mat=3, n_energy=12, voxel_nm=2.0, ewald=W.EWALD_TRILINEAR)
    dev = torch.device("cuda")
    mats = [tuple(None if a is None else torch.from_numpy(a).to(dev) for a in m) for m in base.materials]
    ctx = binding.Context(base.Nx, base.Ny, base.Nz, base.n_mat, base.voxel_nm)
    ctx.set_morphology(mats)
    s = torch.cuda.current_stream().cuda_stream
    steps = [
        dict(idx=range(12), angles=(0.0, 30.0, 150.0), ewald=W.EWALD_TRILINEAR, alg=binding.ALG_AUTO),
        dict(idx=range(3), angles=(0.0, 30.0, 150.0), ewald=W.EWALD_TRILINEAR, alg=binding.ALG_AUTO),
        dict(idx=range(3), angles=(10.0, 7.0, 94.0), ewald=W.EWALD_NEAREST, alg=binding.ALG_AUTO),
        dict(idx=range(2, 11), angles=(10.0, 7.0, 94.0), ewald=W.EWALD_NEAREST, alg=binding.ALG_PER_ENERGY),
        dict(idx=[5], angles=(45.0, 0.0, 45.0), ewald=W.EWALD_TRILINEAR, alg=binding.ALG_SPECTRAL_BASIS),
        dict(idx=range(12), angles=(0.0, 90.0, 270.0), ewald=W.EWALD_TRILINEAR, alg=binding.ALG_AUTO),
    ]
    for k, st in enumerate(steps):
        w = base.restrict_energies(list(st["idx"]))
        w.angles, w.ewald = st["angles"], st["ewald"]
        if k == 4:      # a different morphology on the same context: isotropic-only
            iso = [(m[0], None, None, None) for m in base.materials]
            w = W.Workload("iso", w.Nx, w.Ny, w.Nz, w.voxel_nm, iso, w.energies, w.delta_par, w.beta_par, w.delta_par,
                           w.beta_par, w.angles, w.ewald)
            ctx.set_morphology([(m[0], None, None, None) for m in mats])
        elif k == 5:
            ctx.set_morphology(mats)
        ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
        ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald); ctx.set_algorithm(st["alg"])
        out = torch.empty((w.n_energy, w.Ny, w.Nx), dtype=torch.float32, device=dev)
        cnt = torch.zeros((w.n_energy, w.Ny, w.Nx), dtype=torch.int32, device=dev)
        ctx.set_counts_output(cnt.data_ptr())
        ctx.run(out.data_ptr(), s)
        torch.cuda.synchronize()
        ref, rcnt = oracle_run(w)
        compare(out.cpu().numpy(), cnt.cpu().numpy(), ref, rcnt, f"reconfig step {k}")
    ctx.close()


def test_streamed_cfg3_reduced():
    """The CFG3 recipe (3 materials, Voronoi grains, trilinear) at 64 x 64 x 32 through the streamed mode,
    one material per group, pinned-host output."""
    import torch
    from paper_2209_13121_b200 import binding
    w = W.cfg3(nx=64, ny=64, nz=32, n_energy=4, grain=8.0)
    ref, rcnt = oracle_run(w, linear=True)
    pinned = [tuple(None if a is None else torch.from_numpy(a).pin_memory() for a in m) for m in w.materials]
    ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    ctx.set_morphology_streamed(pinned, 1)
    ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald)
    out = torch.zeros((w.n_energy, w.Ny, w.Nx), dtype=torch.float32).pin_memory()
    s = torch.cuda.current_stream().cuda_stream
    ctx.run(out.data_ptr(), s)
    torch.cuda.synchronize()
    compare(out.numpy(), None, ref, rcnt, "cfg3/64 streamed")
    ctx.close()


@pytest.mark.parametrize("shape,n_mat,n_energy", [((128, 128, 128), 2, 10), ((64, 32, 16), 3, 5), ((256, 256, 1), 2, 1)])
def test_P14_footprint_bound(shape, n_mat, n_energy):
    """Device scratch against the memory model (Table 1 counts (4c + 6) N + 2 NxNy reals for Alg. 1): the
    SPECTRAL_BASIS workspace is at most three pruned copies of the n_pack complex basis cubes plus the interleaved
    images, i.e. <= 3 * 8 * n_pack * N + 16 * NxNy * (n_energy rounded up to a group of 8) bytes, and it does not
    grow when the same run is repeated."""
    from paper_2209_13121_b200 import binding
    nx, ny, nz = shape
    w = W.tiny(seed=5, nx=nx, ny=ny, nz=nz, n_mat=n_mat, n_energy=n_energy, voxel_nm=2.0)
    out, ctx = binding.simulate(w, algorithm=binding.ALG_SPECTRAL_BASIS)
    n_fields = sum(7 if m[1] is not None else 1 for m in w.materials)
    n_pack = (n_fields + 1) // 2
    N = nx * ny * nz
    pitch_factor = max(1.0, 32.0 / nx)                       # rows are padded to 32 complex values
    bound = 3 * 8 * n_pack * N * pitch_factor + 16 * nx * ny * ((n_energy + 7) // 8 * 8) + 4096
    ws = ctx.stats()["workspace_bytes"]
    assert 0 < ws <= bound, (ws, bound)
    import torch
    ctx.run(out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert ctx.stats()["workspace_bytes"] == ws


@pytest.mark.parametrize("n_mat,n_parts", [(2, 2), (4, 2), (4, 3), (3, 3)])
def test_spectra_shards_and_energy_ranges_match_oracle(n_mat, n_parts):
    """The strong-scaling path of DESIGN 11 on ONE GPU, its ranks emulated one after the other (nothing waits on anything):
    context q transforms material group q (cyrsoxs_set_spectra_shard, cyrsoxs_run_spectra), the blocks of the other
    groups are copied in from their owners' buffers (the broadcast of sharding.exchange_spectra as device copies), then
    every context runs its own energy range (cyrsoxs_run_energies) -- images and counts against the oracle."""
    import torch
    from paper_2209_13121_b200 import binding, sharding
    w = W.tiny(seed=90 + n_mat, nx=64, ny=32, nz=16, n_mat=n_mat, n_energy=5, voxel_nm=2.0, ewald=W.EWALD_TRILINEAR, isotropic_last=True)
    ref, rcnt = oracle_run(w, linear=True)
    aligned = [m[1] is not None for m in w.materials]
    s = torch.cuda.current_stream().cuda_stream
    mats = [tuple(None if a is None else torch.from_numpy(a).cuda() for a in m) for m in w.materials]
    slices = sharding.energy_slices(w.n_energy, n_parts)
    ctxs, specs = [], []
    for q in range(n_parts):
        ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
        ctx.set_morphology(mats)
        ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)     # ALL energies
        ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald)
        ctx.set_spectra_shard(q, n_parts)
        ctx.set_energy_range(slices[q][0], slices[q][1] - slices[q][0])
        ctx.run_spectra(s)
        ranges = [ctx.spectra_part(p) for p in range(n_parts)]
        assert ranges == sharding.pack_ranges(aligned, n_parts)
        ctxs.append(ctx); specs.append(sharding.spectra_tensor(ctx))
    torch.cuda.synchronize()
    assert all(sp.shape == specs[0].shape for sp in specs)
    for q in range(n_parts):                                        # "broadcast" part p from its owner p to everybody
        for p, (first, n) in enumerate(ranges):
            if p != q:
                specs[q][first:first + n].copy_(specs[p][first:first + n])
    for q in range(n_parts):
        a, b = slices[q]
        out = torch.empty((b - a, w.Ny, w.Nx), dtype=torch.float32, device="cuda")
        cnt = torch.zeros((b - a, w.Ny, w.Nx), dtype=torch.int32, device="cuda")
        ctxs[q].set_counts_output(cnt.data_ptr())
        ctxs[q].run_energies(out.data_ptr(), s)
        torch.cuda.synchronize()
        compare(out.cpu().numpy(), cnt.cpu().numpy(), ref[a:b], rcnt[a:b], f"shard {q}/{n_parts}")
    # run_energies without spectra is refused; an energy range outside the tables too
    fresh = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    fresh.set_morphology(mats)
    fresh.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    fresh.set_angles(*w.angles)
    out = torch.empty((w.n_energy, w.Ny, w.Nx), dtype=torch.float32, device="cuda")
    with pytest.raises(binding.CyrsoxsError) as ei:
        fresh.run_energies(out.data_ptr(), s)
    assert ei.value.status == binding.ERR_NOT_READY
    fresh.set_energy_range(3, 4)
    with pytest.raises(binding.CyrsoxsError) as ei:
        fresh.run(out.data_ptr(), s)
    assert ei.value.status == binding.ERR_INVALID_ARG
    # an energy range through plain cyrsoxs_run
    fresh.set_energy_range(1, 3)
    fresh.run(out.data_ptr(), s)
    torch.cuda.synchronize()
    compare(out[:3].cpu().numpy(), None, ref[1:4], rcnt[1:4], "energy range 1..3")
    for c in ctxs + [fresh]:
        c.close()


def test_spectra_do_not_survive_an_algorithm_switch():
    """cyrsoxs_run_energies only accepts spectra that the SPECTRAL_BASIS path produced under the current setting: under
    PER_ENERGY phase 1 is empty and phase 2 leaves per-energy chi spectra in the same buffer, so switching the algorithm
    between the phases must give NOT_READY (also for cyrsoxs_get_spectra), not images from the wrong buffer."""
    import torch
    from paper_2209_13121_b200 import binding
    w = W.tiny(seed=77, nx=32, ny=32, nz=8, n_mat=2, n_energy=3, voxel_nm=2.0, ewald=W.EWALD_TRILINEAR)
    ref, rcnt = oracle_run(w)
    s = torch.cuda.current_stream().cuda_stream
    mats = [tuple(None if a is None else torch.from_numpy(a).cuda() for a in m) for m in w.materials]
    ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    ctx.set_morphology(mats)
    ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald)
    out = torch.empty((w.n_energy, w.Ny, w.Nx), dtype=torch.float32, device="cuda")

    def refused(fn):
        with pytest.raises(binding.CyrsoxsError) as ei:
            fn()
        assert ei.value.status == binding.ERR_NOT_READY

    # PER_ENERGY: run_spectra is a no-op, a whole run fills the buffers with chi spectra -- neither makes spectra "ready"
    ctx.set_algorithm(binding.ALG_PER_ENERGY)
    ctx.run_spectra(s)
    refused(ctx.spectra)
    ctx.run(out.data_ptr(), s)
    torch.cuda.synchronize()
    compare(out.cpu().numpy(), None, ref, rcnt, "per-energy")
    ctx.set_algorithm(binding.ALG_SPECTRAL_BASIS)
    refused(lambda: ctx.run_energies(out.data_ptr(), s))
    refused(ctx.spectra)
    # the regular two-phase sequence works, and a later PER_ENERGY run takes the spectra away again
    ctx.run_spectra(s)
    out.zero_()
    ctx.run_energies(out.data_ptr(), s)
    torch.cuda.synchronize()
    compare(out.cpu().numpy(), None, ref, rcnt, "two-phase")
    ctx.set_algorithm(binding.ALG_PER_ENERGY)
    ctx.set_algorithm(binding.ALG_SPECTRAL_BASIS)
    refused(lambda: ctx.run_energies(out.data_ptr(), s))
    ctx.close()


def test_director_angles_of_tens_of_radians():
    """cyrsoxs.h states the angle range: SPECTRAL_BASIS takes sin/cos of theta and psi from the hardware approximation
    without extended range reduction, so unwrapped angles of tens of radians cost accuracy (about 6e-8 |angle| per
    director component) but nothing worse; PER_ENERGY (sincosf) keeps the full gates.  The oracle gets the same float32
    angles and evaluates them in double."""
    w = W.tiny(seed=88, nx=32, ny=32, nz=8, n_mat=3, n_energy=2, voxel_nm=2.0, ewald=W.EWALD_TRILINEAR)
    rng = np.random.default_rng(88)
    mats = []
    for phi, S, th, ps in w.materials:
        if S is None:
            mats.append((phi, S, th, ps))
        else:       # same directors, unwrapped by random multiples of 2 pi up to +-8 turns (|angle| up to 56 rad)
            turns = lambda: rng.integers(-8, 9, phi.shape).astype(np.float64) * 2.0 * np.pi
            mats.append((phi, S, (th.astype(np.float64) + turns()).astype(np.float32), (ps.astype(np.float64) + turns()).astype(np.float32)))
    w2 = W.Workload("unwrapped", w.Nx, w.Ny, w.Nz, w.voxel_nm, mats, w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp,
                    w.angles, w.ewald)
    ref, rcnt = oracle_run(w2)
    out, cnt, _ = _gpu(w2, 1)                                   # PER_ENERGY: full gates
    compare(out, cnt, ref, rcnt, "unwrapped per-energy")
    out, cnt, _ = _gpu(w2, 2)                                   # SPECTRAL_BASIS: the documented degradation, no more
    assert np.isfinite(out).all() and np.array_equal(cnt, rcnt)
    for e in range(w2.n_energy):
        l2 = np.linalg.norm(out[e] - ref[e]) / np.linalg.norm(ref[e])
        assert l2 <= 2e-4, (e, l2)
        print("unwrapped spectral-basis e", e, "relative L2", l2)


def _random_case(i):
    """Seeded random small case: sizes (powers of two or not), 1-6 materials with a random aligned / isotropic pattern,
    1-12 energies, voxel sizes from 0.3 to 8 nm (Ewald disk far inside the detector ... far outside), both Ewald modes,
    random angle lists."""
    rng = np.random.default_rng(7000 + i)
    sizes = [4, 6, 8, 12, 16, 20, 32, 33, 48, 64, 96, 100, 128]
    nx, ny = int(rng.choice(sizes)), int(rng.choice([2, 3] + sizes))
    nz = int(rng.choice([1, 1, 2, 3, 4, 5, 8, 16, 17, 32]))
    n_mat = int(rng.integers(1, 7))
    n_energy = int(rng.integers(1, 13))
    voxel = float(rng.choice([0.3, 0.7, 1.0, 1.3, 2.0, 3.7, 8.0]))
    mode = int(rng.integers(0, 2))
    start = float(rng.choice([0.0, 0.0, 7.5, -30.0]))
    step = float(rng.choice([5.0, 15.0, 22.5, 45.0, 90.0]))
    end = start + step * int(rng.integers(0, 12))
    w = W.tiny(seed=8000 + i, nx=nx, ny=ny, nz=nz, n_mat=n_mat, n_energy=n_energy, voxel_nm=voxel, ewald=mode,
               angles=(start, step, end), energies=np.sort(rng.uniform(250.0, 600.0, n_energy)))
    # random aligned / isotropic pattern (tiny() makes only the last material isotropic)
    mats = []
    for m, (phi, S, th, ps) in enumerate(w.materials):
        if S is not None and rng.random() < 0.35:
            mats.append((phi, None, None, None))
            w.delta_perp[:, m] = w.delta_par[:, m]; w.beta_perp[:, m] = w.beta_par[:, m]
        else:
            mats.append((phi, S, th, ps))
    w.materials = mats
    return w


@pytest.mark.parametrize("i", range(48))
def test_random_cases_match_oracle(i):
    w = _random_case(i)
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, _ = _gpu(w, 0)
    if ref.max() == 0.0:                                     # nothing on the Ewald sphere at all: exact zeros on both sides
        assert (out == 0).all() and (cnt == rcnt).all()
        return
    compare(out, cnt, ref, rcnt, f"random {i}: {w.Nx}x{w.Ny}x{w.Nz}, {w.n_mat} materials, {w.n_energy} energies, {w.voxel_nm} nm")


@pytest.mark.parametrize("case", ["32 aligned materials", "300 energies", "360 angles", "32 materials 2-D"])
def test_extreme_parameters(case):
    """The ends of the accepted parameter ranges: n_mat = 32 all aligned (224 basis fields, 112 packs), 300 energies
    (two energy batches of 256 + 44, three image-group widths), 360 angles (0:1:359), and 32 materials on a 2-D film (more
    packs than the 2-D Ewald kernel's register file holds: the generic kernel takes over)."""
    if case == "32 aligned materials":
        w = W.tiny(seed=201, nx=64, ny=16, nz=4, n_mat=32, n_energy=2, voxel_nm=2.0, ewald=W.EWALD_TRILINEAR, isotropic_last=False)
    elif case == "300 energies":
        w = W.tiny(seed=202, nx=32, ny=32, nz=2, n_mat=2, n_energy=300, voxel_nm=2.0, ewald=W.EWALD_NEAREST,
                   energies=np.linspace(260.0, 700.0, 300))
    elif case == "360 angles":
        w = W.tiny(seed=203, nx=32, ny=16, nz=4, n_mat=2, n_energy=2, voxel_nm=1.0, ewald=W.EWALD_TRILINEAR, angles=(0.0, 1.0, 359.0))
    else:
        w = W.tiny(seed=204, nx=64, ny=64, nz=1, n_mat=32, n_energy=6, voxel_nm=2.0, ewald=W.EWALD_NEAREST)
    ref, rcnt = oracle_run(w, linear=True)
    out, cnt, ctx = _gpu(w, 0)
    compare(out, cnt, ref, rcnt, case)
    if case == "300 energies":
        assert ctx.stats()["energy_batch"] == 256
