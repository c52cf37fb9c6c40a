"""Pins for the CPU oracle (no GPU, no CUDA code): each test ties oracle/ to something
other than itself -- brute force, a library routine (numpy.fft), a closed form, an
invariance the paper states, or a worked value stored under tests/golden/.

Pin numbers follow SURVEY.md 8(c) / DESIGN.md 6.  P:n = /root/reference/PAPER.md line n.
"""
import json
import os

import numpy as np
import pytest
from scipy import special

import oracle
from paper_2209_13121_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
PI = np.pi


def _consts(w, e=0):
    return oracle.coefficients(w.delta_par[e], w.beta_par[e], w.delta_perp[e], w.beta_perp[e])


def _run(w, **kw):
    return oracle.run(w.materials, w.voxel_nm, w.energies, w.delta_par, w.beta_par, w.delta_perp,
                      w.beta_perp, w.angles, w.ewald, **kw)


def _iso_film(phi1, d1, b1, d2, b2, voxel, E, angles, ewald=W.EWALD_NEAREST):
    """Two isotropic materials, phi2 = 1 - phi1."""
    phi1 = np.ascontiguousarray(phi1, np.float32)
    mats = [(phi1, None, None, None), (np.ascontiguousarray(1.0 - phi1, dtype=np.float32), None, None, None)]
    nz, ny, nx = phi1.shape
    f = lambda a, b: np.array([[a, b]], np.float32)
    return W.Workload("iso", nx, ny, nz, voxel, mats, np.array([E]), f(d1, d2), f(b1, b2), f(d1, d2), f(b1, b2),
                      angles, ewald)


# ---------------------------------------------------------------- O0 constants

def test_wavenumber_and_coefficients_closed_form():
    # lambda[nm] = 1239.84197 / E, k = 2 pi / lambda (north_star).  285 eV -> 1.4443033 nm^-1
    k = oracle.wavenumber(285.0)
    assert abs(k - 2 * PI * 285.0 / 1239.84197) < 1e-15
    assert abs(k - 1.4443033) < 1e-7
    dpar, bpar, dperp, bperp = 2e-3, 1e-3, 5e-4, 2e-4
    a, b, c = oracle.coefficients([dpar], [bpar], [dperp], [bperp])
    f = lambda x: float(np.float32(x))
    npar = 1 - f(dpar) + 1j * f(bpar)
    nperp = 1 - f(dperp) + 1j * f(bperp)
    niso = (npar + 2 * nperp) / 3          # Trace(N)/3, Eq. 2
    assert abs(a[0] - (nperp ** 2 - 1)) < 1e-15
    assert abs(b[0] - (npar ** 2 - nperp ** 2)) < 1e-15
    assert abs(c[0] - (niso ** 2 - 1)) < 1e-15
    # the isotropic part is the square of the mean, not the mean of squares (DESIGN 3-A2)
    assert abs(c[0] - ((npar ** 2 + 2 * nperp ** 2) / 3 - 1)) > 1e-8


def test_angle_list_and_snapping():
    assert oracle.num_angles(0, 15, 165) == 12
    assert oracle.num_angles(0, 5, 175) == 36
    assert oracle.num_angles(0, 2, 180) == 91          # P:483 "0 to 180 at an increment of 2"
    assert oracle.num_angles(30, 0, 30) == 1
    assert oracle.num_angles(0, 0, 10) == -1
    assert oracle.num_angles(10, 5, 0) == -1
    assert oracle.angle_cs(90.0) == (0.0, 1.0)
    assert oracle.angle_cs(180.0) == (-1.0, 0.0)
    assert oracle.angle_cs(0.0) == (1.0, 0.0)
    c, s = oracle.angle_cs(30.0)
    assert abs(c - np.sqrt(3) / 2) < 1e-15 and abs(s - 0.5) < 1e-15


# ---------------------------------------------------------------- P1 brute-force DFT

def test_P1_fft_vs_bruteforce_and_library():
    rng = np.random.default_rng(1)
    f = rng.standard_normal((4, 8, 8)) + 1j * rng.standard_normal((4, 8, 8))
    F = oracle.fft3(f)
    Fn = oracle.dft3_naive(f)
    assert np.abs(F - Fn).max() <= 1e-12 * np.abs(Fn).max()
    assert np.abs(F - np.fft.fftn(f)).max() <= 1e-12 * np.abs(Fn).max()
    # a single voxel at (z,y,x) = (1,2,3): sign and axis order of the exponent
    d = np.zeros((4, 8, 8), complex); d[1, 2, 3] = 1.0
    D = oracle.fft3(d)
    kz, ky, kx = np.meshgrid(np.arange(4), np.arange(8), np.arange(8), indexing="ij")
    assert np.abs(D - np.exp(-2j * PI * (kx * 3 / 8 + ky * 2 / 8 + kz * 1 / 4))).max() < 1e-13
    # non-cubic, larger, against the library
    g = rng.standard_normal((8, 16, 32)) + 1j * rng.standard_normal((8, 16, 32))
    assert np.abs(oracle.fft3(g) - np.fft.fftn(g)).max() < 1e-10


def test_P1_full_pipeline_with_bruteforce_dft():
    """Algorithm 1 assembled from the stage functions with the O(N^2) DFT in place of the FFT."""
    w = W.tiny(seed=5, nx=8, ny=8, nz=4, n_mat=3, n_energy=1)
    out, cnt = _run(w)
    a, b, c = _consts(w)
    k = oracle.wavenumber(w.energies[0])
    acc = np.zeros((w.Ny, w.Nx)); n = np.zeros((w.Ny, w.Nx), np.uint32)
    for i in range(w.n_angles):
        z = w.angles[0] + i * w.angles[1]
        C, S = oracle.angle_cs(z)
        p = oracle.polarization(w.materials, a, b, c, (C, S, 0.0))
        P = np.stack([oracle.dft3_naive(p[j]) for j in range(3)])
        img, valid = oracle.ewald(P, w.voxel_nm, k, w.ewald)
        oracle.rotate_accumulate(img, valid, z, acc, n)
    ref = np.where(n > 0, acc / np.maximum(n, 1), 0.0)
    assert (n == cnt[0]).all()
    assert np.abs(out[0] - ref).max() <= 1e-12 * ref.max()


def test_dft_bins_match_fft():
    """Pins only the bin SUMMATION of polarization_dft_bins (Eq. 6 written out for single bins) against the
    FFT of the same field; the polarization itself comes from the one statement orc_polarization on both sides
    and is pinned elsewhere (P2, P3, P9, P10, R2a)."""
    w = W.tiny(seed=6, nx=16, ny=8, nz=4, n_mat=2, n_energy=1)
    a, b, c = _consts(w)
    e = (0.3, -0.8, 0.0)
    P = np.stack([oracle.fft3(x) for x in oracle.polarization(w.materials, a, b, c, e)])
    bins = np.array([[0, 0, 0], [3, 5, 1], [-2, 7, -1], [15, 0, 3], [8, -4, 2]], np.int32)
    got = oracle.polarization_dft_bins(w.materials, a, b, c, e, bins)
    for q, (kx, ky, kz) in enumerate(bins):
        ref = P[:, kz % 4, ky % 8, kx % 16]
        assert np.abs(got[q] - ref).max() <= 1e-12 * np.abs(P).max()


# ---------------------------------------------------------------- P2 uniform film

def test_P2_uniform_isotropic_film_closed_form():
    """All intensity at q = 0 with I(0) = k^4 N^2 |n^2-1|^2 / (16 pi^2); worked value in
    tests/golden/p2_uniform_film.json (256x256x1, delta=1e-3, beta=5e-4, 285 eV)."""
    gold = json.load(open(os.path.join(GOLDEN, "p2_uniform_film.json")))
    n = gold["N_side"]
    phi = np.ones((1, n, n), np.float32)
    f = lambda v: np.array([[v]], np.float32)
    d, b = gold["delta"], gold["beta"]
    out, cnt = oracle.run([(phi, None, None, None)], gold["voxel_nm"], [gold["energy_eV"]], f(d), f(b), f(d), f(b),
                          (0.0, 0.0, 0.0), W.EWALD_NEAREST)
    c = n // 2
    # the stored value is for the decimal constants; the float32-rounded inputs move it by ~1e-7
    assert abs(out[0, c, c] - gold["I0"]) <= 3e-7 * gold["I0"]
    # independent evaluation of the closed form
    k = 2 * PI * gold["energy_eV"] / 1239.84197
    nn = 1 - float(np.float32(d)) + 1j * float(np.float32(b))
    I0 = k ** 4 * (n * n) ** 2 * abs(nn ** 2 - 1) ** 2 / (16 * PI ** 2)
    assert abs(out[0, c, c] - I0) <= 1e-12 * I0
    off = out[0].copy(); off[c, c] = 0
    assert off.max() <= 1e-20 * I0
    assert (cnt == 1).all()                       # k/dq = 294 px > half-diagonal: every pixel on the sphere

    # with the CFG1 angle set the centre keeps I(0); neighbours get the bilinear leakage
    angles = (0.0, 15.0, 165.0)
    out, cnt = oracle.run([(phi, None, None, None)], gold["voxel_nm"], [gold["energy_eV"]], f(d), f(b), f(d), f(b),
                          angles, W.EWALD_NEAREST)
    assert abs(out[0, c, c] - I0) <= 1e-12 * I0
    for (dy, dx) in [(0, 1), (1, 0), (1, 1), (-1, 1), (0, -1), (-1, -1)]:
        tot = 0.0
        for i in range(12):
            z = np.deg2rad(15.0 * i)
            C, S = np.cos(z), np.sin(z)
            fx, fy = C * dx - S * dy, S * dx + C * dy          # source position relative to the centre
            wx = max(0.0, 1 - abs(fx)); wy = max(0.0, 1 - abs(fy))
            tot += wx * wy * I0
        expect = tot / cnt[0, c + dy, c + dx]
        assert abs(out[0, c + dy, c + dx] - expect) <= 1e-9 * I0


# ---------------------------------------------------------------- P3 split materials

def test_P3_split_material_invariance():
    """P:104 (a component may be split into materials with identical dielectric functions and
    volume fractions adding up) and P:110 (s v_frac = absolute oriented fraction)."""
    w = W.tiny(seed=7, nx=8, ny=8, nz=4, n_mat=2, n_energy=1, isotropic_last=False)
    out0, cnt0 = _run(w)
    phi, S, th, ps = w.materials[0]
    rng = np.random.default_rng(0)
    # multiples of 1/8 keep phi' + phi'' == phi exactly in float32
    frac = (rng.integers(1, 8, phi.shape) / 8.0).astype(np.float32)
    m1a = ((phi * frac).astype(np.float32), S, th, ps)
    m1b = ((phi - phi * frac).astype(np.float32), S, th, ps)
    col = lambda x: np.concatenate([x[:, :1], x[:, :1], x[:, 1:]], 1)
    out1, cnt1 = oracle.run([m1a, m1b, w.materials[1]], w.voxel_nm, w.energies, col(w.delta_par), col(w.beta_par),
                            col(w.delta_perp), col(w.beta_perp), w.angles, w.ewald)
    assert (cnt0 == cnt1).all()
    assert np.abs(out1 - out0).max() <= 1e-6 * out0.max()     # float32 rounding of the split only
    # (phi, S) == aligned (phi S, 1) + isotropic (phi (1-S), 0) with the same constants
    S8 = (np.round(S * 8) / 8).astype(np.float32); phi8 = (np.round(phi * 8) / 8).astype(np.float32)
    base, cb = oracle.run([(phi8, S8, th, ps), w.materials[1]], w.voxel_nm, w.energies, w.delta_par, w.beta_par,
                          w.delta_perp, w.beta_perp, w.angles, w.ewald)
    al = ((phi8 * S8).astype(np.float32), np.ones_like(S8), th, ps)
    un = ((phi8 * (1 - S8)).astype(np.float32), None, None, None)
    spl, cs = oracle.run([al, un, w.materials[1]], w.voxel_nm, w.energies, col(w.delta_par), col(w.beta_par),
                         col(w.delta_perp), col(w.beta_perp), w.angles, w.ewald)
    assert (cb == cs).all()
    assert np.abs(spl - base).max() <= 1e-12 * base.max()


# ---------------------------------------------------------------- P4 Parseval

def test_P4_parseval():
    w = W.tiny(seed=8, nx=16, ny=8, nz=8, n_mat=3, n_energy=1)
    a, b, c = _consts(w)
    p = oracle.polarization(w.materials, a, b, c, (0.6, 0.8, 0.0))
    for i in range(3):
        P = oracle.fft3(p[i])
        lhs = (np.abs(P) ** 2).sum(); rhs = p[i].size * (np.abs(p[i]) ** 2).sum()
        assert abs(lhs - rhs) <= 1e-12 * rhs


# ---------------------------------------------------------------- P5 linearity in e

@pytest.mark.parametrize("mode", [W.EWALD_NEAREST, W.EWALD_TRILINEAR])
def test_P5_linearity_and_linear_mode(mode):
    w = W.tiny(seed=9, nx=16, ny=16, nz=8, n_mat=3, n_energy=1, voxel_nm=2.0, ewald=mode)
    a, b, c = _consts(w)
    k = oracle.wavenumber(w.energies[0])
    Px = np.stack([oracle.fft3(x) for x in oracle.polarization(w.materials, a, b, c, (1, 0, 0))])
    Py = np.stack([oracle.fft3(x) for x in oracle.polarization(w.materials, a, b, c, (0, 1, 0))])
    Ixx, Iyy, Ixy, valid = oracle.ewald_linear(Px, Py, w.voxel_nm, k, mode)
    for z in (0.0, 25.0, 90.0, 140.0):
        C, S = oracle.angle_cs(z)
        P = np.stack([oracle.fft3(x) for x in oracle.polarization(w.materials, a, b, c, (C, S, 0))])
        img, v2 = oracle.ewald(P, w.voxel_nm, k, mode)
        assert (v2 == valid).all()
        lin = C * C * Ixx + S * S * Iyy + 2 * C * S * Ixy
        assert np.abs(img - lin).max() <= 1e-12 * img.max()
    o1, c1 = _run(w)
    o2, c2 = _run(w, linear=True)
    assert (c1 == c2).all() and np.abs(o1 - o2).max() <= 1e-12 * o1.max()


def test_linear_mode_equals_definition_mode_cfg1():
    w = W.cfg1(n=64, n_disks=6, radius=5)
    o1, c1 = _run(w); o2, c2 = _run(w, linear=True)
    assert (c1 == c2).all() and np.abs(o1 - o2).max() <= 1e-12 * o1.max()


# ---------------------------------------------------------------- P6 isotropic zeta law

def test_P6_isotropic_zeta_law():
    """All-isotropic input: p~ = chi~ e, so I_zeta (1-(r.e0)^2) = I_0 (1-(r.e_zeta)^2) pixel by pixel."""
    rng = np.random.default_rng(3)
    n = 32
    phi = rng.uniform(0, 1, (1, n, n)).astype(np.float32)
    w = _iso_film(phi, 2e-3, 1e-3, 5e-4, 2e-4, 2.0, 285.0, (0, 0, 0))    # dq = 0.098: r_x, r_y reach 1
    a, b, c = _consts(w); k = oracle.wavenumber(285.0)
    dq = 2 * PI / (n * w.voxel_nm)
    m = np.arange(n) - n // 2
    rx = (m[None, :] * dq / k) * np.ones((n, 1)); ry = (m[:, None] * dq / k) * np.ones((1, n))
    imgs = {}
    for z in (0.0, 35.0):
        C, S = oracle.angle_cs(z)
        P = np.stack([oracle.fft3(x) for x in oracle.polarization(w.materials, a, b, c, (C, S, 0))])
        imgs[z], valid = oracle.ewald(P, w.voxel_nm, k, W.EWALD_NEAREST)
    C, S = oracle.angle_cs(35.0)
    lhs = imgs[35.0] * (1 - rx ** 2)
    rhs = imgs[0.0] * (1 - (rx * C + ry * S) ** 2)
    ok = valid.astype(bool)
    assert ok.sum() > 100 and (~ok).sum() > 0          # the sphere cuts the detector here
    assert np.abs(lhs - rhs)[ok].max() <= 1e-12 * imgs[0.0].max()


# ---------------------------------------------------------------- P7 form factors (Eq. 9)

def _axis_profile(out, axis):
    c = out.shape[0] // 2
    return out[c:, c] if axis == "y" else out[c, c:]


def test_P7_disk_and_projected_sphere_form_factor_zeros():
    """Eq. 9 for a projected sphere, 2 J1(x)/x for a flat disk: the zeros pin
    dq = 2 pi/(N voxel) and the pixel <-> q map.  Zeros: qR = 3.8317 (disk), 4.4934 (sphere)."""
    n, voxel = 512, 5.0
    y, x = np.mgrid[0:n, 0:n]
    dx = np.minimum(x, n - x).astype(float); dy = np.minimum(y, n - y).astype(float)   # centred on voxel 0 (periodic)
    r2 = dx ** 2 + dy ** 2
    dq = 2 * PI / (n * voxel)
    # (a) flat disk, R = 39 voxels: first zero at m = 3.8317 N / (2 pi R) = 8.006 pixels
    R = 39.0
    w = _iso_film((r2 <= R * R).astype(np.float32)[None], 2e-3, 1e-3, 0.0, 0.0, voxel, 285.0, (0, 0, 0))
    out, _ = _run(w)
    prof = _axis_profile(out[0], "y")           # q perpendicular to e: projector factor 1 - r_y^2 only
    m = np.arange(prof.size)
    assert np.argmin(prof[4:12]) + 4 == 8
    qR = m[1:7] * dq * R * voxel
    ana = (2 * special.j1(qR) / qR) ** 2
    got = prof[1:7] / prof[1] * ana[0]
    assert np.abs(got / ana - 1).max() < 0.03    # voxelised disk vs continuum ("finite discretization")
    # (b) projected sphere, phi = chord / diameter, R = 45.77 voxels: zero at m = 8.0
    R = 4.4934 * n / (2 * PI * 8.0)
    chord = np.sqrt(np.maximum(R * R - r2, 0.0)) / R
    w = _iso_film(chord.astype(np.float32)[None], 2e-3, 1e-3, 0.0, 0.0, voxel, 285.0, (0, 0, 0))
    out, _ = _run(w)
    prof = _axis_profile(out[0], "y")
    assert np.argmin(prof[4:12]) + 4 == 8
    qR = m[1:7] * dq * R * voxel
    ana = (3 * (np.sin(qR) - qR * np.cos(qR)) / qR ** 3) ** 2
    got = prof[1:7] / prof[1] * ana[0]
    assert np.abs(got / ana - 1).max() < 0.03


def test_P7_sphere_3d_axis_scale_z():
    """3-D sphere: the same zero seen through the Ewald sphere fixes dq_z's role: with a
    large k (hard x-rays, flat sphere) the q_z = 0 plane is sampled and Eq. 9 holds."""
    n, nz, voxel = 64, 64, 5.0
    R = 4.4934 * n / (2 * PI * 8.0) / 2       # zero at m = 16 -> R = 2.86... too small; use m = 8 on a 64 grid
    R = 4.4934 * n / (2 * PI * 8.0)           # 5.72 voxels, zero at pixel 8
    z, y, x = np.mgrid[0:nz, 0:n, 0:n]
    d2 = np.minimum(x, n - x) ** 2 + np.minimum(y, n - y) ** 2 + np.minimum(z, nz - z) ** 2
    # soft-edged sphere (sub-voxel anti-aliasing) keeps the continuum form factor at this small R
    phi = np.clip(R + 0.5 - np.sqrt(d2), 0.0, 1.0).astype(np.float32)
    w = _iso_film(phi, 2e-3, 1e-3, 0.0, 0.0, voxel, 17000.0, (0, 0, 0))      # 17 keV as in P:459
    out, cnt = _run(w)
    prof = _axis_profile(out[0], "y")
    assert np.argmin(prof[4:12]) + 4 == 8


# ---------------------------------------------------------------- P8 mirror symmetry

def test_P8_mirror_symmetry():
    rng = np.random.default_rng(4)
    n = 16
    half = rng.uniform(0, 1, (1, n, n))
    # symmetric under x -> (N - x) mod N (index reflection about voxel 0), directors mirrored: psi -> pi - psi
    idx = (-np.arange(n)) % n
    sym = lambda a: 0.5 * (a + a[:, :, idx])
    phi = sym(half).astype(np.float32)
    S = sym(rng.uniform(0, 1, (1, n, n))).astype(np.float32)
    th = sym(rng.uniform(0, PI, (1, n, n))).astype(np.float32)
    ps0 = rng.uniform(0, 2 * PI, (1, n, n))
    ps = np.where(np.arange(n)[None, None, :] <= n // 2, ps0, (PI - ps0[:, :, idx])).astype(np.float64)
    ps[:, :, 0] = PI / 2; ps[:, :, n // 2] = PI / 2            # self-mirrored columns: d_x = 0
    mats = [(phi, S, th, ps.astype(np.float32)), ((1 - phi).astype(np.float32), None, None, None)]
    f = lambda a, b: np.array([[a, b]], np.float32)
    out, cnt = oracle.run(mats, 5.0, [285.0], f(2e-3, 1e-3), f(1e-3, 5e-4), f(5e-4, 1e-3), f(2e-4, 5e-4),
                          (0, 0, 0), W.EWALD_NEAREST)
    img = out[0]
    c = n // 2
    # I(qx, qy) = I(-qx, qy): pixel ix <-> 2c - ix (ix = 0 has no partner)
    a_ = img[:, 1:]; b_ = img[:, 1:][:, ::-1]
    assert np.abs(a_ - b_).max() <= 2e-6 * img.max()       # float32 rounding of pi - psi


# ---------------------------------------------------------------- P9 two-fold anisotropy

def _sector_means(img, rmin, rmax, half_width_deg=20):
    n = img.shape[0]; c = n // 2
    y, x = np.mgrid[0:n, 0:n]; u, v = x - c, y - c
    r = np.hypot(u, v); ang = np.degrees(np.arctan2(v, u)) % 180.0
    ring = (r >= rmin) & (r <= rmax)
    par = ring & ((ang < half_width_deg) | (ang > 180 - half_width_deg))
    perp = ring & (np.abs(ang - 90) < half_width_deg)
    return img[par].mean(), img[perp].mean()


@pytest.mark.parametrize("b_sign", [+1, -1])
def test_P9_radial_vs_tangential_anisotropy(b_sign):
    """Disk with S = 1, theta = 90 deg, psi = atan2 (radial) in a matrix equal to the disk's
    isotropic average: chi_xx contrast is b (cos^2 psi - 1/3) = b (1/6 + cos(2 psi)/2), whose
    transform is A0(q)/6 - cos(2 chi) B2(q)/2 with A0, B2 > 0 at low q: more scattering
    perpendicular to e (A < 0) for radial, the opposite for tangential, whatever the sign of b."""
    n, voxel, R = 128, 5.0, 20.0
    y, x = np.mgrid[0:n, 0:n]
    u, v = x - n // 2, y - n // 2
    inside = (u * u + v * v <= R * R)
    phi = inside.astype(np.float32)[None]
    th = np.where(inside, np.float32(PI / 2), 0).astype(np.float32)[None]
    dpar, dperp = (3e-3, 1e-3) if b_sign > 0 else (1e-3, 3e-3)
    bpar = bperp = 0.0
    diso = (dpar + 2 * dperp) / 3
    f = lambda a, b: np.array([[a, b]], np.float32)
    res = {}
    for name, off in (("radial", 0.0), ("tangential", PI / 2)):
        ps = np.where(inside, np.arctan2(v, u) + off, 0).astype(np.float32)[None]
        mats = [(phi, phi.copy(), th, ps), ((1 - phi).astype(np.float32), None, None, None)]
        out, _ = oracle.run(mats, voxel, [285.0], f(dpar, diso), f(bpar, 0.0), f(dperp, diso), f(bperp, 0.0),
                            (0, 0, 0), W.EWALD_NEAREST)
        img = out[0]
        c = n // 2
        # two-fold: inversion symmetric (no absorption -> Friedel), but NOT four-fold
        inv = img[1:, 1:][::-1, ::-1]
        assert np.abs(img[1:, 1:] - inv).max() <= 1e-9 * img[1:, 1:].max()
        Ipar, Iperp = _sector_means(img, 2, 5)
        res[name] = (Ipar - Iperp) / (Ipar + Iperp)
    assert res["radial"] < -0.1
    assert res["tangential"] > 0.1


# ---------------------------------------------------------------- P10 binary film closed form / ISI law

def test_P10_binary_isotropic_film_closed_form_and_isi():
    """I_zeta(q) = k^4 |n1^2 - n2^2|^2 / (16 pi^2) |phi~1(q)|^2 (1 - ((qx C + qy S)/k)^2), q != 0,
    with phi~1 from numpy.fft.fft2; summed over q this is Eq. 10's (d delta^2 + d beta^2) E^4 law."""
    rng = np.random.default_rng(12)
    n, voxel = 32, 10.0
    phi = (rng.integers(0, 257, (1, n, n)) / 256.0).astype(np.float32)    # 1 - phi exact in float32
    d1, b1, d2, b2 = 2.2e-3, 0.9e-3, 0.7e-3, 0.3e-3
    isi = []
    for E in (270.0, 285.0, 310.0):
        for z in (0.0, 40.0):
            w = _iso_film(phi, d1, b1, d2, b2, voxel, E, (z, 0, z))
            a, b, c = _consts(w); k = oracle.wavenumber(E)
            C, S = oracle.angle_cs(z)
            P = np.stack([oracle.fft3(x) for x in oracle.polarization(w.materials, a, b, c, (C, S, 0))])
            img, valid = oracle.ewald(P, voxel, k, W.EWALD_NEAREST)
            F = np.fft.fftshift(np.fft.fft2(phi[0].astype(np.float64)))
            f32 = lambda v: float(np.float32(v))
            n1 = 1 - f32(d1) + 1j * f32(b1); n2 = 1 - f32(d2) + 1j * f32(b2)
            dq = 2 * PI / (n * voxel)
            m = np.arange(n) - n // 2
            qx = m[None, :] * dq; qy = m[:, None] * dq
            ref = k ** 4 * abs(n1 ** 2 - n2 ** 2) ** 2 / (16 * PI ** 2) * np.abs(F) ** 2 * (1 - ((qx * C + qy * S) / k) ** 2)
            ref[n // 2, n // 2] = img[n // 2, n // 2]
            assert valid.all()
            assert np.abs(img - ref).max() <= 1e-12 * ref.max()
            if z == 0.0:
                tmp = img.copy(); tmp[n // 2, n // 2] = 0
                isi.append((E, tmp.sum()))
    # Eq. 10: ISI ~ (d delta^2 + d beta^2) E^4 -> with fixed constants ISI / E^4 is flat to O(delta, (q/k)^2)
    r = [s / E ** 4 for E, s in isi]
    assert max(r) / min(r) - 1 < 2e-2


def test_P10_non_square_film_pins_dq_y_and_the_validity_ellipse():
    """P10 on a 48 x 32 x 1 detector whose Ewald disk is cut by the detector edge (Eq. 7-8).
    q_y = m_y 2 pi / (Ny voxel): with Nx != Ny the disk q_x^2 + q_y^2 <= k^2 is an ELLIPSE in pixels (k/dq_x = 17.65 px,
    k/dq_y = 11.77 px) and r^_y enters the (1 - (r^.e)^2) factor with dq_y, so a dq_y formed from Nx changes both the
    valid set and the values.  Everything on the right-hand side is written out in NumPy."""
    rng = np.random.default_rng(48)
    nx, ny, voxel, E = 48, 32, 1.6, 285.0
    phi = (rng.integers(0, 257, (1, ny, nx)) / 256.0).astype(np.float32)
    d1, b1, d2, b2 = 2.2e-3, 0.9e-3, 0.7e-3, 0.3e-3
    f32 = lambda v: float(np.float32(v))
    n1 = 1 - f32(d1) + 1j * f32(b1); n2 = 1 - f32(d2) + 1j * f32(b2)
    k = 2 * PI * E / 1239.84197
    dqx = 2 * PI / (nx * voxel); dqy = 2 * PI / (ny * voxel)
    qx = (np.arange(nx) - nx // 2)[None, :] * dqx; qy = (np.arange(ny) - ny // 2)[:, None] * dqy
    inside = qx ** 2 + qy ** 2 <= k ** 2
    assert abs(k / dqx - 17.65) < 0.01 and abs(k / dqy - 11.77) < 0.01
    assert 0 < inside.sum() < inside.size and not inside[0, nx // 2] and not inside[ny // 2, 0]     # cut on both axes
    assert np.abs(qx ** 2 + qy ** 2 - k ** 2).min() > 1e-6 * k ** 2                                 # no pixel on the rim
    wrong = qx ** 2 + ((np.arange(ny) - ny // 2)[:, None] * dqx) ** 2 <= k ** 2                     # the mistake this pins
    assert (wrong != inside).sum() > 50
    F = np.fft.fftshift(np.fft.fft2(phi[0].astype(np.float64)))
    for z in (0.0, 40.0):
        w = _iso_film(phi, d1, b1, d2, b2, voxel, E, (z, 0, z))
        a, b, c = _consts(w)
        assert abs(oracle.wavenumber(E) - k) <= 1e-15 * k
        C, S = np.cos(np.deg2rad(z)), np.sin(np.deg2rad(z))
        P = np.stack([oracle.fft3(x) for x in oracle.polarization(w.materials, a, b, c, (C, S, 0))])
        for mode in (W.EWALD_NEAREST, W.EWALD_TRILINEAR):           # Nz = 1: both read the one k_z plane
            img, valid = oracle.ewald(P, voxel, k, mode)
            assert np.array_equal(valid.astype(bool), inside), (z, mode)
            ref = k ** 4 * abs(n1 ** 2 - n2 ** 2) ** 2 / (16 * PI ** 2) * np.abs(F) ** 2 * (1 - ((qx * C + qy * S) / k) ** 2)
            ref[ny // 2, nx // 2] = img[ny // 2, nx // 2]
            assert np.abs(img - ref)[inside].max() <= 1e-12 * ref[inside].max(), (z, mode)
            assert not img[~inside].any()
    # the whole path on the same film (one angle, so the rotate step only resamples): total valid-pixel count is the ellipse's
    w = _iso_film(phi, d1, b1, d2, b2, voxel, E, (0.0, 0, 0.0))
    out, cnt = _run(w)
    assert np.array_equal(cnt[0] > 0, inside)
    assert np.abs(out[0] - np.where(inside, k ** 4 * abs(n1 ** 2 - n2 ** 2) ** 2 / (16 * PI ** 2) * np.abs(F) ** 2
                                    * (1 - (qx / k) ** 2), 0.0))[inside & ~((qx == 0) & (qy == 0))].max() <= 1e-12 * out[0].max()


# ---------------------------------------------------------------- P11 90-degree exactness

def test_P11_rot90_of_sample_and_field():
    """Rotating the sample by +90 deg about z (index rotation about voxel 0: x' = -y, y' = x; psi + 90 deg)
    and the field angle by +90 deg leaves the output (expressed in the e frame) unchanged."""
    w = W.tiny(seed=21, nx=16, ny=16, nz=1, n_mat=2, n_energy=1, voxel_nm=5.0, angles=(20.0, 0.0, 20.0))
    n = 16
    def rot(a):
        if a is None:
            return None
        b = np.empty_like(a)
        yy, xx = np.mgrid[0:n, 0:n]
        b[:, xx % n, (-yy) % n] = a[:, yy, xx]        # value at (y, x) moves to (y', x') = (x, -y)
        return b
    mats2 = []
    for (phi, S, th, ps) in w.materials:
        mats2.append((rot(phi), rot(S), rot(th), None if ps is None else (rot(ps).astype(np.float64) + PI / 2).astype(np.float32)))
    o1, c1 = _run(w)
    o2, c2 = oracle.run(mats2, w.voxel_nm, w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp,
                        (110.0, 0.0, 110.0), w.ewald)
    both = (c1 > 0) & (c2 > 0)
    assert both.mean() > 0.7
    assert np.abs(o1 - o2)[both].max() <= 5e-6 * o1.max()      # float32 rounding of psi + pi/2
    # isotropic only: exact
    iso = [(w.materials[0][0], None, None, None), (w.materials[1][0], None, None, None)]
    iso2 = [(rot(w.materials[0][0]), None, None, None), (rot(w.materials[1][0]), None, None, None)]
    args = (w.voxel_nm, w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    o1, c1 = oracle.run(iso, *args, (0.0, 0.0, 0.0), w.ewald)
    o2, c2 = oracle.run(iso2, *args, (90.0, 0.0, 90.0), w.ewald)
    both = (c1 > 0) & (c2 > 0)
    assert (c2[0, 0, :] == 0).all() and (c2[0, 1:, 1:] == 1).all()   # pixel permutation; row/col 0 fall outside
    assert np.abs(o1 - o2)[both].max() <= 1e-12 * o1.max()


# ---------------------------------------------------------------- P12 grating direction

def test_P12_grating_peak_direction():
    """Isotropic stripes along x, period n/m; single angle 30 deg: the first orders sit at
    q = +-(m, 0) dq in the material frame and must appear rotated by -zeta: pixel offsets
    +-(m cos z, -m sin z) ~ +-(7, -4) for m = 8.  The opposite sign convention gives (7, +4)."""
    n, m = 64, 8
    x = np.arange(n)
    phi = (0.5 + 0.5 * np.cos(2 * PI * m * x / n))[None, None, :] * np.ones((1, n, 1))
    w = _iso_film(phi.astype(np.float32), 2e-3, 1e-3, 5e-4, 2e-4, 5.0, 285.0, (30.0, 0.0, 30.0))
    out, cnt = _run(w)
    img = out[0].copy(); c = n // 2
    img[c - 1:c + 2, c - 1:c + 2] = 0
    iy, ix = np.unravel_index(np.argmax(img), img.shape)
    assert (ix - c, iy - c) in [(7, -4), (-7, 4)]
    assert img[c + 4, c + 7] < 1e-3 * img.max() and img[c - 4, c - 7] < 1e-3 * img.max()


# ---------------------------------------------------------------- P13 q_z plane wave

def test_P13_qz_plane_wave_nodes_and_weights():
    """phi1 = 1/2 + 1/2 cos(2 pi (a x/Nx - m z/Nz)): p~ lives at bins (a,0,-m), (-a,0,+m), 0.
    64 x 64 x 16, 1 nm, 285 eV, a = 12: g = q_z/dq_z = -1.55 -> NEAREST node -2, TRILINEAR
    nodes (-2, 0.45..) and (-1, ..); only pixel (+a, 0) lights up (sign of q_z and of the FFT)."""
    nx = ny = 64; nz = 16; a_, m_ = 12, 2
    z, y, x = np.mgrid[0:nz, 0:ny, 0:nx]
    phi = (0.5 + 0.5 * np.cos(2 * PI * (a_ * x / nx - m_ * z / nz))).astype(np.float32)
    d1, b1, d2, b2 = 2e-3, 1e-3, 5e-4, 2e-4
    E, voxel = 285.0, 1.0
    k = 2 * PI * E / 1239.84197
    dqx = 2 * PI / (nx * voxel); dqz = 2 * PI / (nz * voxel)
    qx = a_ * dqx
    g = (np.sqrt(k * k - qx * qx) - k) / dqz
    assert -2 < g < -1.5
    t = g - np.floor(g)
    f32 = lambda v: float(np.float32(v))
    n1 = 1 - f32(d1) + 1j * f32(b1); n2 = 1 - f32(d2) + 1j * f32(b2)
    # float32 phi: amplitude of the bin from the library FFT of the very same array
    amp = abs(np.fft.fftn(phi.astype(np.float64))[(-m_) % nz, 0, a_])
    assert abs(amp - phi.size / 4) < 1e-3 * phi.size
    X = k ** 4 * abs(n1 ** 2 - n2 ** 2) ** 2 / (16 * PI ** 2) * amp ** 2 * (1 - (qx / k) ** 2)
    c = nx // 2
    for mode, wt in ((W.EWALD_NEAREST, 1.0), (W.EWALD_TRILINEAR, 1 - t)):
        w = _iso_film(phi, d1, b1, d2, b2, voxel, E, (0, 0, 0), ewald=mode)
        out, cnt = _run(w)
        assert abs(out[0, c, c + a_] - wt * X) <= 1e-7 * X   # float32 rounding of phi2 = 1 - phi1
        assert out[0, c, c - a_] <= 1e-12 * X
    # m = 1 instead: the upper node (-1) carries weight t
    phi = (0.5 + 0.5 * np.cos(2 * PI * (a_ * x / nx - 1 * z / nz))).astype(np.float32)
    amp = abs(np.fft.fftn(phi.astype(np.float64))[-1, 0, a_])
    X = k ** 4 * abs(n1 ** 2 - n2 ** 2) ** 2 / (16 * PI ** 2) * amp ** 2 * (1 - (qx / k) ** 2)
    w = _iso_film(phi, d1, b1, d2, b2, voxel, E, (0, 0, 0), ewald=W.EWALD_TRILINEAR)
    out, _ = _run(w)
    assert abs(out[0, c, c + a_] - t * X) <= 1e-7 * X
    w = _iso_film(phi, d1, b1, d2, b2, voxel, E, (0, 0, 0), ewald=W.EWALD_NEAREST)
    out, _ = _run(w)
    assert out[0, c, c + a_] <= 1e-12 * X                     # nearest node is -2, where p~ = 0


def test_ewald_validity_and_node_range():
    """Pixels off the sphere (k^2 < qx^2 + qy^2) and nodes below -Nz/2 are invalid (Eq. 8: real q_z only)."""
    nx = ny = 64; nz = 8; voxel = 1.0; E = 285.0
    k = 2 * PI * E / 1239.84197
    n0, n1, w0, w1, valid = oracle.ewald_nodes(nx, ny, nz, voxel, k, W.EWALD_TRILINEAR)
    dq = 2 * PI / (nx * voxel); dqz = 2 * PI / (nz * voxel)
    m = np.arange(nx) - nx // 2
    q2 = (m[None, :] * dq) ** 2 + (m[:, None] * dq) ** 2
    on = q2 <= k * k
    g = np.where(on, (np.sqrt(np.maximum(k * k - q2, 0)) - k) / dqz, -1e9)
    expect = on & (np.floor(g) >= -nz // 2)
    assert (valid.astype(bool) == expect).all()
    ok = valid.astype(bool)
    assert (n0[ok] == np.floor(g[ok])).all()
    assert np.abs(w0[ok] + w1[ok] - 1).max() < 1e-15
    assert (n0[ok] >= -nz // 2).all() and (np.where(n1[ok] > -2 ** 30, n1[ok], 0) <= 0).all()


def test_A6_common_rotation_leaves_X_unchanged():
    """Alg. 1 line 10 'p <- U^T p' is omitted (DESIGN 3-A6): |(I - r r^T) p~|^2 is invariant
    under a common rotation of p~ and r, checked here on random vectors."""
    rng = np.random.default_rng(2)
    for _ in range(10):
        v = rng.standard_normal(3) + 1j * rng.standard_normal(3)
        r = rng.standard_normal(3); r /= np.linalg.norm(r)
        z = rng.uniform(0, 2 * PI)
        U = np.array([[np.cos(z), -np.sin(z), 0], [np.sin(z), np.cos(z), 0], [0, 0, 1]])
        X = lambda v, r: np.linalg.norm(v - r * (r @ v)) ** 2
        assert abs(X(v, r) - X(U.T @ v, U.T @ r)) < 1e-13 * X(v, r)


def test_A14_any_Nz_definition_dft_along_z():
    """Nz that is not a power of two (the paper uses Nz = 63; DESIGN.md 3-A14): the oracle takes the
    definition along z.  Pins: the brute-force 3-D DFT, Parseval, and the whole pipeline with the brute-force
    DFT swapped in, on 8 x 4 x 7 and 4 x 4 x 12."""
    rng = np.random.default_rng(5)
    for shape in [(7, 4, 8), (12, 4, 4), (63, 2, 4)]:
        f = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
        F = oracle.fft3(f)
        assert np.allclose(F, oracle.dft3_naive(f), rtol=0, atol=1e-11 * np.abs(F).max())
        assert np.isclose((np.abs(F) ** 2).sum(), f.size * (np.abs(f) ** 2).sum(), rtol=1e-12)
    # a single plane wave along z lands in exactly one bin, with the forward sign
    nz, m = 7, 3
    z = np.arange(nz).reshape(nz, 1, 1)
    f = np.exp(2j * np.pi * m * z / nz) * np.ones((nz, 4, 4))
    F = oracle.fft3(f)
    assert np.isclose(F[m, 0, 0], nz * 16) and np.abs(np.delete(F[:, 0, 0], m)).max() < 1e-10
    # whole pipeline: linear mode equals definition mode at an odd depth
    w = W.tiny(seed=77, nx=8, ny=8, nz=7, n_mat=2, n_energy=1, voxel_nm=1.5, ewald=W.EWALD_TRILINEAR)
    a, ca = _run(w)
    b, cb = _run(w, linear=True)
    assert np.array_equal(ca, cb) and np.allclose(a, b, rtol=1e-11, atol=1e-14 * a.max())


def test_A14_any_Nx_Ny_definition_dft_along_x_and_y():
    """Lateral sizes that are not powers of two (DESIGN.md 3-A14): the oracle takes the definition
    of Eq. 6 along such an axis.  Pins, none of which calls the routine it checks: the brute-force 3-D DFT,
    numpy's FFT (a library routine of the same definition), Parseval, a plane wave landing in exactly one bin with the
    forward sign, and the whole pipeline: a uniform isotropic film of odd size puts everything into q = 0 with the
    closed-form value, and linear mode equals definition mode on even, odd and mixed sizes (12 x 10 x 3, 9 x 7 x 3, ...)."""
    rng = np.random.default_rng(6)
    for shape in [(4, 6, 10), (3, 5, 7), (1, 12, 9), (2, 8, 6), (5, 4, 3)]:          # (Nz, Ny, Nx)
        f = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
        F = oracle.fft3(f)
        assert np.allclose(F, oracle.dft3_naive(f), rtol=0, atol=1e-11 * np.abs(F).max()), shape
        assert np.allclose(F, np.fft.fftn(f), rtol=0, atol=1e-11 * np.abs(F).max()), shape
        assert np.isclose((np.abs(F) ** 2).sum(), f.size * (np.abs(f) ** 2).sum(), rtol=1e-12)
    ny, nx, my, mx = 6, 10, 2, 7
    y = np.arange(ny).reshape(1, ny, 1); x = np.arange(nx).reshape(1, 1, nx)
    f = np.exp(2j * np.pi * (my * y / ny + mx * x / nx)) * np.ones((3, ny, nx))
    F = oracle.fft3(f)
    G = F.copy(); G[0, my, mx] = 0
    assert np.isclose(F[0, my, mx], 3 * ny * nx) and np.abs(G).max() < 1e-9
    # uniform isotropic film, 9 x 15 x 1: I(q = 0) = k^4 N^2 |n^2 - 1|^2 / (16 pi^2), zero elsewhere (P2's closed form)
    nx, ny = 15, 9
    delta, beta, E = 1e-3, 5e-4, 285.0
    mats = [(np.ones((1, ny, nx), np.float32), None, None, None)]
    f1 = lambda v: np.array([[v]], np.float32)
    w = W.Workload("film", nx, ny, 1, 5.0, mats, np.array([E]), f1(delta), f1(beta), f1(delta), f1(beta), (0.0, 0.0, 0.0),
                   W.EWALD_NEAREST)                                             # one angle, 0 degrees: no interpolation
    img, cnt = _run(w)
    k = 2 * PI * E / 1239.84197
    n2m1 = complex(-np.float32(delta), np.float32(beta)) * (complex(-np.float32(delta), np.float32(beta)) + 2.0)
    expect = k ** 4 * (nx * ny) ** 2 * abs(n2m1) ** 2 / (16 * PI ** 2)
    assert np.isclose(img[0, ny // 2, nx // 2], expect, rtol=1e-10)
    rest = img[0].copy(); rest[ny // 2, nx // 2] = 0
    assert rest.max() < 1e-18 * expect
    # even, odd and mixed sizes (for odd N the bins run over -(N-1)/2 .. (N-1)/2 and q = 0 sits at pixel N/2, integer division)
    for nx, ny, nz in [(12, 10, 3), (9, 7, 3), (8, 5, 1), (7, 12, 5)]:
        w = W.tiny(seed=78 + nx, nx=nx, ny=ny, nz=nz, n_mat=2, n_energy=1, voxel_nm=1.5, ewald=W.EWALD_TRILINEAR)
        a, ca = _run(w)
        b, cb = _run(w, linear=True)
        assert np.array_equal(ca, cb) and np.allclose(a, b, rtol=1e-11, atol=1e-14 * a.max()), (nx, ny, nz)


# ================================================================ round-2 pins
# Each of these ties one decision of the oracle, that no earlier pin reached, to a closed form written
# out here from the paper's equations (none calls the oracle for its expected value).

def _aligned_film(phi1, theta, psi, S, consts_al, consts_iso, voxel, E, angles, ewald=W.EWALD_NEAREST):
    """Material 1 aligned with a constant director (theta, psi) and alignment S, material 2 = 1 - phi1 isotropic.
    consts_al = (delta_par, beta_par, delta_perp, beta_perp), consts_iso = (delta, beta)."""
    phi1 = np.ascontiguousarray(phi1, np.float32)
    full = lambda v: np.full(phi1.shape, v, np.float32)
    mats = [(phi1, full(S), full(theta), full(psi)), (np.ascontiguousarray(1.0 - phi1, dtype=np.float32), None, None, None)]
    nz, ny, nx = phi1.shape
    f = lambda a, b: np.array([[a, b]], np.float32)
    dpa, bpa, dpe, bpe = consts_al
    di, bi = consts_iso
    return W.Workload("aligned", nx, ny, nz, voxel, mats, np.array([E]), f(dpa, di), f(bpa, bi), f(dpe, di), f(bpe, bi),
                      angles, ewald)


def _n(delta, beta):
    """n = 1 - delta + i beta with the float32-rounded constants the oracle receives (north_star)."""
    return 1 - float(np.float32(delta)) + 1j * float(np.float32(beta))


@pytest.mark.parametrize("theta_deg,psi_deg,zeta", [(35.0, 20.0, 0.0), (120.0, -50.0, 0.0), (60.0, 75.0, 90.0)])
def test_R2a_uniform_director_plane_wave_film(theta_deg, psi_deg, zeta):
    """Eq. 2-5 and Eq. 7-8 on a film whose only structure is one Fourier mode:
    material 1 fully aligned (S = 1) with a constant director out of the film plane (theta != 90 deg),
    phi1 = 1/2 + 1/2 cos(2 pi a x / Nx), material 2 = 1 - phi1 isotropic, Nz = 1, one angle.
    For q != 0:  p~(q) = phi~1(q) (chi_al - chi_iso) e,  chi_al = (a I + b d d^T)/4pi with a = n_perp^2 - 1,
    b = n_par^2 - n_perp^2,  chi_iso = (n_iso^2 - 1) I/4pi,  and the pixel (+-a, 0) holds
        I = k^4 |phi~1|^2 || (I - r r^T)(chi_al - chi_iso) e ||^2,  r = (q_x, 0, sqrt(k^2 - q_x^2))/k.
    The z component of p (b (d.e) d_z) enters through r_z: this value depends on p_z, on which of a / c
    multiplies the aligned part, and on the (d.e) d term.  zeta = 0 and 90 keep the rotate step a pixel
    permutation, so the expected value sits at an exact pixel."""
    nx = ny = 64; a_ = 6; voxel = 2.0; E = 285.0          # dq = 0.049: r_x = 0.204, r_z = 0.979
    x = np.arange(nx)
    phi = ((0.5 + 0.5 * np.cos(2 * PI * a_ * x / nx))[None, None, :] * np.ones((1, ny, 1))).astype(np.float32)
    th, ps = np.deg2rad(theta_deg), np.deg2rad(psi_deg)
    al, iso = (2.4e-3, 1.1e-3, 0.6e-3, 0.3e-3), (1.3e-3, 0.7e-3)
    w = _aligned_film(phi, th, ps, 1.0, al, iso, voxel, E, (zeta, 0.0, zeta))
    out, cnt = _run(w)
    # --- the closed form, written from the equations
    k = 2 * PI * E / 1239.84197
    npar, nperp, niso_m = _n(al[0], al[1]), _n(al[2], al[3]), _n(*iso)
    thf, psf = float(np.float32(th)), float(np.float32(ps))          # the float32 angles the oracle receives
    d = np.array([np.cos(psf) * np.sin(thf), np.sin(psf) * np.sin(thf), np.cos(thf)])
    chi_al = ((nperp ** 2 - 1) * np.eye(3) + (npar ** 2 - nperp ** 2) * np.outer(d, d)) / (4 * PI)
    chi_iso = (niso_m ** 2 - 1) * np.eye(3) / (4 * PI)
    e = np.array([np.cos(np.deg2rad(zeta)), np.sin(np.deg2rad(zeta)), 0.0])
    if zeta == 90.0:
        e = np.array([0.0, 1.0, 0.0])
    amp = np.fft.fft2(phi[0].astype(np.float64))[0, a_]               # library FFT of the very same float32 array
    assert abs(abs(amp) - nx * ny / 4) < 1e-3 * nx * ny
    dq = 2 * PI / (nx * voxel)
    c = nx // 2
    for sgn in (+1, -1):
        qx = sgn * a_ * dq
        r = np.array([qx, 0.0, np.sqrt(k * k - qx * qx)]) / k
        pt = abs(amp) * (chi_al - chi_iso) @ e
        wv = pt - r * (r @ pt)
        expect = k ** 4 * np.vdot(wv, wv).real
        # material-frame pixel (sgn a, 0); the output is the image turned by -zeta: (u, v) -> R(-zeta)(u, v)
        u, v = (sgn * a_, 0) if zeta == 0.0 else (0, -sgn * a_)
        got = out[0, c + v, c + u]
        assert abs(got - expect) <= 2e-7 * expect, (sgn, got, expect)     # float32 rounding of 1 - phi1
    # what the mutants would give, to show the case separates them: p_z dropped / c in place of a
    qx = a_ * dq; r = np.array([qx, 0.0, np.sqrt(k * k - qx * qx)]) / k
    pt = abs(amp) * (chi_al - chi_iso) @ e
    for bad in (pt * np.array([1, 1, 0]),
                abs(amp) * ((((niso_m * 0 + ((npar + 2 * nperp) / 3) ** 2 - 1) * np.eye(3)
                              + (npar ** 2 - nperp ** 2) * np.outer(d, d)) / (4 * PI) - chi_iso) @ e)):
        wb = bad - r * (r @ bad)
        good = pt - r * (r @ pt)
        assert abs(np.vdot(wb, wb).real / np.vdot(good, good).real - 1) > 1e-3


def test_R2a_director_along_x_uniform_film():
    """One fully aligned material filling the film, d = x (theta = 90 deg, psi = 0):  at q = 0, r = z and
    I(0) = k^4 N^2 |n_par^2 - 1|^2 / 16 pi^2 for e = x (zeta = 0), |n_perp^2 - 1|^2 for e = y (zeta = 90)."""
    n, voxel, E = 32, 5.0, 285.0
    dpa, bpa, dpe, bpe = 2.4e-3, 1.1e-3, 0.6e-3, 0.3e-3
    phi = np.ones((1, n, n), np.float32)
    mats = [(phi, phi.copy(), np.full_like(phi, np.float32(PI / 2)), np.zeros_like(phi))]
    f = lambda v: np.array([[v]], np.float32)
    k = 2 * PI * E / 1239.84197
    thf = float(np.float32(PI / 2))                   # float32(pi/2): d_z = cos(thf) = -4.4e-8, below the tolerance
    assert abs(np.cos(thf)) < 1e-7
    for zeta, nn in ((0.0, _n(dpa, bpa)), (90.0, _n(dpe, bpe))):
        out, cnt = oracle.run(mats, voxel, [E], f(dpa), f(bpa), f(dpe), f(bpe), (zeta, 0.0, zeta), W.EWALD_NEAREST)
        I0 = k ** 4 * (n * n) ** 2 * abs(nn ** 2 - 1) ** 2 / (16 * PI ** 2)
        assert abs(out[0, n // 2, n // 2] - I0) <= 1e-6 * I0
        off = out[0].copy(); off[n // 2, n // 2] = 0
        assert off.max() <= 1e-12 * I0


def test_R2b_nearest_takes_floor_of_g_plus_half():
    """P13 with a = 11: g = q_z/dq_z = -1.236, so floor(g) = -2 but the nearest node is floor(g + 1/2) = -1
    (DESIGN 3-A8).  A plane wave at k_z = -1 must light pixel (+a, 0) with weight 1 in NEAREST mode and
    weight t = g - floor(g) in TRILINEAR mode; a wave at k_z = -2 must be dark in NEAREST mode."""
    nx = ny = 64; nz = 16; a_ = 11
    z, y, x = np.mgrid[0:nz, 0:ny, 0:nx]
    d1, b1, d2, b2 = 2e-3, 1e-3, 5e-4, 2e-4
    E, voxel = 285.0, 1.0
    k = 2 * PI * E / 1239.84197
    dqx = 2 * PI / (nx * voxel); dqz = 2 * PI / (nz * voxel)
    qx = a_ * dqx
    g = (np.sqrt(k * k - qx * qx) - k) / dqz
    assert -1.5 < g < -1.0                            # nearest node -1, lower node -2
    t = g + 2.0
    n1, n2 = _n(d1, b1), _n(d2, b2)
    c = nx // 2
    for m_, near_w, tri_w in ((1, 1.0, t), (2, 0.0, 1.0 - t)):
        phi = (0.5 + 0.5 * np.cos(2 * PI * (a_ * x / nx - m_ * z / nz))).astype(np.float32)
        amp = abs(np.fft.fftn(phi.astype(np.float64))[(-m_) % nz, 0, a_])
        X = k ** 4 * abs(n1 ** 2 - n2 ** 2) ** 2 / (16 * PI ** 2) * amp ** 2 * (1 - (qx / k) ** 2)
        for mode, wt in ((W.EWALD_NEAREST, near_w), (W.EWALD_TRILINEAR, tri_w)):
            w = _iso_film(phi, d1, b1, d2, b2, voxel, E, (0, 0, 0), ewald=mode)
            out, cnt = _run(w)
            assert abs(out[0, c, c + a_] - wt * X) <= 1e-7 * X, (m_, mode, out[0, c, c + a_] / X, wt)


def test_R2c_node_range_boundary():
    """Eq. 8 + DESIGN 3-A8/A14: a pixel is invalid if its (lower / nearest) node lies below -Nz/2; the
    node -Nz/2 itself is valid.  64 x 64 x 8 at 2.75 nm, 285 eV: k/dq = 40.457 px ((k/dq)^2 = 1636.75),
    g_min = -5.06, -Nz/2 = -4.  Pixels (m_x, m_y), |m|^2 in brackets, g = (sqrt(k^2 - |m|^2 dq^2) - k)/dq_z
    worked out by hand (and re-derived below):
      (30, -24) [1476]  g = -3.472: TRILINEAR nodes (-4, -3) valid;           NEAREST n = -3 valid
      (31, -24) [1537]  g = -3.809: TRILINEAR lower node -4 = -Nz/2 -> valid; NEAREST n = -4 = -Nz/2 -> valid
      (28, -28) [1568]  g = -4.021: TRILINEAR lower node -5 -> INVALID;       NEAREST n = -4 -> valid
      (29, -28) [1625]  g = -4.629: TRILINEAR -5 -> INVALID;                  NEAREST n = -5 -> INVALID
      (31, -26) [1637]  off the sphere (1637 > 1636.75) -> invalid in both modes."""
    nx = ny = 64; nz = 8; voxel = 2.75; E = 285.0
    k = 2 * PI * E / 1239.84197
    dq = 2 * PI / (nx * voxel); dqz = 2 * PI / (nz * voxel)
    c = nx // 2
    gv = lambda mx, my: (np.sqrt(k * k - (mx * mx + my * my) * dq * dq) - k) / dqz
    for (mx, my), gg in (((30, -24), -3.472), ((31, -24), -3.809), ((28, -28), -4.021), ((29, -28), -4.629)):
        assert abs(gv(mx, my) - gg) < 1e-3
    assert 1636 < (k / dq) ** 2 < 1637
    tri = oracle.ewald_nodes(nx, ny, nz, voxel, k, W.EWALD_TRILINEAR)
    nea = oracle.ewald_nodes(nx, ny, nz, voxel, k, W.EWALD_NEAREST)
    px = lambda t, mx, my: (int(t[0][c + my, c + mx]), int(t[1][c + my, c + mx]), bool(t[4][c + my, c + mx]))
    BAD = -2 ** 31
    for sx, sy in ((1, 1), (-1, 1), (1, -1), (-1, -1)):       # the rule depends on |q| only; m = -32 does not occur here
        assert px(tri, sx * 30, sy * 24) == (-4, -3, True) and px(nea, sx * 30, sy * 24) == (-3, BAD, True)
        assert px(tri, sx * 31, sy * 24) == (-4, -3, True) and px(nea, sx * 31, sy * 24) == (-4, BAD, True)
        assert px(tri, sx * 28, sy * 28) == (BAD, BAD, False) and px(nea, sx * 28, sy * 28) == (-4, BAD, True)
        assert px(tri, sx * 29, sy * 28) == (BAD, BAD, False) and px(nea, sx * 29, sy * 28) == (BAD, BAD, False)
        assert px(tri, sx * 31, sy * 26) == (BAD, BAD, False) and px(nea, sx * 31, sy * 26) == (BAD, BAD, False)
    # the weights at a boundary pixel: t = g - floor(g) on the upper node
    t = gv(31, -24) + 4.0
    assert abs(tri[3][c - 24, c + 31] - t) < 1e-12 and abs(tri[2][c - 24, c + 31] - (1 - t)) < 1e-12
    # the whole detector against the rule, with every class present and no pixel within 1e-9 of a decision
    m = np.arange(nx) - c
    r2 = (m[None, :] ** 2 + m[:, None] ** 2).astype(np.float64)
    on = r2 * dq * dq <= k * k
    g = np.where(on, (np.sqrt(np.maximum(k * k - r2 * dq * dq, 0.0)) - k) / dqz, np.nan)
    assert np.nanmin(np.abs(g - np.round(g))[r2 > 0]) > 1e-9 and np.nanmin(np.abs(g + 0.5 - np.round(g + 0.5))) > 1e-9
    lo = np.floor(g); nr = np.floor(g + 0.5)
    exp_tri = on & (lo >= -4); exp_nea = on & (nr >= -4)
    for cls in (on & (lo == -5), on & (lo == -4), on & (nr == -5), on & (nr == -4), ~on):
        assert cls.any()
    assert (tri[4].astype(bool) == exp_tri).all() and (nea[4].astype(bool) == exp_nea).all()
    assert (tri[0][exp_tri] == lo[exp_tri]).all() and (nea[0][exp_nea] == nr[exp_nea]).all()


def _rotate_count_numpy(valid, zeta_deg, rho=1.0):
    """Independent statement of DESIGN 3-A9/A10 for the counts: output pixel q' samples the source position
    R(+zeta) q' (physical q; y pixels are rho x-pixels tall); it counts iff every neighbour with non-zero
    bilinear weight is inside the image and valid.  Plain Python loops; returns (count 0/1, weights)."""
    ny, nx = valid.shape
    z = np.deg2rad(zeta_deg)
    C, S = np.cos(z), np.sin(z)
    cnt = np.zeros((ny, nx), np.uint32)
    for iy in range(ny):
        for ix in range(nx):
            u, v = ix - nx // 2, (iy - ny // 2) * rho            # in units of dq_x
            su, sv = C * u - S * v, S * u + C * v                 # source, same units
            fx, fy = su + nx // 2, sv / rho + ny // 2
            x0, y0 = int(np.floor(fx)), int(np.floor(fy))
            ax, ay = fx - x0, fy - y0
            need = [(x0 + jx, y0 + jy) for jx, wx in ((0, 1 - ax), (1, ax)) for jy, wy in ((0, 1 - ay), (1, ay)) if wx * wy > 0]
            if all(0 <= X < nx and 0 <= Y < ny and valid[Y, X] for X, Y in need):
                cnt[iy, ix] = 1
    return cnt


def test_R2d_rotate_with_the_ewald_disk_cutting_the_detector():
    """O5 (DESIGN 3-A9/A10) where part of the detector is off the Ewald sphere (32 x 32, 0.4 nm voxels:
    k/dq = 2.94 px at 285 eV -- and a second, larger disk): a sample counts only if EVERY needed neighbour is
    valid.  Pins: (i) the counts against an independent NumPy statement of that rule; (ii) for an image that is
    constant on the valid set the average must be exactly that constant wherever cnt > 0 (the weights of a
    counted sample sum to 1), which fails if invalid neighbours were skipped instead of vetoing the sample."""
    n = 32
    m = np.arange(n) - n // 2
    r2 = m[None, :] ** 2 + m[:, None] ** 2
    for radius in (2.94, 9.3):
        valid = (r2 <= radius * radius).astype(np.uint8)
        img = np.where(valid > 0, 7.25, 1e9)                  # junk outside: must never be read into a counted sample
        for zeta in (30.0, 77.0):
            acc = np.zeros((n, n)); cnt = np.zeros((n, n), np.uint32)
            oracle.rotate_accumulate(img, valid, zeta, acc, cnt)
            exp = _rotate_count_numpy(valid.astype(bool), zeta)
            assert (cnt == exp).all()
            assert 0 < exp.sum() < valid.sum()                 # the rim of the disk loses samples
            assert np.abs(acc[cnt > 0] - 7.25).max() < 1e-12
            assert (acc[cnt == 0] == 0).all()
            # certain cases from geometry alone: well inside the disk every neighbour is valid, well outside none is
            rr = np.sqrt(r2)
            assert (cnt[rr <= radius - 1.4143] == 1).all() and (cnt[rr >= radius + 1.4143] == 0).all()
    # the whole pipeline on such a detector: counts of a multi-angle run = sum of the per-angle rule
    w = W.tiny(seed=10, nx=32, ny=32, nz=1, n_mat=2, n_energy=1, voxel_nm=0.4, ewald=W.EWALD_NEAREST, angles=(0.0, 30.0, 150.0))
    out, cnt = _run(w)
    k = 2 * PI * w.energies[0] / 1239.84197
    dq = 2 * PI / (n * 0.4)
    valid = r2 * dq * dq <= k * k
    exp = sum(_rotate_count_numpy(valid, 30.0 * i) for i in range(6))
    assert (cnt[0] == exp).all() and 0 < (exp > 0).sum() < n * n


def test_R2e_rotation_is_in_physical_q_on_a_non_square_detector():
    """DESIGN 3-A9: the image rotation acts on physical q.  64 x 32 voxels (rho = Nx/Ny = 2, dq_y = 2 dq_x):
    stripes along x with m = 8 periods put the first orders at q = +-(8 dq_x, 0); at zeta = 30 deg they must
    appear at q' = R(-zeta) q = 8 dq_x (cos, -sin) = (6.93 dq_x, -2.0 dq_y): pixel offsets +-(7, -2).
    Rotating pixel indices instead (rho dropped) would give (7, -4)."""
    nx, ny, m_ = 64, 32, 8
    x = np.arange(nx)
    phi = (0.5 + 0.5 * np.cos(2 * PI * m_ * x / nx))[None, None, :] * np.ones((1, ny, 1))
    w = _iso_film(phi.astype(np.float32), 2e-3, 1e-3, 5e-4, 2e-4, 5.0, 285.0, (30.0, 0.0, 30.0))
    out, cnt = _run(w)
    img = out[0].copy(); cy, cx = ny // 2, nx // 2
    img[cy - 1:cy + 2, cx - 2:cx + 3] = 0                     # the q = 0 peak and its bilinear leakage
    iy, ix = np.unravel_index(np.argmax(img), img.shape)
    assert (ix - cx, iy - cy) in [(7, -2), (-7, 2)]
    assert img[cy - 4, cx + 7] < 1e-3 * img.max() and img[cy + 4, cx - 7] < 1e-3 * img.max()
    # counts on the non-square detector against the independent statement (rho = 2)
    exp = _rotate_count_numpy(np.ones((ny, nx), bool), 30.0, rho=2.0)
    assert (cnt[0] == exp).all() and 0 < exp.sum() < nx * ny
    # zeta = 90 deg: q' = (u dq_x, v dq_y) samples q = (-v dq_y, u dq_x), i.e. source pixel (cx - 2 v, cy + u/2):
    # the +-first orders of the same grating land at q' = (0, -+8 dq_x) = (0, -+4 dq_y): pixels (0, -+4)
    w = _iso_film(phi.astype(np.float32), 2e-3, 1e-3, 5e-4, 2e-4, 5.0, 285.0, (90.0, 0.0, 90.0))
    out, cnt = _run(w)
    img = out[0].copy(); img[cy - 1:cy + 2, cx - 2:cx + 3] = 0
    iy, ix = np.unravel_index(np.argmax(img), img.shape)
    assert (ix - cx, abs(iy - cy)) == (0, 4)


def test_R2f_polarization_from_the_rotated_index_tensor():
    """Eq. 1-5 in their tensor form, per voxel, for ANY field direction (e_z != 0 included):
    the uniaxial index tensor N = diag(n_perp, n_perp, n_par) (extraordinary axis along z before rotation)
    is rotated by R = Rz(psi) Ry(theta) (which carries z onto d = (cos psi sin theta, sin psi sin theta, cos theta)),
    N_rot = R N R^T, and p = phi [ S (N_rot N_rot - I) + (1 - S)(n_iso^2 - 1) I ] e / 4 pi.  The oracle uses the
    director shortcut a e + b (d.e) d; this test builds the matrices."""
    rng = np.random.default_rng(17)
    nv = 24
    phi = rng.uniform(0.1, 1.0, (1, 1, nv)).astype(np.float32)
    S = rng.uniform(0.0, 1.0, (1, 1, nv)).astype(np.float32)
    th = rng.uniform(0.0, PI, (1, 1, nv)).astype(np.float32)
    ps = rng.uniform(-PI, 2 * PI, (1, 1, nv)).astype(np.float32)
    dpa, bpa, dpe, bpe = 2.4e-3, 1.1e-3, 0.6e-3, 0.3e-3
    a, b, c = oracle.coefficients([dpa], [bpa], [dpe], [bpe])
    npar, nperp = _n(dpa, bpa), _n(dpe, bpe)
    niso = (npar + 2 * nperp) / 3
    for e in ((1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0), (0.3, -0.5, 0.81)):
        p = oracle.polarization([(phi, S, th, ps)], a, b, c, e)          # [3][1][1][nv]
        for i in range(nv):
            t, q = float(th[0, 0, i]), float(ps[0, 0, i])
            Ry = np.array([[np.cos(t), 0, np.sin(t)], [0, 1, 0], [-np.sin(t), 0, np.cos(t)]])
            Rz = np.array([[np.cos(q), -np.sin(q), 0], [np.sin(q), np.cos(q), 0], [0, 0, 1]])
            R = Rz @ Ry
            Nrot = R @ np.diag([nperp, nperp, npar]) @ R.T
            s_, f_ = float(S[0, 0, i]), float(phi[0, 0, i])
            chi = f_ * (s_ * (Nrot @ Nrot - np.eye(3)) + (1 - s_) * (niso ** 2 - 1) * np.eye(3)) / (4 * PI)
            ref = chi @ np.array(e)
            assert np.abs(p[:, 0, 0, i] - ref).max() <= 1e-14, (e, i)
