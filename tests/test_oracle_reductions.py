"""Pins for the oracle's NEXT-1 reductions (I(|q|), anisotropy A, ISI):
closed forms, symmetries, the paper's Eq. 10 energy law and form-factor zeros -- nothing here
re-types the oracle's loop."""
import numpy as np

import oracle
from paper_2209_13121_b200 import workloads as W
from tests.parity import oracle_run


def test_constant_image_closed_forms():
    Ny, Nx, vox = 32, 64, 2.0
    img = np.full((Ny, Nx), 3.5)
    I, A, npix, isi = oracle.reductions(img, None, vox, 16)
    assert np.allclose(I, 3.5) and np.all(A == 0.0)
    dq = (2 * np.pi / (Nx * vox)) * (2 * np.pi / (Ny * vox))
    assert np.isclose(isi, 3.5 * Nx * Ny * dq, rtol=1e-14)
    # number of lattice points at rounded radius b on the (u, 2v) lattice: brute force with numpy
    u = np.arange(Nx) - Nx // 2
    v = (np.arange(Ny) - Ny // 2) * (Nx / Ny)
    r = np.floor(np.hypot(u[None, :], v[:, None]) + 0.5).astype(int)
    assert np.array_equal(npix, np.bincount(r.ravel(), minlength=16)[:16])
    assert npix[0] == 1


def test_masked_pixels_do_not_take_part():
    rng = np.random.default_rng(0)
    img = rng.uniform(1, 2, (32, 32))
    cnt = (rng.uniform(size=(32, 32)) > 0.3).astype(np.uint32)
    I, A, npix, isi = oracle.reductions(img, cnt, 1.0, 12)
    I2, A2, npix2, isi2 = oracle.reductions(np.where(cnt > 0, img, 1e30), cnt, 1.0, 12)
    assert np.array_equal(I, I2) and np.array_equal(A, A2) and isi == isi2
    dq2 = (2 * np.pi / 32) ** 2
    assert np.isclose(isi, img[cnt > 0].sum() * dq2, rtol=1e-13)


def test_anisotropy_symmetries_and_cos2_law():
    n = 128
    y, x = np.mgrid[0:n, 0:n] - n // 2
    chi = np.arctan2(y, x)
    base = 1.0 / (1.0 + 0.01 * (x * x + y * y))
    img = base * (1.0 + 0.6 * np.cos(2 * chi))
    I, A, npix, _ = oracle.reductions(img, None, 1.0, 48, 10.0)
    # x <-> y swap (transpose) flips the sign of A exactly; a swap-symmetric image has A = 0
    _, At, _, _ = oracle.reductions(img.T.copy(), None, 1.0, 48, 10.0)
    assert np.allclose(A[2:], -At[2:], atol=1e-14)
    _, As, _, _ = oracle.reductions(base, None, 1.0, 48, 10.0)
    assert np.allclose(As, 0.0, atol=1e-14)
    # I = f(r) (1 + a cos 2chi): sector means over |chi| <= w give A = a sinc(2w) to discretisation
    w = np.deg2rad(10.0)
    expect = 0.6 * np.sin(2 * w) / (2 * w)
    assert np.allclose(A[12:], expect, atol=0.02)
    # and the azimuthal mean removes the cos 2chi term
    rr = np.arange(48.0)
    assert np.allclose(I[12:], 1.0 / (1.0 + 0.01 * rr[12:] ** 2), rtol=0.03)


def test_isi_energy_law_eq10_and_disk_profile():
    """2-D binary isotropic film (a disk): ISI(E) ~ |n1^2 - n2^2|^2 E^4 ~ 4 (dd^2 + db^2) E^4
    (Eq. 10), and I(|q|) has the flat-disk zero at qR = 3.8317."""
    n, R, vox = 256, 20.0, 5.0
    y, x = np.mgrid[0:n, 0:n] - n // 2
    phi1 = ((x * x + y * y) <= R * R).astype(np.float32).reshape(1, n, n)
    mats = [(phi1, None, None, None), ((1 - phi1).astype(np.float32), None, None, None)]
    E = np.array([270.0, 285.0, 300.0])
    d = np.array([[2e-3, 1e-3], [3e-3, 5e-4], [1e-3, 1.5e-3]], np.float32)
    b = np.array([[1e-3, 5e-4], [2e-4, 1e-3], [8e-4, 2e-4]], np.float32)
    w = W.Workload("disk", n, n, 1, vox, mats, E, d, b, d, b, (0.0, 0.0, 0.0), W.EWALD_NEAREST)
    out, cnt = oracle_run(w)
    isi, prof = [], []
    for e in range(3):
        o = out[e].copy()
        o[n // 2, n // 2] = 0.0                       # Eq. 10 is about q != 0
        I, A, npix, s = oracle.reductions(o, cnt[e], vox, 100)
        isi.append(s); prof.append(I)
    law = ((d[:, 0] - d[:, 1]).astype(np.float64) ** 2 + (b[:, 0] - b[:, 1]).astype(np.float64) ** 2) * E ** 4
    r = np.array(isi) / law
    assert np.allclose(r / r[0], 1.0, rtol=0.02), r / r[0]
    # first zero of [2 J1(qR)/(qR)]^2: qR = 3.8317 -> bin 3.8317 / (R vox dq), dq = 2 pi / (n vox)
    b0 = 3.8317 / (R * vox * 2 * np.pi / (n * vox))
    k = int(np.argmin(prof[1][3:12])) + 3
    assert abs(k - b0) <= 1.0, (k, b0)
