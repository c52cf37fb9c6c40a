"""CPU oracle for the CyRSoXS hot path -- TEST INFRASTRUCTURE, not product code.

Thin ctypes wrapper around ``cyrsoxs_oracle.c`` (plain C, double precision, written
from PAPER.md; see that file's header for the passage each function follows).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s CPU-baseline legs may import
this package; ``paper_2209_13121_b200`` never does, and this package never imports it.

Arrays are C-order ``[Nz][Ny][Nx]`` (x fastest, SURVEY 8 / DESIGN.md 4).  A material is
a tuple ``(phi, S, theta, psi)`` of float32 arrays; ``S, theta, psi`` may be ``None``
for an isotropic material.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "cyrsoxs_oracle.c"
_LIB = _HERE / "libcyrsoxs_oracle.so"

EWALD_NEAREST = 0
EWALD_TRILINEAR = 1


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc.  -ffp-contract=off: every geometry operation is
    rounded on its own (DESIGN.md 3-A11)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".{os.getpid()}.tmp")
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
             "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(str(_LIB))
        _lib.orc_wavenumber.restype = C.c_double
        _lib.orc_wavenumber.argtypes = [C.c_double]
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_num_angles.restype = C.c_int
        _lib.orc_num_angles.argtypes = [C.c_double] * 3
        _lib.orc_fft3.restype = C.c_int
        _lib.orc_run_energy.restype = C.c_int
        _lib.orc_run_energy_linear.restype = C.c_int
    return _lib


def num_threads() -> int:
    return int(lib().orc_num_threads())


def _p(a, ctype=C.c_void_p):
    return a.ctypes.data_as(ctype) if a is not None else None


class _Morph:
    """Keeps the float32 arrays alive and exposes the four const float* const* tables."""

    def __init__(self, materials):
        self.n_mat = len(materials)
        self.keep = []
        tabs = []
        shape = None
        for k in range(4):
            arr = (C.c_void_p * self.n_mat)()
            for m, mat in enumerate(materials):
                a = mat[k]
                if a is None:
                    if k == 0:
                        raise ValueError("phi must not be None")
                    arr[m] = None
                    continue
                a = np.ascontiguousarray(a, dtype=np.float32)
                if shape is None:
                    shape = a.shape
                if a.shape != shape:
                    raise ValueError("morphology arrays differ in shape")
                self.keep.append(a)
                arr[m] = a.ctypes.data
            tabs.append(arr)
        self.phi, self.S, self.theta, self.psi = tabs
        if len(shape) != 3:
            raise ValueError("morphology arrays must be [Nz][Ny][Nx]")
        self.Nz, self.Ny, self.Nx = (int(s) for s in shape)
        self.n_vox = self.Nx * self.Ny * self.Nz


def _f32(x, n):
    a = np.ascontiguousarray(x, dtype=np.float32).reshape(-1)
    if a.size != n:
        raise ValueError("optical constants: wrong length")
    return a


def wavenumber(energy_eV: float) -> float:
    return float(lib().orc_wavenumber(float(energy_eV)))


def coefficients(delta_par, beta_par, delta_perp, beta_perp):
    """O0: per-material complex a = n_perp^2-1, b = n_par^2-n_perp^2, c = n_iso^2-1."""
    n = len(delta_par)
    a = np.empty(n, np.complex128); b = np.empty(n, np.complex128); c = np.empty(n, np.complex128)
    lib().orc_coefficients(C.c_int(n), _p(_f32(delta_par, n)), _p(_f32(beta_par, n)),
                           _p(_f32(delta_perp, n)), _p(_f32(beta_perp, n)), _p(a), _p(b), _p(c))
    return a, b, c


def polarization(materials, a, b, c, e):
    """O2: p[3][Nz][Ny][Nx] complex128 for field direction e = (ex, ey, ez)."""
    M = _Morph(materials)
    a = np.ascontiguousarray(a, np.complex128); b = np.ascontiguousarray(b, np.complex128)
    c = np.ascontiguousarray(c, np.complex128)
    p = np.empty((3, M.Nz, M.Ny, M.Nx), np.complex128)
    lib().orc_polarization(C.c_int64(M.n_vox), C.c_int(M.n_mat), M.phi, M.S, M.theta, M.psi,
                           _p(a), _p(b), _p(c), C.c_double(e[0]), C.c_double(e[1]), C.c_double(e[2]),
                           _p(p[0]), _p(p[1]), _p(p[2]))
    return p


def fft3(f):
    """O3: forward unnormalised 3-D FFT (own radix-2) of f[Nz][Ny][Nx]; returns a new array."""
    g = np.array(f, dtype=np.complex128, order="C", copy=True)
    Nz, Ny, Nx = g.shape
    rc = lib().orc_fft3(C.c_int(Nx), C.c_int(Ny), C.c_int(Nz), _p(g))
    if rc != 0:
        raise ValueError("sizes must be powers of two")
    return g


def dft3_naive(f):
    """Eq. 6 written out, O(N^2)."""
    g = np.ascontiguousarray(f, dtype=np.complex128)
    Nz, Ny, Nx = g.shape
    out = np.empty_like(g)
    lib().orc_dft3_naive(C.c_int(Nx), C.c_int(Ny), C.c_int(Nz), _p(g), _p(out))
    return out


def polarization_dft_bins(materials, a, b, c, e, bins):
    """p~ at the listed (kx, ky, kz) bins by direct summation over all voxels."""
    M = _Morph(materials)
    a = np.ascontiguousarray(a, np.complex128); b = np.ascontiguousarray(b, np.complex128)
    c = np.ascontiguousarray(c, np.complex128)
    bins = np.ascontiguousarray(bins, dtype=np.int32).reshape(-1, 3)
    out = np.empty((bins.shape[0], 3), np.complex128)
    lib().orc_polarization_dft_bins(
        C.c_int(M.Nx), C.c_int(M.Ny), C.c_int(M.Nz), C.c_int(M.n_mat), M.phi, M.S, M.theta, M.psi,
        _p(a), _p(b), _p(c), C.c_double(e[0]), C.c_double(e[1]), C.c_double(e[2]),
        C.c_int(bins.shape[0]), _p(bins), _p(out))
    return out


def ewald(P, voxel_nm, k, mode):
    """O4: detector image of one angle from p~ = P[3][Nz][Ny][Nx]; returns (img, valid)."""
    P = np.ascontiguousarray(P, np.complex128)
    _, Nz, Ny, Nx = P.shape
    img = np.empty((Ny, Nx), np.float64); valid = np.empty((Ny, Nx), np.uint8)
    lib().orc_ewald(C.c_int(Nx), C.c_int(Ny), C.c_int(Nz), C.c_double(voxel_nm), C.c_double(k),
                    C.c_int(mode), _p(P[0]), _p(P[1]), _p(P[2]), _p(img), _p(valid))
    return img, valid


def ewald_linear(Px, Py, voxel_nm, k, mode):
    """Linear mode images (Ixx, Iyy, Ixy, valid) from p~ for e=x (Px[3]) and e=y (Py[3])."""
    Px = np.ascontiguousarray(Px, np.complex128); Py = np.ascontiguousarray(Py, np.complex128)
    _, Nz, Ny, Nx = Px.shape
    Ixx = np.empty((Ny, Nx)); Iyy = np.empty((Ny, Nx)); Ixy = np.empty((Ny, Nx))
    valid = np.empty((Ny, Nx), np.uint8)
    lib().orc_ewald_linear(C.c_int(Nx), C.c_int(Ny), C.c_int(Nz), C.c_double(voxel_nm), C.c_double(k),
                           C.c_int(mode), _p(Px[0]), _p(Px[1]), _p(Px[2]), _p(Py[0]), _p(Py[1]), _p(Py[2]),
                           _p(Ixx), _p(Iyy), _p(Ixy), _p(valid))
    return Ixx, Iyy, Ixy, valid


def ewald_nodes(Nx, Ny, Nz, voxel_nm, k, mode):
    n0 = np.empty((Ny, Nx), np.int32); n1 = np.empty((Ny, Nx), np.int32)
    w0 = np.empty((Ny, Nx)); w1 = np.empty((Ny, Nx)); valid = np.empty((Ny, Nx), np.uint8)
    lib().orc_ewald_nodes(C.c_int(Nx), C.c_int(Ny), C.c_int(Nz), C.c_double(voxel_nm), C.c_double(k),
                          C.c_int(mode), _p(n0), _p(n1), _p(w0), _p(w1), _p(valid))
    return n0, n1, w0, w1, valid


def angle_cs(zeta_deg):
    c = C.c_double(); s = C.c_double()
    lib().orc_angle_cs(C.c_double(zeta_deg), C.byref(c), C.byref(s))
    return c.value, s.value


def num_angles(start, step, end) -> int:
    return int(lib().orc_num_angles(float(start), float(step), float(end)))


def rotate_accumulate(img, valid, zeta_deg, acc_sum, acc_cnt):
    """O5: adds one angle's rotated-back image into (acc_sum float64, acc_cnt uint32)."""
    img = np.ascontiguousarray(img, np.float64); valid = np.ascontiguousarray(valid, np.uint8)
    Ny, Nx = img.shape
    assert acc_sum.dtype == np.float64 and acc_cnt.dtype == np.uint32
    assert acc_sum.flags.c_contiguous and acc_cnt.flags.c_contiguous
    c, s = angle_cs(zeta_deg)
    lib().orc_rotate_accumulate(C.c_int(Nx), C.c_int(Ny), _p(img), _p(valid), C.c_double(c), C.c_double(s),
                                _p(acc_sum), _p(acc_cnt))


def run(materials, voxel_nm, energies_eV, delta_par, beta_par, delta_perp, beta_perp,
        angles, ewald_mode, linear=False, return_images=False):
    """Algorithm 1 over all energies.  Optical constants are [n_energy][n_mat].
    angles = (start, step, end) in degrees.  Returns (out[nE][Ny][Nx] float64,
    cnt[nE][Ny][Nx] uint32) and, for linear=True and return_images=True, also the
    per-energy (Ixx, Iyy, Ixy, valid) stacks."""
    M = _Morph(materials)
    energies = np.atleast_1d(np.asarray(energies_eV, dtype=np.float64))
    nE = energies.size
    consts = [np.ascontiguousarray(x, np.float32).reshape(nE, M.n_mat)
              for x in (delta_par, beta_par, delta_perp, beta_perp)]
    out = np.zeros((nE, M.Ny, M.Nx), np.float64)
    cnt = np.zeros((nE, M.Ny, M.Nx), np.uint32)
    imgs = None
    if linear and return_images:
        imgs = (np.zeros((nE, M.Ny, M.Nx)), np.zeros((nE, M.Ny, M.Nx)), np.zeros((nE, M.Ny, M.Nx)),
                np.zeros((nE, M.Ny, M.Nx), np.uint8))
    for i in range(nE):
        common = [C.c_int(M.Nx), C.c_int(M.Ny), C.c_int(M.Nz), C.c_int(M.n_mat), C.c_double(voxel_nm),
                  M.phi, M.S, M.theta, M.psi, C.c_double(energies[i]),
                  _p(consts[0][i]), _p(consts[1][i]), _p(consts[2][i]), _p(consts[3][i]),
                  C.c_double(angles[0]), C.c_double(angles[1]), C.c_double(angles[2]), C.c_int(ewald_mode),
                  _p(out[i]), _p(cnt[i])]
        if linear:
            extra = [_p(imgs[j][i]) for j in range(4)] if imgs is not None else [None] * 4
            rc = lib().orc_run_energy_linear(*common, *extra)
        else:
            rc = lib().orc_run_energy(*common)
        if rc != 0:
            raise RuntimeError(f"oracle run failed (rc={rc})")
    if imgs is not None:
        return out, cnt, imgs
    return out, cnt


def reductions(img, cnt, voxel_nm, n_bins, sector_half_width_deg=20.0):
    """NEXT-1 reductions of one image [Ny][Nx]: (I[n_bins], A[n_bins], npix[n_bins], ISI).
    cnt may be None (every pixel takes part)."""
    img = np.ascontiguousarray(img, np.float64)
    Ny, Nx = img.shape
    c = None if cnt is None else np.ascontiguousarray(cnt, np.uint32)
    I = np.zeros(n_bins); A = np.zeros(n_bins); npix = np.zeros(n_bins, np.uint32); isi = C.c_double(0.0)
    tan_w = float(np.tan(np.deg2rad(np.float64(sector_half_width_deg))))
    lib().orc_reductions(C.c_int(Nx), C.c_int(Ny), C.c_double(voxel_nm), _p(img), None if c is None else _p(c),
                         C.c_int(n_bins), C.c_double(tan_w), _p(I), _p(A), _p(npix), C.byref(isi))
    return I, A, npix, isi.value
