"""Seeded synthetic workloads (inputs only -- none of the method's arithmetic lives here).

The paper measures on no public dataset: its performance workloads are shapes only
 and its validation inputs need tables that are not
available.  These generators restate the five BASELINE.json configs
plus tiny cases; the exact recipes are written out in DESIGN.md section 5.  Both the
CPU oracle and the CUDA path consume the float32 arrays produced here.

Arrays are C-order [Nz][Ny][Nx]; a material is (phi, S, theta, psi) with S/theta/psi
None for an isotropic material.  Angles are (start, step, end) in degrees.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

EWALD_NEAREST = 0
EWALD_TRILINEAR = 1

Material = Tuple[np.ndarray, Optional[np.ndarray], Optional[np.ndarray], Optional[np.ndarray]]


@dataclass
class Workload:
    name: str
    Nx: int
    Ny: int
    Nz: int
    voxel_nm: float
    materials: List[Material]
    energies: np.ndarray            # float64 [nE]
    delta_par: np.ndarray           # float32 [nE][c]
    beta_par: np.ndarray
    delta_perp: np.ndarray
    beta_perp: np.ndarray
    angles: Tuple[float, float, float]
    ewald: int
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def n_mat(self) -> int:
        return len(self.materials)

    @property
    def n_energy(self) -> int:
        return int(self.energies.size)

    @property
    def n_angles(self) -> int:
        s, d, e = self.angles
        return 1 if s == e else int(np.floor((e - s) / d + 1e-9)) + 1

    @property
    def n_vox(self) -> int:
        return self.Nx * self.Ny * self.Nz

    def restrict_energies(self, idx) -> "Workload":
        idx = np.atleast_1d(np.asarray(idx))
        return Workload(self.name, self.Nx, self.Ny, self.Nz, self.voxel_nm, self.materials,
                        self.energies[idx].copy(), self.delta_par[idx].copy(), self.beta_par[idx].copy(),
                        self.delta_perp[idx].copy(), self.beta_perp[idx].copy(), self.angles, self.ewald,
                        self.notes, dict(self.extra))


# --------------------------------------------------------------------------- helpers

def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def grf(shape, ell, rng):
    """Unit-variance periodic Gaussian random field: white N(0,1) noise filtered in
    Fourier space by exp(-|kappa|^2 ell^2 / 2) (kappa in rad/voxel), renormalised to std 1."""
    noise = rng.standard_normal(shape).astype(np.float32)
    F = np.fft.rfftn(noise)
    k2 = np.zeros(F.shape, np.float32)
    nd = len(shape)
    for ax, n in enumerate(shape):
        kap = 2.0 * np.pi * (np.fft.rfftfreq(n) if ax == nd - 1 else np.fft.fftfreq(n))
        sh = [1] * nd
        sh[ax] = kap.size
        k2 = k2 + (kap.astype(np.float32) ** 2).reshape(sh)
    F *= np.exp(-0.5 * k2 * np.float32(ell) ** 2)
    g = np.fft.irfftn(F, s=shape, axes=tuple(range(nd)))
    g -= g.mean()
    g /= g.std()
    return g.astype(np.float32)


def lorentz_L(E, E0, w):
    return (w / 2.0) ** 2 / ((E - E0) ** 2 + (w / 2.0) ** 2)


def lorentz_D(E, E0, w):
    return (E0 - E) * (w / 2.0) / ((E - E0) ** 2 + (w / 2.0) ** 2)


_PEAKS = [(285.0, 0.6), (288.5, 1.0), (293.0, 3.0), (305.0, 12.0)]
# oscillator strengths T per (material, axis): (par, perp)
_MULTI_T = [
    ((3.0, 0.5, 1.0, 0.8), (0.5, 1.5, 1.0, 0.8)),
    ((0.8, 2.5, 1.2, 0.6), (1.6, 0.6, 1.2, 0.6)),
    ((1.2, 1.0, 1.5, 1.0), (1.2, 1.0, 1.5, 1.0)),
    ((0.3, 0.4, 0.8, 1.2), (0.3, 0.4, 0.8, 1.2)),
]


def multi_lorentzian_constants(energies, n_mat):
    """beta = 2e-4 + 1e-3 sum_j T_j L_j, delta = 1e-3 + 1e-3 sum_j T_j D_j."""
    E = np.asarray(energies, np.float64)
    out = [np.zeros((E.size, n_mat)) for _ in range(4)]  # dpar, bpar, dperp, bperp
    for m in range(n_mat):
        for axis, (d_i, b_i) in enumerate(((0, 1), (2, 3))):
            T = _MULTI_T[m][axis]
            L = sum(t * lorentz_L(E, e0, w) for t, (e0, w) in zip(T, _PEAKS))
            D = sum(t * lorentz_D(E, e0, w) for t, (e0, w) in zip(T, _PEAKS))
            out[d_i][:, m] = 1e-3 + 1e-3 * D
            out[b_i][:, m] = 2e-4 + 1e-3 * L
    return tuple(_f32(x) for x in out)


# --------------------------------------------------------------------------- configs

def cfg1(seed: int = 0, n: int = 256, n_disks: int = 40, radius: int = 8) -> Workload:
    """BASELINE.json configs[0]: 2-D film n x n x 1, 5 nm voxels, radial disks."""
    rng = np.random.default_rng(seed)
    centres = []
    lo, hi = radius + 1, n - radius - 1
    while len(centres) < n_disks:
        c = rng.uniform(lo, hi, size=2)
        if all((c[0] - d[0]) ** 2 + (c[1] - d[1]) ** 2 >= (2 * radius + 1) ** 2 for d in centres):
            centres.append(c)
    centres = np.round(np.array(centres))
    y, x = np.mgrid[0:n, 0:n].astype(np.float64)
    phi1 = np.zeros((n, n), np.float32)
    psi1 = np.zeros((n, n), np.float32)
    for cx, cy in centres:
        inside = (x - cx) ** 2 + (y - cy) ** 2 <= radius ** 2
        phi1[inside] = 1.0
        psi1[inside] = np.arctan2(y - cy, x - cx)[inside]
    S1 = phi1.copy()
    th1 = np.where(phi1 > 0, np.float32(np.pi / 2), np.float32(0)).astype(np.float32)
    sh = (1, n, n)
    mats = [(_f32(phi1).reshape(sh), _f32(S1).reshape(sh), _f32(th1).reshape(sh), _f32(psi1).reshape(sh)),
            (_f32(1.0 - phi1).reshape(sh), None, None, None)]
    return Workload(
        "cfg1_film256_disks", n, n, 1, 5.0, mats, np.array([285.0]),
        _f32([[2e-3, 1e-3]]), _f32([[1e-3, 5e-4]]), _f32([[5e-4, 1e-3]]), _f32([[2e-4, 5e-4]]),
        (0.0, 15.0, 165.0), EWALD_NEAREST, extra={"centres": centres})


def cfg2(seed: int = 2, n: int = 128, n_energy: int = 10) -> Workload:
    """BASELINE.json configs[1]: 3-D cube n^3, 2 nm voxels, GRF two-phase, random directors."""
    rng = np.random.default_rng(seed)
    shape = (n, n, n)
    ind = (grf(shape, 6.0, rng) > 0).astype(np.float32)
    # smooth with a sigma = 1 voxel periodic Gaussian (Fourier-space multiplication)
    F = np.fft.rfftn(ind)
    k2 = np.zeros(F.shape, np.float32)
    for ax, m in enumerate(shape):
        kap = 2.0 * np.pi * (np.fft.rfftfreq(m) if ax == 2 else np.fft.fftfreq(m))
        s = [1, 1, 1]
        s[ax] = kap.size
        k2 = k2 + (kap.astype(np.float32) ** 2).reshape(s)
    phi1 = np.clip(np.fft.irfftn(F * np.exp(-0.5 * k2), s=shape, axes=(0, 1, 2)), 0.0, 1.0).astype(np.float32)
    S1 = rng.uniform(0.0, 1.0, shape).astype(np.float32)
    th1 = rng.uniform(0.0, np.pi, shape).astype(np.float32)
    ps1 = rng.uniform(0.0, 2.0 * np.pi, shape).astype(np.float32)
    mats = [(phi1, S1, th1, ps1), (_f32(1.0 - phi1), None, None, None)]
    E = np.linspace(280.0, 290.0, n_energy)
    L, D = lorentz_L(E, 285.0, 0.5), lorentz_D(E, 285.0, 0.5)
    A_par, A_perp, A_iso = 3e-3, 1e-3, 1.5e-3
    dpar = np.stack([1e-4 + A_par * D, 1e-4 + A_iso * D], 1)
    bpar = np.stack([1e-4 + A_par * L, 1e-4 + A_iso * L], 1)
    dperp = np.stack([1e-4 + A_perp * D, 1e-4 + A_iso * D], 1)
    bperp = np.stack([1e-4 + A_perp * L, 1e-4 + A_iso * L], 1)
    return Workload("cfg2_cube128_grf", n, n, n, 2.0, mats, E, _f32(dpar), _f32(bpar), _f32(dperp), _f32(bperp),
                    (0.0, 5.0, 175.0), EWALD_NEAREST)


def cfg3(seed: int = 3, nx: int = 512, ny: int = 512, nz: int = 256, n_energy: int = 50,
         grain: float = 20.0) -> Workload:
    """BASELINE.json configs[2]: 3-phase periodic Voronoi tessellation, per-grain directors."""
    from scipy.spatial import cKDTree
    rng = np.random.default_rng(seed)
    n_seeds = max(3, int(round(nx * ny * nz / grain ** 3)))
    pts = rng.uniform(0.0, 1.0, (n_seeds, 3)) * np.array([nz, ny, nx])
    phase = rng.integers(0, 3, n_seeds)
    cos_t = rng.uniform(-1.0, 1.0, n_seeds)
    g_theta = np.arccos(cos_t).astype(np.float32)
    g_psi = rng.uniform(0.0, 2.0 * np.pi, n_seeds).astype(np.float32)
    tree = cKDTree(pts, boxsize=np.array([nz, ny, nx], dtype=np.float64))
    label = np.empty((nz, ny, nx), np.int32)
    yy, xx = np.mgrid[0:ny, 0:nx]
    for z in range(nz):
        q = np.stack([np.full(yy.size, z + 0.0), yy.ravel() + 0.0, xx.ravel() + 0.0], 1)
        _, idx = tree.query(q, workers=-1)
        label[z] = idx.reshape(ny, nx)
    ph = phase[label]
    mats = []
    for m in range(2):
        mine = ph == m
        phi = mine.astype(np.float32)
        S = np.where(mine, np.float32(0.8), np.float32(0)).astype(np.float32)
        th = np.where(mine, g_theta[label], np.float32(0)).astype(np.float32)
        ps = np.where(mine, g_psi[label], np.float32(0)).astype(np.float32)
        mats.append((phi, S, th, ps))
    mats.append(((ph == 2).astype(np.float32), None, None, None))
    E = np.linspace(270.0, 340.0, n_energy)
    dpar, bpar, dperp, bperp = multi_lorentzian_constants(E, 3)
    return Workload(f"cfg3_voronoi_{nx}x{ny}x{nz}", nx, ny, nz, 1.0, mats, E, dpar, bpar, dperp, bperp,
                    (0.0, 10.0, 170.0), EWALD_TRILINEAR)


def cfg4(seed: int = 4, n: int = 2048, n_energy: int = 100, n_walks: int = 300, n_steps: int = 400) -> Workload:
    """BASELINE.json configs[3]: 2-D fibril film, 4 materials."""
    from scipy import ndimage
    rng = np.random.default_rng(seed)
    scale = n / 2048.0
    n_walks = max(2, int(round(n_walks * scale * scale)))
    pos = rng.uniform(0.0, n, (n_walks, 2))
    head = rng.uniform(0.0, 2.0 * np.pi, n_walks)
    occupied = np.zeros((n, n), bool)
    heading = np.zeros((n, n), np.float32)
    for _ in range(n_steps):
        head = head + 0.05 * rng.standard_normal(n_walks)
        pos = (pos + np.stack([np.cos(head), np.sin(head)], 1)) % n   # (x, y)
        ix = np.floor(pos[:, 0]).astype(int) % n
        iy = np.floor(pos[:, 1]).astype(int) % n
        occupied[iy, ix] = True
        heading[iy, ix] = head
    dist, (jy, jx) = ndimage.distance_transform_edt(~occupied, return_indices=True)
    near_head = heading[jy, jx]
    fib = dist <= 3.0
    shell = (dist > 3.0) & (dist <= 6.0)
    rest = ~(fib | shell)
    g = np.clip(0.5 + 0.25 * grf((n, n), 10.0, rng), 0.0, 1.0).astype(np.float32)
    half_pi = np.float32(np.pi / 2)
    sh = (1, n, n)

    def mk(mask, s, psi):
        return (_f32(mask).reshape(sh), _f32(np.where(mask, s, 0)).reshape(sh),
                _f32(np.where(mask, half_pi, 0)).reshape(sh), _f32(np.where(mask, psi, 0)).reshape(sh))

    mats = [mk(fib, 0.9, near_head), mk(shell, 0.5, near_head + half_pi),
            (_f32(np.where(rest, g, 0)).reshape(sh), None, None, None),
            (_f32(np.where(rest, 1.0 - g, 0)).reshape(sh), None, None, None)]
    E = np.linspace(270.0, 340.0, n_energy)
    dpar, bpar, dperp, bperp = multi_lorentzian_constants(E, 4)
    return Workload(f"cfg4_fibrils_{n}x{n}x1", n, n, 1, 2.0, mats, E, dpar, bpar, dperp, bperp,
                    (0.0, 5.0, 175.0), EWALD_NEAREST)


def cfg5(seed: int = 5, nx: int = 1024, ny: int = 1024, nz: int = 512, n_energy: int = 20,
         coarse: int = 8) -> Workload:
    """BASELINE.json configs[4]: radial spheres (30 % volume) in a smoothly varying matrix.

    Smooth matrix fields come from coarse-grid Gaussian random fields (grid / `coarse`,
    correlation lengths 16/32 voxels) upsampled by nearest-cell lookup blended trilinearly;
    spheres are stamped one by one (union; the later sphere owns the overlap)."""
    rng = np.random.default_rng(seed)
    shape = (nz, ny, nx)
    n_vox = nx * ny * nz
    phi1 = np.zeros(shape, np.float32)
    th1 = np.zeros(shape, np.float32)
    ps1 = np.zeros(shape, np.float32)
    target = 0.30 * n_vox
    filled = 0
    n_sph = 0
    while filled < target:
        r = 10.0 * np.exp(0.3 * rng.standard_normal())
        c = rng.uniform(0.0, 1.0, 3) * np.array([nz, ny, nx])
        R = int(np.ceil(r))
        zz, yy, xx = np.mgrid[-R:R + 1, -R:R + 1, -R:R + 1]
        cz, cy, cx = np.floor(c).astype(int)
        dz, dy, dx = zz - (c[0] - cz), yy - (c[1] - cy), xx - (c[2] - cx)
        d2 = dx * dx + dy * dy + dz * dz
        inside = d2 <= r * r
        Z, Y, X = (zz + cz) % nz, (yy + cy) % ny, (xx + cx) % nx
        Zi, Yi, Xi = Z[inside], Y[inside], X[inside]
        filled += int(np.count_nonzero(phi1[Zi, Yi, Xi] == 0))
        phi1[Zi, Yi, Xi] = 1.0
        rr = np.sqrt(np.maximum(d2[inside], 1e-12))
        th1[Zi, Yi, Xi] = np.arccos(np.clip(dz[inside] / rr, -1.0, 1.0))
        ps1[Zi, Yi, Xi] = np.arctan2(dy[inside], dx[inside])
        n_sph += 1
    S1 = phi1.copy()

    def smooth(ell):
        cs = tuple(max(2, s // coarse) for s in shape)
        gcoarse = grf(cs, ell / coarse, rng)
        out = np.empty(shape, np.float32)
        # trilinear periodic upsampling, one z-slab at a time
        def axis_w(n, nc):
            pos = (np.arange(n) + 0.5) * nc / n - 0.5
            i0 = np.floor(pos).astype(int)
            t = (pos - i0).astype(np.float32)
            return i0 % nc, (i0 + 1) % nc, t
        z0, z1, tz = axis_w(nz, cs[0]); y0, y1, ty = axis_w(ny, cs[1]); x0, x1, tx = axis_w(nx, cs[2])
        gx = gcoarse[:, :, x0] * (1 - tx) + gcoarse[:, :, x1] * tx              # [cz][cy][nx]
        gxy = gx[:, y0, :] * (1 - ty)[None, :, None] + gx[:, y1, :] * ty[None, :, None]  # [cz][ny][nx]
        for z in range(nz):
            out[z] = gxy[z0[z]] * (1 - tz[z]) + gxy[z1[z]] * tz[z]
        return out

    S2 = (0.5 * np.clip(0.5 + 0.5 * smooth(16.0), 0.0, 1.0)).astype(np.float32)
    th2 = (np.float32(np.pi / 2) + np.float32(0.4) * smooth(32.0)).astype(np.float32)
    ps2 = (np.float32(np.pi) * smooth(32.0)).astype(np.float32)
    mats = [(phi1, S1, th1, ps1), (_f32(1.0 - phi1), S2, th2, ps2)]
    E = np.linspace(280.0, 300.0, n_energy)
    dpar, bpar, dperp, bperp = multi_lorentzian_constants(E, 2)
    return Workload(f"cfg5_spheres_{nx}x{ny}x{nz}", nx, ny, nz, 1.0, mats, E, dpar, bpar, dperp, bperp,
                    (0.0, 20.0, 160.0), EWALD_TRILINEAR, extra={"n_spheres": n_sph})


def tiny(seed: int = 11, nx: int = 8, ny: int = 8, nz: int = 4, n_mat: int = 3, n_energy: int = 2,
         voxel_nm: float = 5.0, ewald: int = EWALD_TRILINEAR, angles=(0.0, 30.0, 150.0),
         energies=None, isotropic_last: bool = True) -> Workload:
    """Random-everything small case (several tiles and ragged tails come from odd sizes
    such as 32 x 16 x 8): phi is a random partition of unity, S ~ U(0,1), theta ~ U(0,pi),
    psi ~ U(0,2pi), constants ~ U(1e-4, 3e-3)."""
    rng = np.random.default_rng(seed)
    shape = (nz, ny, nx)
    raw = rng.uniform(0.05, 1.0, (n_mat,) + shape)
    raw /= raw.sum(0, keepdims=True)
    mats = []
    for m in range(n_mat):
        if isotropic_last and m == n_mat - 1 and n_mat > 1:
            mats.append((_f32(raw[m]), None, None, None))
        else:
            mats.append((_f32(raw[m]), _f32(rng.uniform(0, 1, shape)), _f32(rng.uniform(0, np.pi, shape)),
                         _f32(rng.uniform(0, 2 * np.pi, shape))))
    E = np.linspace(280.0, 290.0, n_energy) if energies is None else np.asarray(energies, np.float64)
    cs = [_f32(rng.uniform(1e-4, 3e-3, (E.size, n_mat))) for _ in range(4)]
    if isotropic_last and n_mat > 1:
        cs[2][:, -1] = cs[0][:, -1]
        cs[3][:, -1] = cs[1][:, -1]
    return Workload(f"tiny_{nx}x{ny}x{nz}_c{n_mat}", nx, ny, nz, voxel_nm, mats, E, cs[0], cs[1], cs[2], cs[3],
                    tuple(angles), ewald)


CONFIGS = {"cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4, "cfg5": cfg5}
