"""Thin ctypes binding over libcyrsoxs.so -- same names as include/cyrsoxs.h, argument
marshalling only.  PyTorch supplies device memory and streams; every step of the path runs
in the library's CUDA kernels.  There is no CPU fallback: `load()` raises if the library has
not been built (python -m paper_2209_13121_b200.build) or cannot be loaded.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path
from typing import Optional, Sequence

PKG = Path(__file__).resolve().parent
LIB_PATH = PKG / "libcyrsoxs.so"

OK, ERR_INVALID_ARG, ERR_NOT_READY, ERR_CUDA, ERR_OOM, ERR_NOT_IMPLEMENTED = range(6)
EWALD_NEAREST, EWALD_TRILINEAR = 0, 1
ALG_AUTO, ALG_PER_ENERGY, ALG_SPECTRAL_BASIS = 0, 1, 2
REDUCE_STATIC_MAX_BINS, REDUCE_STATIC_MAX_ENERGIES, REDUCE_STATIC_MAX_CELLS = 1024, 1024, 32768   # include/cyrsoxs.h
STAGES = ("xpass", "zpass", "ypass", "ewald", "rotate")
N_STAGES = len(STAGES)

EXPORTS = [
    "cyrsoxs_create", "cyrsoxs_set_morphology", "cyrsoxs_set_morphology_host", "cyrsoxs_set_morphology_aos", "cyrsoxs_set_morphology_streamed",
    "cyrsoxs_set_optical_constants", "cyrsoxs_set_angles", "cyrsoxs_set_ewald", "cyrsoxs_set_algorithm",
    "cyrsoxs_set_counts_output", "cyrsoxs_set_profiling", "cyrsoxs_run", "cyrsoxs_num_angles",
    "cyrsoxs_set_spectra_shard", "cyrsoxs_set_energy_range", "cyrsoxs_run_spectra", "cyrsoxs_get_spectra", "cyrsoxs_get_spectra_part",
    "cyrsoxs_run_energies",
    "cyrsoxs_get_stats", "cyrsoxs_reduce", "cyrsoxs_reduce_static", "cyrsoxs_debug_fetch_images", "cyrsoxs_last_error", "cyrsoxs_destroy",
    "cyrsoxs_version",
]


class Stats(C.Structure):
    _fields_ = [
        ("algorithm", C.c_int), ("n_energy", C.c_int), ("n_angles", C.c_int), ("energy_batch", C.c_int),
        ("kernel_launches", C.c_longlong), ("stage_launches", C.c_longlong * N_STAGES),
        ("stage_bytes", C.c_double * N_STAGES), ("stage_ms", C.c_float * N_STAGES),
        ("workspace_bytes", C.c_double),
    ]


class CyrsoxsError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"cyrsoxs status {status}: {msg}")
        self.status = status


_lib: Optional[C.CDLL] = None


def load() -> C.CDLL:
    """Loads libcyrsoxs.so; raises (loudly) if it is missing -- there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise RuntimeError(f"{LIB_PATH} not built: run `python -m paper_2209_13121_b200.build` "
                           "(the CUDA library is the only implementation; there is no CPU fallback)")
    lib = C.CDLL(str(LIB_PATH))
    vp, fpp = C.c_void_p, C.POINTER(C.c_void_p)
    lib.cyrsoxs_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.POINTER(vp)]
    lib.cyrsoxs_set_morphology.argtypes = [vp, fpp, fpp, fpp, fpp]
    lib.cyrsoxs_set_morphology_host.argtypes = [vp, fpp, fpp, fpp, fpp, vp]
    lib.cyrsoxs_set_morphology_aos.argtypes = [vp, vp, vp]
    lib.cyrsoxs_set_morphology_streamed.argtypes = [vp, fpp, fpp, fpp, fpp, C.c_int]
    lib.cyrsoxs_set_optical_constants.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp]
    lib.cyrsoxs_set_angles.argtypes = [vp, C.c_double, C.c_double, C.c_double]
    lib.cyrsoxs_set_ewald.argtypes = [vp, C.c_int]
    lib.cyrsoxs_set_algorithm.argtypes = [vp, C.c_int]
    lib.cyrsoxs_set_counts_output.argtypes = [vp, vp]
    lib.cyrsoxs_set_profiling.argtypes = [vp, C.c_int]
    lib.cyrsoxs_run.argtypes = [vp, vp, vp]
    lib.cyrsoxs_set_spectra_shard.argtypes = [vp, C.c_int, C.c_int]
    lib.cyrsoxs_set_energy_range.argtypes = [vp, C.c_int, C.c_int]
    lib.cyrsoxs_run_spectra.argtypes = [vp, vp]
    lib.cyrsoxs_get_spectra.argtypes = [vp, C.POINTER(vp), C.POINTER(C.c_ulonglong), C.POINTER(C.c_int)]
    lib.cyrsoxs_get_spectra_part.argtypes = [vp, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int)]
    lib.cyrsoxs_run_energies.argtypes = [vp, vp, vp]
    lib.cyrsoxs_num_angles.argtypes = [vp]
    lib.cyrsoxs_get_stats.argtypes = [vp, C.POINTER(Stats)]
    lib.cyrsoxs_debug_fetch_images.argtypes = [vp, C.c_int, vp]
    lib.cyrsoxs_reduce.argtypes = [vp, vp, vp, vp, C.c_int, C.c_int, C.c_double, vp, vp, vp]
    lib.cyrsoxs_reduce_static.argtypes = [vp, vp, vp, vp, C.c_int, C.c_int, C.c_double, vp, vp, vp]
    lib.cyrsoxs_last_error.argtypes = [vp]
    lib.cyrsoxs_last_error.restype = C.c_char_p
    lib.cyrsoxs_destroy.argtypes = [vp]
    lib.cyrsoxs_destroy.restype = None
    lib.cyrsoxs_version.restype = C.c_char_p
    for name in EXPORTS:
        getattr(lib, name)
    _lib = lib
    return lib


def _table(ptrs: Sequence[Optional[int]]):
    arr = (C.c_void_p * len(ptrs))()
    for i, p in enumerate(ptrs):
        arr[i] = p
    return arr


class Context:
    """RAII wrapper of a cyrsoxs_ctx.  Methods mirror the C calls one to one."""

    def __init__(self, Nx: int, Ny: int, Nz: int, n_mat: int, voxel_nm: float):
        self.lib = load()
        self.h = C.c_void_p()
        st = self.lib.cyrsoxs_create(Nx, Ny, Nz, n_mat, voxel_nm, C.byref(self.h))
        if st != OK:
            raise CyrsoxsError(st, self.lib.cyrsoxs_last_error(None).decode())
        self.Nx, self.Ny, self.Nz, self.n_mat = Nx, Ny, Nz, n_mat
        self.n_energy = 0
        self._keep = []

    def _check(self, st: int):
        if st != OK:
            raise CyrsoxsError(st, self.lib.cyrsoxs_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None) is not None and self.h:
            self.lib.cyrsoxs_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- setters ---------------------------------------------------------------------------
    def set_morphology(self, materials):
        """materials: list of (phi, S, theta, psi) CUDA float32 tensors (S/theta/psi may be None)."""
        tabs = []
        keep = []
        for k in range(4):
            col = []
            for mat in materials:
                t = mat[k]
                if t is None:
                    col.append(None)
                else:
                    assert t.is_cuda and t.is_contiguous() and t.dtype.itemsize == 4, "need contiguous CUDA float32"
                    keep.append(t)
                    col.append(t.data_ptr())
            tabs.append(_table(col))
        self._check(self.lib.cyrsoxs_set_morphology(self.h, *tabs))
        self._keep = keep

    def _host_tables(self, materials):
        tabs = []
        keep = []
        for k in range(4):
            col = []
            for mat in materials:
                t = mat[k]
                if t is None:
                    col.append(None)
                elif hasattr(t, "data_ptr"):
                    keep.append(t); col.append(t.data_ptr())
                else:
                    keep.append(t); col.append(t.ctypes.data)
            tabs.append(_table(col))
        return tabs, keep

    def set_morphology_host(self, materials, stream: int = 0):
        """materials: list of (phi, S, theta, psi) host arrays (numpy or pinned torch), copied by the library."""
        tabs, keep = self._host_tables(materials)
        self._check(self.lib.cyrsoxs_set_morphology_host(self.h, *tabs, C.c_void_p(stream)))
        self._keep = keep

    def set_morphology_streamed(self, materials, materials_per_group: int = 1):
        """materials: list of (phi, S, theta, psi) pinned host arrays, BORROWED for every later run: the
        morphology is streamed through a 2 x materials_per_group staging area at each run."""
        tabs, keep = self._host_tables(materials)
        self._check(self.lib.cyrsoxs_set_morphology_streamed(self.h, *tabs, int(materials_per_group)))
        self._keep = keep

    def set_morphology_aos(self, real4_ptr: int, stream: int = 0):
        """The paper's Real4 layout: [n_mat][Nz*Ny*Nx] entries (phi, S, psi, theta), device memory."""
        self._mats = None
        self._check(self.lib.cyrsoxs_set_morphology_aos(self.h, real4_ptr, stream or None))

    def set_optical_constants(self, energies, delta_par, beta_par, delta_perp, beta_perp):
        import numpy as np
        E = np.ascontiguousarray(energies, np.float64).reshape(-1)
        tabs = [np.ascontiguousarray(x, np.float32).reshape(E.size, self.n_mat) for x in
                (delta_par, beta_par, delta_perp, beta_perp)]
        self._check(self.lib.cyrsoxs_set_optical_constants(self.h, E.size, E.ctypes.data, *(t.ctypes.data for t in tabs)))
        self.n_energy = int(E.size)

    def set_angles(self, start, step, end):
        self._check(self.lib.cyrsoxs_set_angles(self.h, start, step, end))

    def set_ewald(self, mode: int):
        self._check(self.lib.cyrsoxs_set_ewald(self.h, mode))

    def set_algorithm(self, alg: int):
        self._check(self.lib.cyrsoxs_set_algorithm(self.h, alg))

    def set_counts_output(self, counts_ptr: Optional[int]):
        self._check(self.lib.cyrsoxs_set_counts_output(self.h, C.c_void_p(counts_ptr)))

    def set_profiling(self, on: bool):
        self._check(self.lib.cyrsoxs_set_profiling(self.h, int(on)))

    # -- run -------------------------------------------------------------------------------
    def run(self, out_ptr: int, stream: int = 0):
        self._check(self.lib.cyrsoxs_run(self.h, C.c_void_p(stream), C.c_void_p(out_ptr)))

    # -- two-phase run, spectra shards (multi-GPU; cyrsoxs.h) -------------------------------
    def set_spectra_shard(self, part: int, n_parts: int):
        self._check(self.lib.cyrsoxs_set_spectra_shard(self.h, part, n_parts))

    def set_energy_range(self, first: int, count: int):
        self._check(self.lib.cyrsoxs_set_energy_range(self.h, first, count))

    def run_spectra(self, stream: int = 0):
        self._check(self.lib.cyrsoxs_run_spectra(self.h, C.c_void_p(stream)))

    def run_energies(self, out_ptr: int, stream: int = 0):
        self._check(self.lib.cyrsoxs_run_energies(self.h, C.c_void_p(stream), C.c_void_p(out_ptr)))

    def spectra(self):
        """(device pointer, bytes per pack, n_pack) of the context-owned pruned spectra."""
        p, nb, n = C.c_void_p(), C.c_ulonglong(), C.c_int()
        self._check(self.lib.cyrsoxs_get_spectra(self.h, C.byref(p), C.byref(nb), C.byref(n)))
        return int(p.value), int(nb.value), int(n.value)

    def spectra_part(self, part: int):
        """(first pack, number of packs) of a part of the spectra shard."""
        a, n = C.c_int(), C.c_int()
        self._check(self.lib.cyrsoxs_get_spectra_part(self.h, part, C.byref(a), C.byref(n)))
        return int(a.value), int(n.value)

    def num_angles(self) -> int:
        return int(self.lib.cyrsoxs_num_angles(self.h))

    def stats(self) -> dict:
        s = Stats()
        self._check(self.lib.cyrsoxs_get_stats(self.h, C.byref(s)))
        return {
            "algorithm": s.algorithm, "n_energy": s.n_energy, "n_angles": s.n_angles, "energy_batch": s.energy_batch,
            "kernel_launches": int(s.kernel_launches),
            "stage_launches": {n: int(s.stage_launches[i]) for i, n in enumerate(STAGES)},
            "stage_bytes": {n: float(s.stage_bytes[i]) for i, n in enumerate(STAGES)},
            "stage_ms": {n: float(s.stage_ms[i]) for i, n in enumerate(STAGES)},
            "workspace_bytes": float(s.workspace_bytes),
        }

    def reduce(self, images_ptr: int, counts_ptr: Optional[int], n_energy: int, n_bins: int, sector_half_width_deg: float,
               I_ptr: int, A_ptr: Optional[int] = None, isi_ptr: Optional[int] = None, stream: int = 0):
        self._check(self.lib.cyrsoxs_reduce(self.h, stream or None, images_ptr, counts_ptr or None, n_energy, n_bins,
                                            float(sector_half_width_deg), I_ptr, A_ptr or None, isi_ptr or None))

    def reduce_static(self, images_ptr: int, counts_ptr: Optional[int], n_energy: int, n_bins: int, sector_half_width_deg: float,
                      I_ptr: int, A_ptr: Optional[int] = None, isi_ptr: Optional[int] = None, stream: int = 0):
        """cyrsoxs_reduce_static: `reduce` for callers that must not allocate device memory (another pool owns the HBM, or
        cudaMalloc's device-wide synchronisation is unacceptable).  Scratch is a fixed array inside the library, shared by
        all calls on a GPU: at most REDUCE_STATIC_MAX_BINS bins, REDUCE_STATIC_MAX_ENERGIES energies and
        REDUCE_STATIC_MAX_CELLS energies x bins; calls that overlap on the GPU race (include/cyrsoxs.h)."""
        self._check(self.lib.cyrsoxs_reduce_static(self.h, stream or None, images_ptr, counts_ptr or None, n_energy, n_bins,
                                                   float(sector_half_width_deg), I_ptr, A_ptr or None, isi_ptr or None))

    def debug_fetch_images(self, e_in_batch: int, dst_ptr: int):
        self._check(self.lib.cyrsoxs_debug_fetch_images(self.h, e_in_batch, C.c_void_p(dst_ptr)))


def simulate(workload, algorithm: int = ALG_AUTO, device: str = "cuda:0", want_counts: bool = False,
             want_images: bool = False):
    """Convenience for tests/bench: uploads a `workloads.Workload` with torch, runs it on the
    current stream and returns the images as a CUDA tensor [nE][Ny][Nx] (plus counts/images)."""
    import torch
    dev = torch.device(device)
    mats = [tuple(None if a is None else torch.from_numpy(a).to(dev) for a in m) for m in workload.materials]
    ctx = Context(workload.Nx, workload.Ny, workload.Nz, workload.n_mat, workload.voxel_nm)
    ctx.set_morphology(mats)
    ctx.set_optical_constants(workload.energies, workload.delta_par, workload.beta_par, workload.delta_perp,
                              workload.beta_perp)
    ctx.set_angles(*workload.angles)
    ctx.set_ewald(workload.ewald)
    ctx.set_algorithm(algorithm)
    out = torch.empty((workload.n_energy, workload.Ny, workload.Nx), dtype=torch.float32, device=dev)
    res = [out]
    counts = None
    if want_counts:
        counts = torch.zeros((workload.n_energy, workload.Ny, workload.Nx), dtype=torch.int32, device=dev)
        ctx.set_counts_output(counts.data_ptr())
        res.append(counts)
    stream = torch.cuda.current_stream(dev).cuda_stream
    ctx.run(out.data_ptr(), stream)
    if want_images:
        n = min(workload.n_energy, ctx.stats()["energy_batch"])
        last = workload.n_energy - ((workload.n_energy - 1) // n) * n
        imgs = torch.empty((last, workload.Ny, workload.Nx, 4), dtype=torch.float32, device=dev)
        for e in range(last):
            ctx.debug_fetch_images(e, imgs[e].data_ptr())
        res.append(imgs)
    torch.cuda.synchronize(dev)
    res.append(ctx)
    return tuple(res)
