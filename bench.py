#!/usr/bin/env python
"""bench.py -- throughput of the CyRSoXS hot path on B200 (contract: task prompt section 4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg5]

A "step" is one pass of the whole hot path (all energies x all E-field angles of the
workload) over one synthetic morphology.  Metric: E-angle patterns/s (BASELINE.json), device
timed with CUDA events on the launching stream; voxel.angle evaluations/s is reported beside
it.  BASELINE.json's metric names no config, so the default workload is the largest single-GPU one,
configs[4] (1024 x 1024 x 512, 20 energies x 9 angles; configs[2] if the device or host is too small);
the other configs are timed with fewer steps into the `per_config` key.  N > 1: energies are independent units, so every rank simulates its
own slice of a N-times longer energy list on the same morphology -- no data-path collective,
weak scaling.  `--impl reference` times the CPU oracle (as it stands) on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2209_13121_b200 import workloads as W  # noqa: E402

METRIC = "E-angle patterns/s (device-timed)"
UNIT = "patterns/s"

def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def make_workload(name: str, rank: int, world: int):
    if name == "cfg1":
        w = W.cfg1()
    elif name == "cfg2":
        w = W.cfg2()
    elif name == "cfg3":
        w = W.cfg3()
    elif name == "cfg4":
        w = W.cfg4()
    elif name == "cfg5":
        w = W.cfg5()
    else:
        raise SystemExit(f"unknown workload {name}")
    if world > 1:
        # weak scaling: a world-times longer energy list over the same range, rank r owns slice r
        E = np.linspace(w.energies[0], w.energies[-1], w.n_energy * world) if w.n_energy > 1 else np.repeat(w.energies, world)
        tabs = []
        for t in (w.delta_par, w.beta_par, w.delta_perp, w.beta_perp):
            full = np.stack([np.interp(E, w.energies, t[:, m]) if w.n_energy > 1 else np.repeat(t[:, m], world)
                             for m in range(w.n_mat)], 1).astype(np.float32)
            tabs.append(full[rank * w.n_energy:(rank + 1) * w.n_energy])
        w.energies = E[rank * w.n_energy:(rank + 1) * w.n_energy].copy()
        w.delta_par, w.beta_par, w.delta_perp, w.beta_perp = tabs
    return w


def workload_label(w, name: str) -> str:
    idx = {"cfg1": 0, "cfg2": 1, "cfg3": 2, "cfg4": 3, "cfg5": 4}[name]
    return (f"{w.name}: {w.Nx}x{w.Ny}x{w.Nz} voxels, {w.n_mat} materials, {w.n_energy} energies x {w.n_angles} angles per GPU, "
            f"ewald={'trilinear' if w.ewald else 'nearest'} (BASELINE.json configs[{idx}])")


class ClockSampler(threading.Thread):
    """Samples SM clock, power and throttle reasons while the timed region runs.  Uses NVML in
    process (pynvml); spawning nvidia-smi every 100 ms stalls kernel launches of a 0.15 ms step
    for milliseconds, so it is only the fallback."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False
        self.nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and all(x.strip().isdigit() for x in vis.split(",")) else index
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.nvml = pynvml
        except Exception:
            self.nvml = None

    def _sample_nvml(self):
        n, h = self.nvml, self.handle
        sm = n.nvmlDeviceGetClockInfo(h, n.NVML_CLOCK_SM)
        mx = n.nvmlDeviceGetMaxClockInfo(h, n.NVML_CLOCK_SM)
        pw = n.nvmlDeviceGetPowerUsage(h) / 1000.0
        r = n.nvmlDeviceGetCurrentClocksEventReasons(h) if hasattr(n, "nvmlDeviceGetCurrentClocksEventReasons") \
            else n.nvmlDeviceGetCurrentClocksThrottleReasons(h)
        bits = [getattr(n, "nvmlClocksThrottleReasonHwSlowdown", 0x8), getattr(n, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                getattr(n, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20), getattr(n, "nvmlClocksThrottleReasonSwPowerCap", 0x4)]
        return [str(sm), str(mx), str(pw)] + ["Active" if r & b else "Not Active" for b in bits]

    def sample_once(self):
        try:
            if self.nvml is not None:
                self.rows.append(self._sample_nvml())
            else:
                o = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                   capture_output=True, text=True, timeout=5).stdout.strip()
                if o:
                    self.rows.append([x.strip() for x in o.split(",")])
        except Exception:
            pass

    def run(self):
        while not self.stop_flag:
            self.sample_once()
            time.sleep(0.005 if self.nvml is not None else 0.1)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for j, n in enumerate(names) if any(r[3 + j].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(sm), "power_w_max": max(float(r[2]) for r in self.rows),
                "source": "nvml" if self.nvml is not None else "nvidia-smi"}


def oracle_sample(w, budget_s: float = 20.0):
    """The oracle as it stands (definition mode: per angle polarization, three FFTs, Ewald, rotate) on a bounded
    sample of the workload that takes about `budget_s` seconds: the first `planes` z planes of the morphology (all of
    them if one full-size angle fits the budget), as many of the workload's angles as fit for the first energy and, if
    all of them fit, as many further energies as fit.  A sample thinner than the workload is scaled to the full size by
    its voxel.angle rate (the paper reports wall time O(N) in the number of voxels).
    Returns (patterns/s of the full-size workload, description, seconds, threads)."""
    import oracle

    def run(planes, n_e, n_a):
        mats = [tuple(None if a is None else a[:planes] for a in m) for m in w.materials]
        t0 = time.perf_counter()
        oracle.run(mats, w.voxel_nm, w.energies[:n_e], w.delta_par[:n_e], w.beta_par[:n_e], w.delta_perp[:n_e],
                   w.beta_perp[:n_e], (w.angles[0], w.angles[1], w.angles[0] + (n_a - 1) * w.angles[1]), w.ewald)
        return time.perf_counter() - t0

    p0 = min(w.Nz, 2)
    run(p0, 1, 1)                                            # warms the page cache / thread pool
    t0 = run(p0, 1, 1)
    planes = p0
    while planes * 2 <= w.Nz and t0 * (planes * 2 / p0) * 1.3 <= budget_s:      # 1.3: the FFT's log factor and cache effects
        planes *= 2
    if planes * 2 > w.Nz and t0 * (w.Nz / p0) * 1.3 <= budget_s:
        planes = w.Nz
    t1 = t0 * planes / p0 * (1.3 if planes > p0 else 1.0)
    n_a = int(max(1, min(w.n_angles, budget_s / max(t1, 1e-9)))) if planes == w.Nz else 1
    n_e = int(max(1, min(w.n_energy, budget_s / max(t1 * n_a, 1e-9)))) if n_a == w.n_angles else 1
    dt = run(planes, n_e, n_a)
    vox_angle_per_s = float(planes) * w.Ny * w.Nx * n_e * n_a / dt
    desc = (f"{n_e} of {w.n_energy} energies x {n_a} of {w.n_angles} angles on {planes} of {w.Nz} z planes of the same morphology, "
            f"definition mode (polarization, 3 FFTs, Ewald, rotate per angle), {dt:.1f} s"
            + ("" if planes == w.Nz else "; scaled to the full depth by voxel.angle/s (wall time O(N), PAPER.md:473)"))
    return vox_angle_per_s / w.n_vox, desc, dt, oracle.num_threads()


def resolve_workload(name: str) -> str:
    if name != "auto":
        return name
    try:
        import torch
        if torch.cuda.is_available():
            return pick_default_workload(torch.device("cuda", 0))
    except Exception:
        pass
    return "cfg3"


def run_reference(args, rank, world):
    if rank != 0:
        return
    name = resolve_workload(args.workload)
    w = make_workload(name, 0, 1)
    vals = []
    for i in range(args.warmup + args.steps):
        v, desc, dt, cores = oracle_sample(w, budget_s=max(1.0, 90.0 / (args.warmup + args.steps)))
        if i >= args.warmup:
            vals.append((v, dt, desc))
    value = sum(v[0] * v[1] for v in vals) / sum(v[1] for v in vals)          # time-weighted mean rate
    sample = vals[0][2] + " per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * sum(v[1] for v in vals) / len(vals), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(w, name), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def kernel_groups(st):
    """Stages (cyrsoxs_stats) grouped by the kernel that runs them, with what bounds each kernel.  The
    names are those of the SPECTRAL_BASIS kernels the default run launches."""
    g = {"k_xbasis3 (fields + FFT along x)": (["xpass"], "HBM stream, instruction-issue limited (DESIGN 7.1)"),
         "k_col2p (FFT along z, then along y)": (["zpass", "ypass"], "HBM stream")}
    g["k_ewald_basis (Ewald gather)"] = (["ewald"], "instruction issue + L2 gather latency, not HBM (DESIGN 7.3)")
    g["k_rotate_avg (rotate back + average)"] = (["rotate"], "L1 data-pipe wavefronts / latency of the bilinear gathers, not HBM (DESIGN 7.4)")
    return g


def ncu_traffic(workload: str, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload`, from the tracked ncu captures
    listed in profiles/ncu_traffic.json (each entry names its capture file and the commit it was taken at)."""
    try:
        tab = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
    except Exception:
        return None, None
    short = kernel.split(" ")[0]
    ent = tab.get(workload, {}).get(short)
    if not ent:
        return None, None
    return float(ent["dram_bytes_per_launch"]), {k: ent[k] for k in ("capture", "commit") if k in ent}


def measure(name, args, rank, world, dev, steps, warmup, with_e2e, with_clocks, alg, streamed=0):
    """Device-timed steps of one workload (+ per-stage pass, + e2e through host buffers).  Returns a dict."""
    import torch
    import torch.distributed as dist
    from paper_2209_13121_b200 import binding
    strong = getattr(args, "scaling", "weak") == "strong" and world > 1
    w = make_workload(name, 0, 1) if strong else make_workload(name, rank, world)
    local_rank = dev.index
    mats = [tuple(None if a is None else torch.from_numpy(a).to(dev) for a in m) for m in w.materials]
    ctx = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
    if streamed > 0:
        # memory-minimising mode: the morphology stays in pinned host memory and is streamed
        # through the device group by group at every run -- PCIe traffic is then inside every timed step
        del mats
        pinned_main = [tuple(None if a is None else torch.from_numpy(a).pin_memory() for a in m) for m in w.materials]
        ctx.set_morphology_streamed(pinned_main, streamed)
    else:
        ctx.set_morphology(mats)
    ctx.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
    ctx.set_angles(*w.angles); ctx.set_ewald(w.ewald); ctx.set_algorithm(alg)
    out = torch.empty((w.n_energy, w.Ny, w.Nx), dtype=torch.float32, device=dev)
    stream = torch.cuda.current_stream(dev)
    sptr = stream.cuda_stream
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    if strong:
        # strong scaling (DESIGN 11): the SAME workload on all ranks; rank r transforms material group r % n_parts,
        # the pruned spectra are exchanged once per run (NCCL broadcasts on the run's stream), then every rank does
        # its slice of the energies
        from paper_2209_13121_b200 import sharding
        n_parts = min(world, w.n_mat)
        a_e, b_e = sharding.energy_slices(w.n_energy, world)[rank]
        ctx.set_spectra_shard(rank % n_parts, n_parts)
        if b_e > a_e:
            ctx.set_energy_range(a_e, b_e - a_e)
        # more ranks than energies: this rank transforms and exchanges but has no energy of its own (zero-row `out`)
        out = torch.empty((b_e - a_e, w.Ny, w.Nx), dtype=torch.float32, device=dev)

    def one_step():
        flush.fill_(1)                                  # L2 flush between timed iterations (outside the events)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        if strong:
            sharding.run_strong(ctx, w, out, sptr, device=dev.index)
        else:
            ctx.run(out.data_ptr(), sptr)
        b.record(stream)
        return a, b

    for _ in range(warmup):
        one_step()
    barrier()
    sampler = ClockSampler(local_rank) if with_clocks else None
    if sampler:
        sampler.start()
    evs = [one_step() for _ in range(steps)]
    if sampler and sampler.nvml is not None:
        sampler.sample_once()                           # at least one sample while the queue is still draining
    barrier()
    if sampler:
        sampler.stop_flag = True
        sampler.join(timeout=3)
    total_ms = float(sum(a.elapsed_time(b) for a, b in evs))
    if world > 1:
        t = torch.tensor([total_ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    st = ctx.stats()
    res = {"w": w, "ms_per_step": total_ms / steps, "total_ms": total_ms, "launches_per_step": int(st["kernel_launches"]), "st": st,
           "clocks": sampler.summary() if sampler else None}
    if args.quick or strong:
        res["strong"] = strong
        return res

    # ---- per-stage device times (CUDA events on the run's stream, inside the library) for the roofline
    ctx.set_profiling(True)
    stage_ms = {k: 0.0 for k in binding.STAGES}
    nprof = max(1, min(steps, 5))
    for _ in range(nprof):
        flush.fill_(1)
        ctx.run(out.data_ptr(), sptr)
        s2 = ctx.stats()
        for k in stage_ms:
            stage_ms[k] += s2["stage_ms"][k] / nprof
    ctx.set_profiling(False)
    res["stage_ms"] = stage_ms

    # ---- end to end through the C ABI with host buffers (H2D + D2H inside the timed region)
    if with_e2e:
        pinned = [tuple(None if a is None else torch.from_numpy(a).pin_memory() for a in m) for m in w.materials]
        h_out = torch.empty((w.n_energy, w.Ny, w.Nx), dtype=torch.float32).pin_memory()
        del ctx, mats                                   # the e2e context owns its own device copy of the morphology
        ctx2 = binding.Context(w.Nx, w.Ny, w.Nz, w.n_mat, w.voxel_nm)
        ctx2.set_optical_constants(w.energies, w.delta_par, w.beta_par, w.delta_perp, w.beta_perp)
        ctx2.set_angles(*w.angles); ctx2.set_ewald(w.ewald); ctx2.set_algorithm(alg)

        def e2e_step():
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ctx2.set_morphology_host(pinned, sptr)
            ctx2.run(h_out.data_ptr(), sptr)
            b.record(stream)
            return a, b

        for _ in range(max(1, min(warmup, 3))):
            e2e_step()
        barrier()
        n_e2e = max(1, min(steps, 10))
        ev2 = [e2e_step() for _ in range(n_e2e)]
        barrier()
        e2e_all = sorted(a.elapsed_time(b) for a, b in ev2)
        e2e_ms = float(sum(e2e_all)) / n_e2e
        if world > 1:
            t = torch.tensor([e2e_ms], device=dev, dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e2e_ms = float(t.item())
        res["e2e"] = {"ms": e2e_ms, "median_ms": float(e2e_all[len(e2e_all) // 2]),
                      "h2d": sum(a.numel() * 4 for m in pinned for a in m if a is not None), "d2h": h_out.numel() * 4}
        del ctx2, pinned, h_out
    torch.cuda.empty_cache()
    return res


def roofline_of(name, res, peak, peak_src):
    """The roofline object of one measured workload: the kernel with the largest summed device time."""
    w, st, stage_ms = res["w"], res["st"], res["stage_ms"]
    groups = kernel_groups(st)
    ktime = {k: sum(stage_ms[s_] for s_ in v[0]) for k, v in groups.items()}
    dom = max(ktime, key=lambda k: ktime[k])
    dom_stages = groups[dom][0]
    dom_launches = max(1, sum(st["stage_launches"][s_] for s_ in dom_stages))
    dom_ms_per_launch = ktime[dom] / dom_launches
    dom_bytes_per_launch = sum(st["stage_bytes"][s_] for s_ in dom_stages) / dom_launches
    achieved = dom_bytes_per_launch / (dom_ms_per_launch * 1e-3) / 1e9 if dom_ms_per_launch > 0 else 0.0
    whole_bytes = sum(st["stage_bytes"].values())
    ms = res["ms_per_step"]
    # SURVEY.md 8(d) contract model M0: (16 c + 96) bytes per voxel per energy (+28 per pixel in 2-D)
    m0_bytes = w.n_energy * ((16.0 * w.n_mat + 96.0) * w.n_vox + (28.0 * w.Nx * w.Ny if w.Nz == 1 else 0.0))
    traffic, traffic_src = ncu_traffic(name, dom)
    if dom_stages == ["rotate"]:
        # The rotate/average kernel is not an HBM kernel (DRAM 3 % busy at CFG4): its binding resource is the L1 data pipe,
        # one 128-byte wavefront per clock and SM (DESIGN 7.4).  Algorithmic work per launch: pixels x energies x angles
        # bilinear samples, 4 taps each, a warp-wide tap of 16-byte texels = 32 x 16 / 128 = 4 wavefronts.
        import torch
        n_sm = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
        sm_mhz = float((res.get("clocks") or {}).get("sm_max_mhz") or 1965.0)
        wavefronts = float(w.Nx) * w.Ny * w.n_energy * w.n_angles * 4.0 / 32.0 * 4.0 / dom_launches
        l1_peak = n_sm * sm_mhz * 1e6 / 1e9                          # G wavefronts/s
        l1_ach = wavefronts / (dom_ms_per_launch * 1e-3) / 1e9 if dom_ms_per_launch > 0 else 0.0
        return {"bound": "l1", "kernel": dom, "stages": dom_stages, "launches_per_step": dom_launches,
                "share_of_step": ktime[dom] / max(sum(ktime.values()), 1e-12),
                "achieved": l1_ach, "peak": l1_peak, "unit": "Gwavefront/s", "frac": l1_ach / l1_peak,
                "peak_source": f"L1 data pipe: 1 wavefront (128 B) per clock and SM x {n_sm} SMs x {sm_mhz:.0f} MHz (DESIGN 7.4)",
                "wavefronts_per_launch": wavefronts, "floor_ms_per_launch": wavefronts / (l1_peak * 1e9) * 1e3,
                "traffic": traffic, "traffic_source": traffic_src, "limiter": groups[dom][1],
                "hbm_frac": achieved / peak, "bytes_per_launch": dom_bytes_per_launch, "ms_per_launch": dom_ms_per_launch,
                "stage_ms_per_step": stage_ms,
                "stage_gbs": {k: (st["stage_bytes"][k] / (stage_ms[k] * 1e-3) / 1e9 if stage_ms[k] > 0 else 0.0) for k in stage_ms},
                "whole_step": {"bytes": whole_bytes, "achieved": whole_bytes / (ms * 1e-3) / 1e9, "frac": whole_bytes / (ms * 1e-3) / 1e9 / peak},
                "whole_step_vs_M0": {"bytes": m0_bytes, "achieved": m0_bytes / (ms * 1e-3) / 1e9, "frac": m0_bytes / (ms * 1e-3) / 1e9 / peak,
                                     "note": "M0 = (16c+96) B/voxel/energy (SURVEY 8(d))"}}
    return {"bound": "hbm", "kernel": dom, "stages": dom_stages, "launches_per_step": dom_launches,
            "share_of_step": ktime[dom] / max(sum(ktime.values()), 1e-12),
            "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "frac_vs_nominal_8000": achieved / 8000.0,
            "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src, "limiter": groups[dom][1],
            "bytes_per_launch": dom_bytes_per_launch, "ms_per_launch": dom_ms_per_launch,
            "stage_ms_per_step": stage_ms,
            "stage_gbs": {k: (st["stage_bytes"][k] / (stage_ms[k] * 1e-3) / 1e9 if stage_ms[k] > 0 else 0.0) for k in stage_ms},
            "whole_step": {"bytes": whole_bytes, "achieved": whole_bytes / (ms * 1e-3) / 1e9, "frac": whole_bytes / (ms * 1e-3) / 1e9 / peak},
            "whole_step_vs_M0": {"bytes": m0_bytes, "achieved": m0_bytes / (ms * 1e-3) / 1e9, "frac": m0_bytes / (ms * 1e-3) / 1e9 / peak,
                                 "note": "M0 = (16c+96) B/voxel/energy (SURVEY 8(d)); this build moves fewer bytes "
                                         "(energy-independent spectra, pruned windows), so frac > 1 is possible"}}


def cufft_comparison(w, dev, stage_ms):
    """cuFFT (through torch.fft.fftn) on the same transforms, as an outside yardstick for the hand-written passes
    (north_star: "cuFFT may be timed only as a comparison"; it is not on the product path).  One unpruned complex64 3-D
    transform of the workload's size per basis pack; no field generation, no morphology read, no pruning -- so it is the
    library's time for the FFT part alone, next to the build's fields + x + z + y passes."""
    import torch
    n_fields = sum(7 if m[1] is not None else 1 for m in w.materials)
    n_pack = (n_fields + 1) // 2
    try:
        x = torch.empty((w.Nz, w.Ny, w.Nx), dtype=torch.complex64, device=dev)
        torch.view_as_real(x).normal_()
        dims = (-3, -2, -1) if w.Nz > 1 else (-2, -1)
        for _ in range(2):
            y = torch.fft.fftn(x, dim=dims)
        torch.cuda.synchronize(dev)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 3
        a.record()
        for _ in range(reps):
            y = torch.fft.fftn(x, dim=dims)
        b.record()
        torch.cuda.synchronize(dev)
        per = a.elapsed_time(b) / reps
        del x, y
        torch.cuda.empty_cache()
        ours = stage_ms["xpass"] + stage_ms["zpass"] + stage_ms["ypass"]
        return {"library": "cuFFT via torch.fft.fftn, complex64, unpruned, out of place", "ms_per_transform": per, "n_transforms": n_pack,
                "ms_total": per * n_pack, "ours_fields_plus_fft_ms": ours, "ours_over_cufft": ours / (per * n_pack),
                "note": "comparison only; cuFFT is not linked into libcyrsoxs.so"}
    except Exception as ex:                                  # out of memory on a small device, or no cuFFT
        return {"unavailable": str(ex)[:200]}


def pick_default_workload(dev) -> str:
    """BASELINE.json names no config for the metric: the headline is the largest single-GPU one, configs[4]
    (1024 x 1024 x 512; 17 GB of morphology, 11 GB of workspace, 17 GB pinned for e2e).  A smaller device or
    host falls back to configs[2] and says so in config.workload."""
    import torch
    try:
        free_b, _ = torch.cuda.mem_get_info(dev)
        host_gb = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES") / 2**30
        return "cfg5" if free_b >= 60 * 2**30 and host_gb >= 100 else "cfg3"
    except Exception:
        return "cfg3"


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2209_13121_b200 import binding, build
    build.build()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    alg = {"auto": binding.ALG_AUTO, "per_energy": binding.ALG_PER_ENERGY, "spectral": binding.ALG_SPECTRAL_BASIS}[args.alg]
    name = resolve_workload(args.workload)
    fallback = " [fallback: configs[4] does not fit this device/host]" if args.workload == "auto" and name != "cfg5" else ""
    res = measure(name, args, rank, world, dev, args.steps, args.warmup, with_e2e=True, with_clocks=True, alg=alg, streamed=args.streamed)
    w, st = res["w"], res["st"]
    if args.quick:
        if rank == 0:
            print(json.dumps({"quick": True, "workload": name, "ms_per_step": res["ms_per_step"], "launches_per_step": res["launches_per_step"]}), flush=True)
        return
    peak, peak_src = load_peaks()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    if res.get("strong"):
        # total work is fixed: all energies x angles of the workload, whatever the number of GPUs
        line = {"metric": METRIC, "value": w.n_energy * w.n_angles / (res["ms_per_step"] * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": res["ms_per_step"], "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": workload_label(w, name), "l2": "flushed between timed steps (256 MB write)",
                           "parallelism": f"spectra sharded over min({world}, {w.n_mat}) material groups, one broadcast of the pruned "
                                          f"spectra per group and run over NCCL, then energies sharded over {world} GPUs"},
                "gpu_launches": int(res["launches_per_step"] * args.steps), "clocks": res["clocks"]}
        print(json.dumps(line), flush=True)
        dist.destroy_process_group()
        return
    patterns = w.n_energy * w.n_angles * world
    value = patterns / (res["ms_per_step"] * 1e-3)
    e2e = res["e2e"]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": res["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {
            "workload": workload_label(w, name) + fallback,
            "algorithm": {1: "per_energy", 2: "spectral_basis"}.get(st["algorithm"], "?"),
            "energy_batch": st["energy_batch"], "l2": "flushed between timed steps (256 MB write)",
            "parallelism": f"energies sharded over {world} GPU(s), no collective",
            "morphology": (f"streamed from pinned host memory, {args.streamed} material(s) per group" if args.streamed > 0
                           else "resident in HBM"),
        },
        "voxel_angle_evals_per_s": value * w.n_vox,
        "device_bytes": {"morphology": int(sum(a.nbytes for m in w.materials for a in m if a is not None)) if args.streamed == 0 else 0,
                         "workspace": int(st["workspace_bytes"])},
        "e2e": {"value": patterns / (e2e["ms"] * 1e-3), "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"],
                "d2h_bytes_per_step": e2e["d2h"], "ms_per_step": e2e["ms"], "ms_per_step_median": e2e["median_ms"],
                "note": "PCIe-bound: uploads the whole morphology every step"},
        "gpu_launches": int(res["launches_per_step"] * args.steps),
        "clocks": res["clocks"],
        "roofline": roofline_of(name, res, peak, peak_src),
    }
    if world == 1:
        line["cufft_comparison"] = cufft_comparison(w, dev, res["stage_ms"])
    if world == 1 and not args.no_cpu_baseline:
        v, desc, dt, cores = oracle_sample(w, budget_s=20.0)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
    del res, w
    if world == 1 and not args.no_per_config:
        # the other BASELINE.json configs, measured the same way with fewer steps (no e2e, no CPU baseline)
        per = {}
        for other in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5"):
            if other == name or (other == "cfg5" and name != "cfg5"):
                continue
            r = measure(other, args, 0, 1, dev, 5, 3, with_e2e=False, with_clocks=False, alg=alg)
            rf = roofline_of(other, r, peak, peak_src)
            wo = r["w"]
            per[other] = {"workload": workload_label(wo, other), "ms_per_step": r["ms_per_step"],
                          "patterns_per_s": wo.n_energy * wo.n_angles / (r["ms_per_step"] * 1e-3),
                          "dominant_kernel": rf["kernel"], "bound": rf["bound"], "frac": rf["frac"], "unit": rf["unit"],
                          "ms_per_launch": rf["ms_per_launch"], "traffic": rf["traffic"],
                          "stage_ms_per_step": rf["stage_ms_per_step"], "cufft_comparison": cufft_comparison(wo, dev, r["stage_ms"]),
                          "whole_step_frac": rf["whole_step"]["frac"], "whole_step_vs_M0_frac": rf["whole_step_vs_M0"]["frac"]}
            del r, wo
        line["per_config"] = per
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="auto", help="cfg1 .. cfg5; auto: cfg5 (BASELINE.json configs[4]), cfg3 if it does not fit")
    ap.add_argument("--alg", default="auto", choices=["auto", "per_energy", "spectral"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank its own energies of an N-times finer grid (default); strong = the same workload, "
                         "spectra sharded over materials and exchanged, energies sharded (DESIGN 11)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config key (the other BASELINE.json configs)")
    ap.add_argument("--quick", action="store_true", help="device-timed steps only (no e2e, no per-stage pass, no CPU baseline): the command ncu wraps")
    ap.add_argument("--streamed", type=int, default=0, help="materials per group of cyrsoxs_set_morphology_streamed (0: resident)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world == 1 and args.gpus > 1 and args.impl == "ours":
        # launched without torchrun: re-exec under torch.distributed.run on this node
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", "29531", os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
