#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path (S1..S7) on synthetic detector data.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload C4] [--nz NZ_TOTAL] [--e2e-nz NZ] [--no-cpu]

A step is one pass of the whole path over one volume of the workload (default C4 of
BASELINE.json: 2048 projections of 2048 x 2048 uint16 -> 2048^3 voxels, fp16, 32-slice chunks).
`value`  : GVoxel/s with the raw volume already resident in HBM (device-timed, CUDA events).
`e2e`    : the same metric through tcp_recon_volume_host with pinned HOST buffers, H2D and D2H
           copies inside the timed region (three-stream chunk pipeline).
`roofline`: the dominant kernel's algorithmic bytes or flops / its CUDA-event time (per-kernel
           events recorded inside the timed region by the library, TCP_OPT_PROFILE).
`cpu_baseline`: the CPU oracle, as it stands, on a bounded sample of the same workload.
N > 1 (torchrun): independent replicas, one volume per rank, no collective on the data path
(the method has none: slices are independent); value = all voxels / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), float(p.get("sm_max_mhz", 1965.0)), "measured"
    except Exception:
        return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            pass
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


KERNEL_NAMES = {"normalize": "normalize_half_kernel / normalize_kernel", "rows": "rows_kernel", "ifft_cols": "ifft_cols_pf_kernel / ifft_cols_kernel",
                "ifft_rows": "ifft_rows_kernel", "grid": "grid_tile_kernel"}
KERNEL_NAMES_MMA = {"rows": "rows_mma_kernel", "ifft_cols": "cols_mma_kernel", "ifft_rows": "irows_mma_kernel", "grid": "grid_mma_kernel"}


def kernel_label(m):
    return "Kaiser-Bessel half-width %d" % (m & 15) if m >> 4 else "Gaussian half-width %d" % m


def stage_model(w, nz, m, half_store, half_out, fused_s12=False):
    """Algorithmic HBM bytes and flops of one tcp_recon call (one chunk of nz slices), per kernel
    (SURVEY 8(d)).  fused_s12: S1+S2 run in the row kernel's loader
    (TCP_OPT_FUSE_NORMALIZE): no normalise kernel, the row kernel reads the uint16 counts."""
    n, M, P = w.n, 2 * w.n, w.nproj
    npair = (nz + 1) // 2
    br = 2 if half_store else 4
    bc = 2 * br
    bo = 2 if half_out else 4
    lg = np.log2(M)
    fft = 5.0 * M * lg                      # flops of one length-M complex transform
    if fused_s12:
        return {
            "rows": {"bytes": P * nz * n * 2 + npair * P * M * bc, "flops": 3 * fft * npair * P + 10.0 * P * nz * n},
            "grid": {"bytes": npair * P * M * bc + npair * M * M * bc, "flops": 4.0 * (2 * (m & 15)) ** 2 * npair * P * M},
            "ifft_cols": {"bytes": npair * M * M * bc + npair * n * M * bc, "flops": fft * npair * M},
            "ifft_rows": {"bytes": npair * n * M * bc + nz * n * n * bo, "flops": fft * npair * n},
        }
    m = m & 15                              # kernel code -> half-width (taps per axis = 2 m)
    return {
        "normalize": {"bytes": P * nz * n * (2 + br), "flops": 10.0 * P * nz * n},
        "rows": {"bytes": P * nz * n * br + npair * P * M * bc, "flops": 3 * fft * npair * P},
        "grid": {"bytes": npair * P * M * bc + npair * M * M * bc, "flops": 4.0 * (2 * m) ** 2 * npair * P * M},
        "ifft_cols": {"bytes": npair * M * M * bc + npair * n * M * bc, "flops": fft * npair * M},
        "ifft_rows": {"bytes": npair * n * M * bc + nz * n * n * bo, "flops": fft * npair * n},
    }


def build_volume(w, nz_total, device, ndistinct=4):
    """Device-resident synthetic volume, chunk-major [nchunks][nproj][nz_chunk][n] uint16, plus the
    averaged flat/dark [nchunks][nz_chunk][n].  `ndistinct` chunks spread over the stack are
    manufactured from the phantom (closed-form line integrals + count noise); the others repeat
    them cyclically -- the path has no data-dependent control flow, so timing is unaffected."""
    import torch
    import synthgen as sg
    import paper_2209_08450_b200 as tcp

    nzc = w.nz_chunk
    nchunks = nz_total // nzc
    raw = torch.empty((nchunks, w.nproj, nzc, w.n), dtype=torch.uint16, device=device)
    flat = torch.empty((nchunks, nzc, w.n), dtype=torch.float32, device=device)
    dark = torch.empty_like(flat)
    nd = min(ndistinct, nchunks)
    made = []
    for d in range(nd):
        ch = (d * nchunks) // nd + (nchunks // (2 * nd))        # spread over the stack
        z0 = int(ch * nzc * (w.nz_total / max(nz_total, 1)))     # same relative height in the phantom
        z0 = min(max(z0, 0), w.nz_total - nzc)
        r, ff, df = sg.make_counts_torch(w, list(range(z0, z0 + nzc)), device=device)
        f = torch.empty((nzc, w.n), dtype=torch.float32, device=device)
        dk = torch.empty_like(f)
        tcp.tcp_mean_frames_u16(ff.contiguous(), f)             # C4: "10 flat and 10 dark frames"
        tcp.tcp_mean_frames_u16(df.contiguous(), dk)
        made.append((r.contiguous(), f, dk, z0))
    torch.cuda.synchronize()
    for ch in range(nchunks):
        r, f, dk, _ = made[ch % nd]
        raw[ch].copy_(r)
        flat[ch].copy_(f)
        dark[ch].copy_(dk)
    return raw, flat, dark, made


def cpu_baseline(w, made, m, cores_hint=None):
    """The oracle as it stands (double precision, OpenMP over slices) on a bounded sample: as many
    slices of the first manufactured chunk as there are host threads."""
    import oracle as orc

    r, f, dk, z0 = made[0]
    cores = orc.num_threads()
    ns = min(cores, r.shape[1])
    import torch
    raw = r.view(torch.int16)[:, :ns].contiguous().cpu().numpy().view(np.uint16)
    flat = f[:ns].cpu().numpy()
    dark = dk[:ns].cpu().numpy()
    t0 = time.perf_counter()
    ref = orc.recon(raw, flat, dark, w.theta, w.center, w.filter, m, "grid")
    dt = time.perf_counter() - t0
    return {"value": ns * w.n * w.n / dt / 1e9, "unit": "GVoxel/s", "cores": cores, "kind": "oracle",
            "sample": "%d slices of %s (%d proj x %d px), oracle B_grid in fp64, %.1f s" % (ns, w.name, w.nproj, w.n, dt),
            "slices_per_s": ns / dt}, ref, (z0, ns)


def max_over_ranks(value, world, device=None):
    """Whole-job time = the slowest rank's (device-timed) value; no data-path collective exists (replicas)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_slices(nz_total, nz_chunk, world):
    """Replicas only: every rank reconstructs one full volume of nz_total slices
    (rounded down to whole chunks); the job's voxel count is world times that."""
    nz = nz_total - nz_total % nz_chunk
    return nz, world * nz


def measure_config(name, dtype, m, steps, warmup, dev, hbm_gbs):
    """Compute-only throughput of another BASELINE.json config (whole volume resident in HBM, CUDA events around the
    chunk loop, per-kernel events from the library): the `configs` entries of the bench line."""
    import torch
    import synthgen as sg
    import paper_2209_08450_b200 as tcp

    w = sg.make_workload(name, dtype=dtype)
    nzc, n = w.nz_chunk, w.n
    nz_total = w.nz_total - w.nz_total % nzc
    nchunks = nz_total // nzc
    half_store, half_out = w.dtype != "f32", w.dtype == "f16"
    raw, flat, dark, _ = build_volume(w, nz_total, dev)
    theta = torch.from_numpy(w.theta).to(dev)
    out = torch.empty((nz_total, n, n), dtype=torch.float16 if half_out else torch.float32, device=dev)
    r = tcp.Recon(n, w.nproj, nzc, w.center, w.dtype, w.filter, m)
    stream = torch.cuda.current_stream()

    def step():
        for ch in range(nchunks):
            r.recon(raw[ch], flat[ch], dark[ch], theta, out=out[ch * nzc:(ch + 1) * nzc], stream=stream)

    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    r.set_profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_ms, ncalls = {k: 0.0 for k in r.STAGES}, 0
    e0.record(stream)
    for _ in range(steps):
        step()
        ms, nc = r.profile_collect()
        for k in ms:
            stage_ms[k] += ms[k]
        ncalls += nc
    e1.record(stream)
    torch.cuda.synchronize()
    ms_step = e0.elapsed_time(e1) / steps
    r.set_profile(False)
    launches = r.launches_per_recon
    r.close()
    whole = sum(v["bytes"] for v in stage_model(w, nzc, m, half_store, half_out).values()) * nchunks
    res = {"workload": "%s: %d proj x %d x %d u16 -> %d^2 x %d voxels, %s, %d-slice chunks, %s, %s filter"
                       % (w.name, w.nproj, nz_total, n, n, nz_total, w.dtype, nzc, kernel_label(m), w.filter),
           "value": float(nz_total) * n * n / (ms_step * 1e-3) / 1e9, "unit": "GVoxel/s", "ms_per_step": ms_step,
           "slices_per_s": nz_total / (ms_step * 1e-3), "steps": steps, "warmup": warmup,
           "whole_path_hbm_frac": whole / (ms_step * 1e-3) / 1e9 / hbm_gbs, "launches_per_chunk": launches,
           "ms_per_chunk": {k: stage_ms[k] / max(ncalls, 1) for k in stage_ms}}
    del raw, flat, dark, out
    torch.cuda.empty_cache()
    return res


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    import synthgen as sg
    import paper_2209_08450_b200 as tcp

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    w = sg.make_workload(args.workload, dtype=args.dtype or None)
    if args.nz_chunk:
        w.nz_chunk = args.nz_chunk
    nz_total = args.nz or w.nz_total
    nz_total -= nz_total % w.nz_chunk
    nzc, n = w.nz_chunk, w.n
    nchunks = nz_total // nzc
    m = args.m
    half_store, half_out = w.dtype != "f32", w.dtype == "f16"
    out_dt = torch.float16 if half_out else torch.float32

    raw, flat, dark, made = build_volume(w, nz_total, dev)
    theta = torch.from_numpy(w.theta).to(dev)
    out = torch.empty((nz_total, n, n), dtype=out_dt, device=dev)
    r = tcp.Recon(n, w.nproj, nzc, w.center, w.dtype, w.filter, m)
    variant = ""
    if args.fused_filter:
        r.set_filter_fused(True)
        variant += ", VARIANT: fused (uncropped) filter + spectrum"
    if args.algorithm == "line":
        r.set_algorithm("line")
        variant += ", VARIANT: LineRec (direct line summation)"
    stream = torch.cuda.current_stream()

    def step():
        for ch in range(nchunks):
            r.recon(raw[ch], flat[ch], dark[ch], theta, out=out[ch * nzc:(ch + 1) * nzc], stream=stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    # ---- timed region: K steps, device-timed, per-kernel events inside
    r.set_profile(True)
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_ms = {k: 0.0 for k in r.STAGES}
    ncalls = 0
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        step()
        ms, nc = r.profile_collect()
        for k in ms:
            stage_ms[k] += ms[k]
        ncalls += nc
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop()
    r.set_profile(False)
    ms_total = max_over_ranks(ms_total, world, dev)
    ms_step = ms_total / args.steps
    voxels = float(nz_total) * n * n
    value = world * voxels / (ms_step * 1e-3) / 1e9

    # ---- end to end: pinned host -> pinned host through the three-stream pipeline
    e2e = None
    if not args.no_e2e:
        nz_e = min(nz_total, args.e2e_nz or nz_total)
        nz_e -= nz_e % nzc
        while True:
            try:
                raw_h = torch.empty((w.nproj, nz_e, n), dtype=torch.uint16).pin_memory()
                out_h = torch.empty((nz_e, n, n), dtype=out_dt).pin_memory()
                break
            except RuntimeError:          # not enough pinned host memory on this box: stream a shorter stack
                raw_h = out_h = None
                if nz_e <= 2 * nzc:
                    raise
                nz_e = (nz_e // 2) - (nz_e // 2) % nzc
        flat_h = torch.empty((nz_e, n), dtype=torch.float32).pin_memory()
        dark_h = torch.empty((nz_e, n), dtype=torch.float32).pin_memory()
        for ch in range(nz_e // nzc):
            raw_h.view(torch.int16)[:, ch * nzc:(ch + 1) * nzc].copy_(raw[ch].view(torch.int16))
            flat_h[ch * nzc:(ch + 1) * nzc].copy_(flat[ch])
            dark_h[ch * nzc:(ch + 1) * nzc].copy_(dark[ch])
        theta_h = torch.from_numpy(w.theta).pin_memory()
        for _ in range(min(args.warmup, 2)):
            r.recon_volume_host(raw_h, flat_h, dark_h, theta_h, out_h, nbuf=3)
        barrier()
        t0 = time.perf_counter()
        dev_ms = 0.0
        for _ in range(args.steps):
            _, ms = r.recon_volume_host(raw_h, flat_h, dark_h, theta_h, out_h, nbuf=3)
            dev_ms += ms
        barrier()
        wall = time.perf_counter() - t0
        wall = max_over_ranks(wall, world, dev)
        e2e = {"value": world * args.steps * float(nz_e) * n * n / wall / 1e9, "unit": "GVoxel/s",
               "h2d_bytes_per_step": int(raw_h.numel() * 2 + flat_h.numel() * 8 + w.nproj * 4),
               "d2h_bytes_per_step": int(out_h.numel() * out_h.element_size()),
               "slices": nz_e, "ms_per_step_wall": wall / args.steps * 1e3, "ms_per_step_device": dev_ms / args.steps,
               "pipeline": "3 streams, 3 buffer sets, pinned host", "timed": "wall clock, barrier+sync both sides"}
        del raw_h, out_h

    if rank != 0:
        return
    # ---- roofline of the dominant kernel.  Denominators are MEASURED: the HBM copy rate of MEASURED_PEAKS.json and the
    # fp32 FFMA / fp16 mma.sync issue rates of this GPU at this moment (tcp_measure_rates; both kernels are in the library).
    hbm_gbs, sm_max_mhz, which = _peaks()
    fp32_peak, hmma_peak = tcp.tcp_measure_rates()
    fused_s12 = half_store and not args.fused_filter and args.algorithm == "fourier"      # tcp.h: TCP_OPT_FUSE_NORMALIZE
    on_mma = half_store and n == 2048 and args.algorithm == "fourier"                     # tcp.h: TCP_OPT_TCFFT default
    model = stage_model(w, nzc, m, half_store, half_out, fused_s12)
    alu_peak = fp32_peak
    kernels = {}
    for k in model:
        t = stage_ms[k] / max(ncalls, 1) * 1e-3               # average launch duration, s
        kernels[k] = {"ms_per_launch": t * 1e3, "share": stage_ms[k] / max(sum(stage_ms.values()), 1e-9),
                      "GBps": model[k]["bytes"] / t / 1e9 if t > 0 else None,
                      "TFLOPps": model[k]["flops"] / t / 1e12 if t > 0 else None,
                      # fractions of roofline: algorithmic bytes against the measured HBM peak, algorithmic flops
                      # (5 N log2 N per transform, 4 per gridding tap, pair and sample) against the measured fp32 peak
                      "frac_hbm": model[k]["bytes"] / t / 1e9 / hbm_gbs if t > 0 else None,
                      "frac_alu": model[k]["flops"] / t / 1e12 / alu_peak if t > 0 else None}
    dom = max(model, key=lambda k: stage_ms[k])
    traffic = None           # DRAM bytes per launch of the dominant kernel from the committed ncu capture
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for ln in f.read().splitlines()[1:]:
                if ln.split(",")[0] == dom:
                    traffic = int(ln.split(",")[1])
    except Exception:
        pass
    names = dict(KERNEL_NAMES, **(KERNEL_NAMES_MMA if on_mma else ({"grid": "grid_mma_kernel"} if half_store else {})))
    # SURVEY 8(d) assigns the roofs: normalise and the 2D transform passes HBM, gridding "plain ALUs / smem / L2", the
    # row kernel "HBM if half2 math; else fp32 ALUs".  Both fractions are reported for every kernel; `bound` names the
    # roof assigned to the dominant one and `frac` is the fraction of that roof.  One departure from 8(d), fp16 storage
    # only: its gridding row describes a CUDA-core kernel; grid_mma_kernel multiplies on the tensor cores and replays
    # cached weights, its FMA pipe is 16 % busy and its DRAM traffic 53-56 % of peak (profiles/r2_kernels.md), so HBM is
    # the nearer roof and the one reported.  The fp32 tile kernel keeps "alu".
    assigned = {"normalize": "hbm", "rows": "alu", "grid": "hbm" if half_store else "alu", "ifft_cols": "hbm",
                "ifft_rows": "hbm"}[dom]
    roof = {"kernel": names.get(dom, dom), "bound": assigned,
            "achieved": kernels[dom]["TFLOPps"] if assigned == "alu" else kernels[dom]["GBps"],
            "peak": alu_peak if assigned == "alu" else hbm_gbs, "unit": "TFLOP/s" if assigned == "alu" else "GB/s",
            "frac": kernels[dom]["frac_alu"] if assigned == "alu" else kernels[dom]["frac_hbm"],
            "frac_hbm": kernels[dom]["frac_hbm"], "frac_alu": kernels[dom]["frac_alu"], "traffic": traffic,
            "peak_source": "fp32: tcp_measure_rates (FFMA issue rate measured in this run); HBM: MEASURED_PEAKS.json (%s)" % which,
            "peaks": {"hbm_GBps": hbm_gbs, "fp32_TFLOPps": fp32_peak, "hmma_f16_TFLOPps": hmma_peak,
                      "fp32_nominal_TFLOPps": 148 * 128 * 2 * sm_max_mhz * 1e6 / 1e12}}
    # whole path: SURVEY 8(d)'s algorithmic figure of the method (40 B/voxel at C4), whether or not a stage is fused away
    whole_bytes = sum(v["bytes"] for v in stage_model(w, nzc, m, half_store, half_out).values()) * nchunks
    if fused_s12:
        kernels["normalize"] = "fused into rows_kernel's loader (TCP_OPT_FUSE_NORMALIZE)"
    line = {
        "metric": "reconstructed GVoxel/s", "value": value, "unit": "GVoxel/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": {"f32": "f32", "f16": "f16", "f16_out32": "f16"}[w.dtype], "data": "synthetic",
        "config": {"workload": "%s: %d proj x %d x %d u16 -> %d^2 x %d voxels, %s, %d-slice chunks, %s, %s filter"
                   % (w.name, w.nproj, nz_total, n, n, nz_total, w.dtype, nzc, kernel_label(m), w.filter) + variant,
                   "gridding_kernel": kernel_label(m) + " (tcp_create_ex code %d)" % m,
                   "transforms": "radix-16 butterflies on mma.sync (TCP_OPT_TCFFT = 7)" if on_mma else "fp32 Stockham on the CUDA cores",
                   "l2": "inputs larger than L2 (%.1f GB raw resident in HBM)" % (raw.numel() * 2 / 1e9),
                   "replicas": world},
        "slices_per_s": world * nz_total / (ms_step * 1e-3),
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(args.steps * nchunks * r.launches_per_recon),
        "roofline": roof, "kernels": kernels,
        "whole_path": {"algorithmic_GB_per_step": whole_bytes / 1e9,
                       "hbm_frac": whole_bytes / (ms_step * 1e-3) / 1e9 / hbm_gbs, "hbm_peak_GBps": hbm_gbs},
    }
    if not args.no_cpu and world >= 1:
        cb, ref, (z0, ns) = cpu_baseline(w, made, m)
        # parity of the same slices, as a by-product (the gates live in tests/)
        ch0 = 0
        got = out[ch0 * nzc:ch0 * nzc + ns].float().cpu().numpy()
        err = [float(np.linalg.norm(got[z] - ref[z]) / np.linalg.norm(ref[z])) for z in range(ns)]
        if not variant:      # the oracle leg reconstructs the contract's default chain
            cb["parity_rel_l2_max"] = max(err)
        line["cpu_baseline"] = cb
    if args.configs and world == 1 and not variant:
        # the other configs of BASELINE.json, compute-only, in the same run (the headline config is the line itself)
        r.close()
        del raw, flat, dark, out
        torch.cuda.empty_cache()
        line["configs"] = []
        for name, dt in (("C1", None), ("C2", "f32"), ("C2", "f16"), ("C3", None), ("C5", None)):
            try:
                line["configs"].append(measure_config(name, dt, m, 2, 3, dev, hbm_gbs))
            except Exception as e:        # a config that does not fit this box is reported, not fatal
                line["configs"].append({"workload": name, "error": str(e)[:200]})
    print(json.dumps(line))


def run_reference(args, rank, world):
    """--impl reference: for this tier the reference arm is the CPU oracle, as it stands, on the
    box's host cores, each step a bounded sample (as many slices as host threads) of the same
    workload.  Rank 0 alone runs it."""
    if rank != 0:
        return
    import oracle as orc
    import synthgen as sg

    w = sg.make_workload(args.workload)
    m = args.m
    cores = orc.num_threads()
    ns = min(cores, w.nz_chunk)
    z0 = w.nz_total // 2
    rows = list(range(z0, z0 + ns))
    try:
        import torch
        use_gpu = torch.cuda.is_available()
    except Exception:
        use_gpu = False
    if use_gpu:       # manufacture the inputs on the GPU (minutes in numpy at 2048^2 x 500 ellipsoids)
        import torch
        r, ff, df = sg.make_counts_torch(w, rows, device="cuda")
        raw = r.view(torch.int16).cpu().numpy().view(np.uint16)
        flat = ff.view(torch.int16).cpu().numpy().view(np.uint16).astype(np.float32).mean(0, dtype=np.float32)
        dark = df.view(torch.int16).cpu().numpy().view(np.uint16).astype(np.float32).mean(0, dtype=np.float32)
    else:
        raw, _ = sg.make_counts(w, rows)
        flat, dark, _, _ = sg.make_flat_dark(w, rows)
    times = []
    for i in range(args.warmup + args.steps):
        if i >= 1 and i < args.warmup:
            continue                      # one untimed warm-up is enough for a CPU program
        t0 = time.perf_counter()
        orc.recon(raw, flat, dark, w.theta, w.center, w.filter, m, "grid")
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
    dt = float(np.mean(times))
    v = ns * w.n * w.n / dt / 1e9
    sample = "%d slices of %s per step (%d proj x %d px), oracle B_grid fp64" % (ns, w.name, w.nproj, w.n)
    print(json.dumps({
        "impl": "reference", "metric": "reconstructed GVoxel/s", "value": v, "unit": "GVoxel/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: %d proj x %d px, %s, %s filter (bounded sample)" % (w.name, w.nproj, w.n, kernel_label(m), w.filter)},
        "cpu_baseline": {"value": v, "unit": "GVoxel/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "GVoxel/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C4")
    ap.add_argument("--nz", type=int, default=0, help="override the number of slices in the volume")
    ap.add_argument("--nz-chunk", type=int, default=0)
    ap.add_argument("--m", type=int, default=16 + 2,
                    help="gridding kernel code of tcp_create_ex: 3, 4 = Gaussian half-width; 16 + 2 (default), 16 + 3 = Kaiser-Bessel")
    ap.add_argument("--no-configs", dest="configs", action="store_false",
                    help="skip the compute-only runs of the other BASELINE.json configs (the `configs` key)")
    ap.add_argument("--e2e-nz", type=int, default=0,
                    help="slices streamed through the host pipeline per step (0: the whole volume; halved if pinned host memory runs out)")
    ap.add_argument("--dtype", default="", choices=["", "f32", "f16", "f16_out32"],
                    help="override the workload's dtype (C2 is specified in both f32 and f16)")
    ap.add_argument("--fused-filter", action="store_true",
                    help="TCP_OPT_FILTER_FUSED: the uncropped one-transform reading of S3 + S4 (NOT the contract's default chain)")
    ap.add_argument("--algorithm", default="fourier", choices=["fourier", "line"],
                    help="backprojection operator: FourierRec (the contract's path) or LineRec (O(N^4) line summation)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
