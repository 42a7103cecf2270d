#!/usr/bin/env python
"""bench.py -- throughput of the BPM hot path on B200 (contract: see DESIGN.md "Measurement").

A "step" is one pass of the whole hot path over one batch of synthetic input: for the
default workload C4 (BASELINE.json configs[3], the one the metric is quoted on -- ~1000
multiplexed point sources through a 1024^3 float32 volume) that is bb_multiplex_psf
followed by bb_propagate over all 1024 slices, i.e. ONE full propagation.

  python bench.py [--gpus N] [--steps K] [--warmup W]          # our CUDA path
  python bench.py --impl reference ...                         # the CPU oracle, as it stands
  torchrun --nproc-per-node N bench.py --gpus N ...            # N independent replicas

Prints ONE JSON line (rank 0).  `value` is pixel-slices per second (Mvox/s) with all inputs
resident in HBM; `e2e` is the same metric through the host-buffer entry point with the
host<->device copies inside the timed region.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1706_02261_b200 import replicas, workloads as wl  # noqa: E402

# nominal FP32 rate of the non-tensor pipe: 148 SMs x 128 lanes x 2 flop x 1.965 GHz
# (/opt/skills/guides/B200_PROFILING.md: 148 SMs, clocks.max.sm 1965 MHz)
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
HBM_FALLBACK_GBS = 6650.0


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def committed_dram_traffic(workload: str):
    """DRAM bytes per launch of the persistent kernel from the committed ncu capture
    (profiles/dram_traffic.csv; the command that made it is in the file it names) -- but only if that
    capture was taken from the library source that is being timed now (its digest is in the row);
    otherwise None: a traffic figure of another build would be a claim about code that is not running."""
    import csv
    from paper_1706_02261_b200 import build
    p = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    try:
        digest = build._digest(build._sources())
        with open(p) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload and row.get("source_digest", "") == digest:
                    return int(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


def algorithmic_per_step(w: wl.Workload, per_field_intensity=False):
    """Algorithmic HBM bytes, L2 bytes and flops of ONE z-step."""
    npx = w.Nx * w.Ny
    B = w.batch
    hbm = 4 * npx + 4 * npx * (B if per_field_intensity else 1)
    l2 = 32 * npx * B + 8 * npx + hbm
    flops = (10 * npx * (math.log2(w.Nx) + math.log2(w.Ny)) + 40 * npx) * B
    return hbm, l2, flops


def roofline_fracs(w, dur_s, peaks, per_field=False):
    """T_roof / T and the three fractions for a propagation of w.Nz steps that took dur_s."""
    hbm_b, l2_b, flop = algorithmic_per_step(w, per_field)
    t = dur_s / w.Nz
    out = {"us_per_z_step": t * 1e6,
           "hbm_frac": hbm_b / (peaks["hbm"] * 1e9) / t,
           "alu_frac": flop / (FP32_PEAK_TFLOPS * 1e12) / t}
    if peaks.get("l2_copy"):
        out["l2_frac"] = l2_b / (peaks["l2_copy"] * 1e9) / t
        out["l2_frac_vs_read_peak"] = l2_b / (peaks["l2_read"] * 1e9) / t
        out["hbm_l2_roofline_frac"] = max(hbm_b / (peaks["hbm"] * 1e9), l2_b / (peaks["l2_copy"] * 1e9)) / t
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index: int):
        self.proc = None
        try:
            uuid = str(torch.cuda.get_device_properties(device_index).uuid)
            if not uuid.startswith("GPU-"):
                uuid = "GPU-" + uuid
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", uuid, "--query-gpu=" + self.FIELDS, "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for line in out.strip().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 8:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); pw.append(float(parts[2]))
            except ValueError:
                continue
            for n, v in zip(names, parts[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def make_inputs(w: wl.Workload, device):
    dn = wl.make_dn(w, device=device)
    f0 = wl.make_field(w)
    em = None
    if f0 is None:
        pos, ph, amp = wl.make_emitters(w)
        em = tuple(torch.from_numpy(a) for a in (pos, ph, amp))
    return dn, f0, em


# --------------------------------------------------------------------------------------------
def flush_l2(scratch):
    """A 256 MiB write between timed runs, so that a small dn volume is not found in the 126 MB L2."""
    scratch.add_(1.0)


def time_propagation(bb, w, dev, field0_fn, dn, nref, inten, flags=0, runs=10, warmup=3, scratch=None):
    """CUDA-event times (ms) of `runs` propagations of workload w, each from a fresh input field."""
    field = field0_fn()
    ts = []
    for i in range(warmup + runs):
        field = field0_fn(field)
        if scratch is not None:
            flush_l2(scratch)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        bb.propagate(field, dn, w.dx, w.dz, w.lam, w.n0, intensity=inten, nref=nref, flags=flags)
        b.record()
        torch.cuda.synchronize()
        if i >= warmup:
            ts.append(a.elapsed_time(b))
    return ts


def time_config(bb, dev, name, peaks, scratch, per_field=False, runs=10):
    """One entry of the `configs` array: a parity-test configuration timed the way SURVEY 8d asks
    (3 warm-ups, median and min of >= 10 runs, L2 flushed in between, plan and tables resident)."""
    if name == "P31":
        # the lateral grid of the paper's own runs (1024 x 2048 x 1024 voxels), a slab of 128 slices:
        # C4's recipe on 2048 x 1024 pixels -- 2048-point lines (class radix 8)
        import dataclasses
        w = dataclasses.replace(wl.config("C4"), name="P31", Nx=2048, Nz=128, n_cells=500)
    elif name.startswith("C4x"):
        # north_star item 4 at the headline size ("100s to 1000s ... PSFs ... within single, highly
        # multiplexed simulations", many such runs per sample): B multiplexed 1024 x 1024 fields through the shared
        # 1024^3 volume, summed intensity; field b = C4's emitters with their phases re-drawn from seed b
        import dataclasses
        w = dataclasses.replace(wl.config("C4"), name=name, batch=int(name[3:]))
    else:
        w = wl.config(name)
    dn, f0, em = make_inputs(w, dev)
    nref = bb.nref_from_dn(dn, w.n0, w.nref_slab).numpy()
    if em is not None:
        em_d = tuple(t.to(dev) for t in em)
        fields = []
        for b in range(w.batch):
            ph = em_d[1] if b == 0 else torch.from_numpy(
                np.random.default_rng(1000 + b).uniform(0, 2 * np.pi, size=em[1].shape).astype(np.float32)).to(dev)
            fields.append(bb.multiplex_psf(em_d[0], ph, em_d[2], w.NA, w.Nx, w.Ny, w.dx, w.lam))
        src = torch.stack(fields).contiguous()
    else:
        src = torch.from_numpy(f0).to(dev)

    def field0(buf=None):
        if buf is None:
            return src.clone()
        buf.copy_(src)
        return buf

    B = w.batch
    flags = bb.INTENSITY_PER_FIELD if per_field else 0
    inten = torch.empty(((B,) if per_field else ()) + (w.Nz, w.Ny, w.Nx), dtype=torch.float32, device=dev)
    ts = time_propagation(bb, w, dev, field0, dn, nref, inten, flags=flags, runs=runs, scratch=scratch)
    med, mn = statistics.median(ts), min(ts)
    units = float(w.Nx) * w.Ny * w.Nz * B
    out = {"workload": "%s%s: %d field(s) of %dx%d, %d z-slices%s" % (w.name, " per-field intensity" if per_field else "", B, w.Nx, w.Ny, w.Nz,
                                                                     ", %.1f GiB intensity out" % (inten.numel() * 4 / 2**30) if per_field else ""),
           "baseline_config": ("BASELINE.json configs[%d]" % w.index) if name != "P31" and not name.startswith("C4x")
                              else ("none: PAPER.md line 31 grid, C4 recipe" if name == "P31" else
                                    "none: BASELINE.json configs[3] volume and emitters, %d fields (north_star item 4)" % B),
           "us_per_field_z_step": med * 1e3 / w.Nz / B,
           "propagate_ms": med, "propagate_ms_min": mn, "runs": len(ts),
           "value": units / (med * 1e-3) / 1e6, "unit": "Mvox/s", "kernel": bb.last_kernel(),
           "roofline": roofline_fracs(w, med * 1e-3, peaks, per_field)}
    del inten, dn
    return out


def time_next_rows(bb, dev, peaks, runs=10):
    """The NEXT rows of SURVEY 8f, each timed on a C3/C4-sized input (median of `runs` after 3 warm-ups, CUDA events)
    with the roofline that bounds it: algorithmic bytes or flops over the measured duration."""
    def timed(fn):
        ts = []
        for i in range(3 + runs):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); fn(); b.record()
            torch.cuda.synchronize()
            if i >= 3:
                ts.append(a.elapsed_time(b))
        return statistics.median(ts)

    out = []
    hbm = peaks["hbm"]
    # NEXT-4 backward propagation: C4's grid and phantom recipe, 64 slices, n_ref slabs of 32
    w = wl.config("C4").with_nz(64)
    dn, _, em = make_inputs(w, dev)
    nref = bb.nref_from_dn(dn, w.n0, w.nref_slab).numpy()
    f = bb.multiplex_psf(*(t.to(dev) for t in em), w.NA, w.Nx, w.Ny, w.dx, w.lam)[None].contiguous()
    I = torch.empty((w.Nz, w.Ny, w.Nx), device=dev)
    for name, flags in (("forward, for comparison", 0), ("BB_BACKWARD", bb.BACKWARD)):
        ms = timed(lambda: bb.propagate(f, dn, w.dx, w.dz, w.lam, w.n0, intensity=I, nref=nref, flags=flags))
        out.append({"row": "NEXT-4", "what": "%s: 1024x1024, 64 slices" % name, "ms": ms, "kernel": bb.last_kernel(),
                    "roofline": roofline_fracs(w, ms * 1e-3, peaks)})
    # NEXT-1: refocus (one H-only step), through-focus stack (64 homogeneous steps with intensity), PSF tiles
    ms = timed(lambda: bb.refocus(f, w.dx, -6.4, w.lam, w.n0))
    out.append({"row": "NEXT-1", "what": "bb_refocus: 1024x1024, one signed step", "ms": ms,
                "note": "three phases of the persistent kernel (two grid barriers): latency-bound, %.1f us" % (ms * 1e3)})
    ms = timed(lambda: bb.propagate(f, None, w.dx, w.dz, w.lam, w.n0, intensity=I, flags=bb.HOMOGENEOUS, nz=w.Nz))
    wh = w
    out.append({"row": "NEXT-1", "what": "BB_HOMOGENEOUS through-focus stack: 1024x1024, 64 planes", "ms": ms,
                "roofline": roofline_fracs(wh, ms * 1e-3, peaks)})
    pos = em[0].to(dev)
    T = 32
    tiles = None
    def do_tiles():
        nonlocal tiles
        tiles = bb.extract_tiles(I, pos, w.dx, T)
    ms = timed(do_tiles)
    nbytes = 2 * pos.shape[0] * w.Nz * T * T * 4
    out.append({"row": "NEXT-1", "what": "bb_extract_tiles: %d emitters x 64 planes x 32x32 floats" % pos.shape[0], "ms": ms,
                "roofline": {"bound": "hbm", "achieved_gbs": nbytes / (ms * 1e-3) / 1e9, "peak_gbs": hbm,
                             "frac": nbytes / (ms * 1e-3) / 1e9 / hbm, "algorithmic_bytes": nbytes}})
    # NEXT-2: generators
    ms = timed(lambda: bb.lightsheet(1024, 1024, 0.1, 0.5, 1.33, 0.2, 25.6, device=dev))
    out.append({"row": "NEXT-2", "what": "bb_lightsheet: 1024x1024 (fill + one back-propagation step)", "ms": ms,
                "note": "latency-bound like bb_refocus"})
    ms = timed(lambda: bb.multiplex_annular(pos, em[1].to(dev), None, 0.55, 0.6, w.Nx, w.Ny, w.dx, w.lam))
    out.append({"row": "NEXT-2", "what": "bb_multiplex_annular: 1024 Bessel foci on 1024x1024, NA 0.55-0.6", "ms": ms})
    # NEXT-3: image formation, 1024x1024 source, 32x32 emitter grid, 32x32 tiles: 2 T^2 flop per pixel
    S = torch.rand((w.Ny, w.Nx), device=dev)
    psf = torch.rand((pos.shape[0], T, T), device=dev)
    ms = timed(lambda: bb.image_formation(S, pos, w.dx, psf))
    flop = 2.0 * w.Nx * w.Ny * T * T
    out.append({"row": "NEXT-3", "what": "bb_image_formation: 1024x1024, %d PSF tiles of 32x32" % pos.shape[0], "ms": ms,
                "roofline": {"bound": "alu", "achieved_tflops": flop / (ms * 1e-3) / 1e12, "peak_tflops": FP32_PEAK_TFLOPS,
                             "frac": flop / (ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS, "algorithmic_flop": flop,
                             "note": "includes the nearest-emitter map (1024 distance tests per pixel in double)"}})
    return out


def run_ours(args):
    from paper_1706_02261_b200 import binding as bb, build
    rank, local_rank, _ = replicas.env_world()
    world = replicas.init()
    if world != args.gpus:
        raise SystemExit("bench.py --gpus %d runs under a world of %d ranks: launch it with torchrun --nproc-per-node %d "
                         "(or let `python bench.py --gpus N` start the ranks itself)" % (args.gpus, world, args.gpus))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    dev = torch.device("cuda", local_rank if world > 1 else 0)
    torch.cuda.set_device(dev)
    build.build_library()
    bb.load()

    w = wl.config(args.workload)
    if args.nz:
        w = w.with_nz(args.nz)
    B, npx = w.batch, w.Nx * w.Ny
    flags = bb.LAUNCH_PER_PHASE if args.per_phase else 0
    dn, f0, em = make_inputs(w, dev)
    if em is not None:
        em_d = tuple(t.to(dev) for t in em)
        field = torch.empty((1, w.Ny, w.Nx), dtype=torch.complex64, device=dev)
    else:
        f0_d = torch.from_numpy(f0).to(dev)
        field = torch.empty_like(f0_d)
    inten = torch.empty((w.Nz, w.Ny, w.Nx), dtype=torch.float32, device=dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step(marks=None, nref=None):
        if em is not None:
            bb.multiplex_psf(em_d[0], em_d[1], em_d[2], w.NA, w.Nx, w.Ny, w.dx, w.lam, out=field[0])
        else:
            field.copy_(f0_d)
        if marks is not None:
            a = ev(); a.record()
        bb.propagate(field, dn, w.dx, w.dz, w.lam, w.n0, intensity=inten, nref=nref, flags=flags)
        if marks is not None:
            b = ev(); b.record()
            marks.append((a, b))

    # cold: the first pass of the hot path in this process -- plan, twiddle and propagator tables,
    # the n_ref helper (one pass over dn) and the propagation itself (SURVEY 8d "reported additionally cold")
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    nref = bb.nref_from_dn(dn, w.n0, w.nref_slab).numpy()
    step(nref=nref)
    torch.cuda.synchronize()
    cold_ms = (time.perf_counter() - t0) * 1e3

    for _ in range(args.warmup):
        step(nref=nref)
    torch.cuda.synchronize()
    bb.device_status()
    replicas.barrier()
    sampler = ClockSampler(dev.index) if rank == 0 else None
    launches0 = bb.launch_count()
    marks = []
    e0, e1 = ev(), ev()
    torch.cuda.synchronize()
    e0.record()
    for _ in range(args.steps):
        step(marks, nref=nref)
    e1.record()
    torch.cuda.synchronize()
    replicas.barrier()
    clocks = sampler.stop() if sampler else None
    launches = bb.launch_count() - launches0
    bb.device_status()
    t_local = e0.elapsed_time(e1) * 1e-3
    t = replicas.max_over_ranks(t_local)
    units = float(npx) * w.Nz * B * args.steps                 # pixel-slices this rank processed
    value = replicas.sum_over_ranks(units) / t / 1e6
    prop_all = [a.elapsed_time(b) for a, b in marks]           # the propagate call = the BPM kernel(s)
    prop_ms = statistics.mean(prop_all)
    kernel_name = bb.last_kernel()

    result = {
        "metric": "pixel-slices per second through the split-step BPM (ms per full propagation = ms_per_step)",
        "value": value, "unit": "Mvox/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": t / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "%s: %dx%d grid, %d z-slices, B=%d, dx=%g dz=%g lambda=%g n0=%g, %s, n_ref slabs of %d; "
                               "one step = %s + bb_propagate over all slices"
                               % (w.name, w.Nx, w.Ny, w.Nz, B, w.dx, w.dz, w.lam, w.n0,
                                  ("%dx%d emitters NA %.2g" % (w.emitters, w.emitters, w.NA)) if em is not None else w.field,
                                  w.nref_slab, "bb_multiplex_psf" if em is not None else "field reset"),
                   "baseline_config": "BASELINE.json configs[%d]" % w.index,
                   "parallelism": "replicas only (%d independent propagation(s), no collective)" % world,
                   "l2": "inputs larger than L2: %.2f GiB dn + %.2f GiB intensity streamed per step"
                         % (dn.numel() * 4 / 2**30, inten.numel() * 4 / 2**30),
                   "launch_mode": "per-phase kernels" if args.per_phase else "one persistent cooperative kernel per propagation",
                   "headline": bool(args.workload == "C4" and not args.nz)},
        "gpu_launches": int(launches),
        "propagate_ms": prop_ms, "propagate_ms_median": statistics.median(prop_all), "propagate_ms_min": min(prop_all),
        "cold_ms": cold_ms,
    }
    if clocks is not None:
        result["clocks"] = clocks
    if rank == 0:
        # fingerprints of the seeded inputs: the emitter arrays / initial fields in full, the dn volume by its
        # first and last slice (hashing 4 GiB would take longer than the measurement)
        import hashlib
        sha = lambda a: hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()[:16]
        fp = {"dn_first_slice": sha(dn[0].cpu().numpy()), "dn_last_slice": sha(dn[-1].cpu().numpy())}
        if em is not None:
            fp["emitters"] = sha(np.concatenate([t.numpy().ravel() for t in em]))
        else:
            fp["field"] = sha(f0)
        result["config"]["inputs_sha256_16"] = fp

    # ---- roofline of the dominant kernel (the persistent BPM kernel, one launch per propagation) ----
    hbm_b, l2_b, flop = algorithmic_per_step(w)
    hbm_peak, hbm_src = measured_peaks()
    peaks = {"hbm": hbm_peak}
    dur = prop_ms * 1e-3
    traffic = committed_dram_traffic(w.name if (not args.nz and B == 1) else "")
    traffic_note = ("ncu capture of this source digest (profiles/dram_traffic.csv)" if traffic is not None
                    else "null: no ncu capture of the library source being timed (profiles/dram_traffic.csv holds other digests)")
    alu_ach = flop * w.Nz / dur / 1e12
    hbm_ach = hbm_b * w.Nz / dur / 1e9
    t_step = dur / w.Nz
    t_hbm = hbm_b / (hbm_peak * 1e9)
    # fraction of the roofline = T_roof / T per z-step, T_roof = max(T_HBM, T_L2).  `roofline` is that bound
    # (the L2 one whenever the in-run L2 probe ran, as it binds on every grid: 6 x the HBM bytes at ~2 x the bandwidth);
    # the HBM and FP32 views follow as roofline_hbm / roofline_alu.
    result["roofline"] = {"bound": "hbm", "achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s",
                          "frac": t_hbm / t_step, "traffic": traffic, "traffic_source": traffic_note,
                          "kernel": kernel_name, "peak_source": hbm_src,
                          "algorithmic_bytes_per_launch": hbm_b * w.Nz, "us_per_z_step": t_step * 1e6,
                          "definition": "SURVEY 8d: T_roof / T per z-step, T_roof = max(T_HBM, T_L2); L2 probe not run: HBM bound only"}
    result["roofline_hbm"] = {"bound": "hbm", "achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s",
                              "frac": hbm_ach / hbm_peak, "traffic": traffic, "peak_source": hbm_src,
                              "algorithmic_bytes_per_launch": hbm_b * w.Nz}
    result["roofline_alu"] = {"bound": "alu", "achieved": alu_ach, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                              "frac": alu_ach / FP32_PEAK_TFLOPS,
                              "peak_source": "nominal FMA peak: 148 SM x 128 lanes x 2 x 1.965 GHz (DESIGN.md); the transforms are "
                                             "two-thirds additions, so the ceiling for this instruction mix is about half of it",
                              "algorithmic_flop_per_launch": flop * w.Nz}
    if rank == 0 and not args.no_probe:
        try:
            peaks["l2_copy"] = bb.probe_l2_bandwidth(32 << 20, 200, 0)
            peaks["l2_read"] = bb.probe_l2_bandwidth(32 << 20, 200, 1)
            fp32_meas = bb.probe_fp32(20000, False)
            l2_ach = l2_b * w.Nz / dur / 1e9
            t_l2 = l2_b / (peaks["l2_copy"] * 1e9)
            result["roofline_l2"] = {"bound": "l2", "achieved": l2_ach, "peak": peaks["l2_copy"], "unit": "GB/s",
                                     "frac": l2_ach / peaks["l2_copy"],
                                     "peak_read_only": peaks["l2_read"], "frac_vs_read_peak": l2_ach / peaks["l2_read"],
                                     "peak_source": "measured now: bb_probe_l2_bandwidth, 32 MiB resident, copy (half read, half "
                                                    "write, like the field's traffic) and read-only",
                                     "algorithmic_bytes_per_launch": l2_b * w.Nz}
            result["roofline_alu"]["peak_measured_fma_loop"] = fp32_meas
            mix = bb.probe_fp32(4000, 2)
            result["roofline_alu"]["peak_butterfly_mix"] = mix
            result["roofline_alu"]["frac_vs_mix_peak"] = alu_ach / mix
            result["roofline_alu"]["mix_note"] = ("bb_probe_fp32 mode 2: the kernel's own butterflies of a 1024-point phase from registers, "
                                                  "no memory, at the kernel's occupancy, in SURVEY 8d's flop count; T_ALU at that rate = "
                                                  "%.2f us per z-step" % (flop / (mix * 1e12) * 1e6))
            t_roof = max(t_hbm, t_l2)
            if t_l2 >= t_hbm:
                result["roofline"].update({"bound": "l2", "achieved": l2_ach, "peak": peaks["l2_copy"],
                                           "peak_source": result["roofline_l2"]["peak_source"],
                                           "algorithmic_bytes_per_launch": l2_b * w.Nz})
            result["roofline"].update({"frac": t_roof / t_step, "t_roof_us_per_z_step": t_roof * 1e6,
                                       "t_hbm_us_per_z_step": t_hbm * 1e6, "t_l2_us_per_z_step": t_l2 * 1e6,
                                       "definition": "SURVEY 8d: T_roof / T per z-step, T_roof = max(T_HBM, T_L2); `traffic` is the "
                                                     "kernel's DRAM bytes per launch (ncu), to be held against roofline_hbm"})
            result["hbm_l2_roofline_frac"] = t_roof / t_step             # the same number (key kept from rounds 1-2)
        except Exception as e:                                            # noqa: BLE001
            result["roofline_l2"] = {"error": str(e)}

    # ---- end to end through the host-buffer entry point ----
    if not args.no_e2e:
        fh = torch.empty((B, w.Ny, w.Nx), dtype=torch.complex64).pin_memory()
        dnh = torch.empty(dn.shape, dtype=torch.float32).pin_memory()
        dnh.copy_(dn)
        Ih = torch.empty(inten.shape, dtype=torch.float32).pin_memory()
        if em is not None:
            em_h = tuple(t.pin_memory() for t in em)
        else:
            f0_h = torch.from_numpy(f0).pin_memory()
        h2d = dnh.numel() * 4 + fh.numel() * 8 + (sum(t.numel() * 4 for t in em) if em is not None else 0)
        d2h = Ih.numel() * 4 + fh.numel() * 8 + (fh.numel() * 8 if em is not None else 0)

        def e2e_step():
            if em is not None:
                d = tuple(t.to(dev, non_blocking=True) for t in em_h)
                bb.multiplex_psf(d[0], d[1], d[2], w.NA, w.Nx, w.Ny, w.dx, w.lam, out=field[0])
                fh.copy_(field, non_blocking=True)
                torch.cuda.synchronize()
            else:
                fh.copy_(f0_h)
            bb.propagate(fh, dnh, w.dx, w.dz, w.lam, w.n0, intensity=Ih, nref=nref, flags=flags)

        n_e2e = max(1, min(args.steps, args.e2e_steps))
        e2e_step()
        torch.cuda.synchronize()
        replicas.barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            e2e_step()
        torch.cuda.synchronize()
        t_e2e = replicas.max_over_ranks(time.perf_counter() - t0)
        replicas.barrier()
        e2e_val = replicas.sum_over_ranks(float(npx) * w.Nz * B * n_e2e) / t_e2e / 1e6
        same = torch.equal(Ih[-1], inten[-1].cpu())
        result["e2e"] = {"value": e2e_val, "unit": "Mvox/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                         "steps": n_e2e, "ms_per_step": t_e2e / n_e2e * 1e3, "host_memory": "pinned",
                         "api": "bb_propagate_host (dn streamed in z-chunks, intensity streamed back)",
                         "matches_device_path": bool(same)}
        del dnh, Ih

    # ---- the oracle on this box's host cores (reported baseline, rank 0, N = 1 only) ----
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        result["cpu_baseline"] = oracle_sample(w, dn, f0, em, nref, budget_s=args.cpu_seconds)
        try:
            result["cpu_baseline"]["one_thread"] = oracle_sample(w, dn, f0, em, nref, budget_s=args.cpu_seconds / 2, threads=1)
        except Exception as e:                                            # noqa: BLE001
            result["cpu_baseline"]["one_thread"] = {"error": str(e)}

    # ---- the other configurations of BASELINE.json (parity-test cases), timed for information ----
    if rank == 0 and world == 1 and args.workload == "C4" and not args.nz and not args.no_configs:
        del dn, inten
        torch.cuda.empty_cache()
        scratch = torch.zeros(64 << 20, dtype=torch.float32, device=dev)          # 256 MiB
        cfgs = []
        for name, per_field in (("C1", False), ("C2", False), ("C3", False), ("C5", False), ("C5", True), ("P31", False),
                                ("C4x4", False), ("C4x8", False)):
            try:
                cfgs.append(time_config(bb, dev, name, peaks, scratch, per_field=per_field))
            except Exception as e:                                        # noqa: BLE001
                cfgs.append({"workload": name, "error": str(e)})
        result["configs"] = cfgs
        try:
            result["next_rows"] = time_next_rows(bb, dev, peaks)
        except Exception as e:                                            # noqa: BLE001
            result["next_rows"] = [{"error": str(e)}]
        result["configs_note"] = ("3 warm-ups, median (propagate_ms) and min of 10 propagations each, 256 MiB written between runs; "
                                  "C1-C3 are latency-bound (T_roof is sub-microsecond per step): their fractions are for information")

    if rank == 0:
        print(json.dumps(result))
    replicas.shutdown()


def run_trace(args):
    """Per-phase timeline of the persistent kernel (bb_probe_trace) on the first N z-steps of the
    workload: medians over CTAs and steps of work / arrive / staging / wait, per phase kind."""
    from paper_1706_02261_b200 import binding as bb, build
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    build.build_library()
    bb.load()
    w = wl.config(args.workload).with_nz(args.trace)
    dn, f0, em = make_inputs(w, dev)
    nref = bb.nref_from_dn(dn, w.n0, w.nref_slab).numpy()
    if em is not None:
        field0 = bb.multiplex_psf(*(t.to(dev) for t in em), w.NA, w.Nx, w.Ny, w.dx, w.lam)[None]
    else:
        field0 = torch.from_numpy(f0).to(dev)
    inten = torch.empty((w.Nz, w.Ny, w.Nx), dtype=torch.float32, device=dev)
    grid = torch.cuda.get_device_properties(dev).multi_processor_count
    phases = 2 * w.Nz + 1
    buf = torch.zeros((phases, grid, 6), dtype=torch.int64, device=dev)
    for it in range(3):
        field = field0.clone()
        if it == 2:
            bb.probe_trace(buf)
        bb.propagate(field, dn, w.dx, w.dz, w.lam, w.n0, intensity=inten, nref=nref)
        torch.cuda.synchronize()
    bb.probe_trace(None)
    kernel = bb.last_kernel()
    cluster = "bpmc_kernel" in kernel                         # grid = one cluster: the stamps of its CTAs come first
    if cluster:
        grid = int(kernel.split("<")[1].split(",")[2])
    t = buf.cpu().numpy().astype(np.float64).reshape(-1)[: phases * grid * 6].reshape(phases, grid, 6)
    if not t[1:-1, :, 4].all():
        raise SystemExit("no trace recorded: this shape / batch does not run the traced kernel")
    # SM cycles per microsecond from the global timer (ns) at release of consecutive phases
    cyc_per_us = np.median((t[2:-1, :, 4] - t[1:-2, :, 4]) / np.maximum(t[2:-1, :, 5] - t[1:-2, :, 5], 1.0)) * 1e3
    out = {"workload": w.name, "z_steps": w.Nz, "kernel": kernel, "sm_cycles_per_us": cyc_per_us,
           "unit": "us (median over CTAs and steps)"}
    # grid kernels: work / barrier arrive / staging of the next factors / barrier wait;
    # cluster kernel: transforms / send to the owners' shared memory / arrive + staging / wait
    names = ("transforms", "send", "staging", "wait") if cluster else ("work", "arrive", "staging", "wait")
    for name, sel in (("row_phase", slice(2, phases - 1, 2)), ("column_phase", slice(1, phases - 1, 2))):
        p = t[sel]
        seg = {names[i]: p[:, :, i + 1] - p[:, :, i] for i in range(4)}
        seg["total"] = p[:, :, 4] - p[:, :, 0]
        out[name] = {k: float(np.median(v) / cyc_per_us) for k, v in seg.items()}
        out[name][names[0] + "_max_over_ctas"] = float(np.median(seg[names[0]].max(axis=1)) / cyc_per_us)
    rel = t[1:-1, :, 5].max(axis=1)
    out["us_per_z_step"] = float(np.median(rel[2:] - rel[:-2]) * 1e-3)
    print(json.dumps(out))


def oracle_sample(w, dn, f0, em, nref, budget_s=15.0, slices=None, threads=None):
    """Times the oracle, as it stands, on the first `slices` z-slices of the workload (threads: OpenMP
    thread count for this sample, None = all cores of the affinity mask)."""
    import ctypes
    import oracle
    oracle.build()
    ncores = oracle.num_threads()
    if threads is not None:
        gomp = ctypes.CDLL("libgomp.so.1")
        gomp.omp_set_num_threads(int(threads))
        try:
            r = oracle_sample(w, dn, f0, em, nref, budget_s=budget_s, slices=slices)
        finally:
            gomp.omp_set_num_threads(ncores)
        r["cores"] = int(threads)
        return r
    if f0 is None:
        pos, ph, amp = (t.numpy() for t in em)
        u0 = oracle.multiplex_psf(pos, ph, amp, w.NA, w.Nx, w.Ny, w.dx, w.lam).astype(np.complex64)
    else:
        u0 = f0[0]
    dn0 = dn[:1].cpu().numpy()
    oracle.propagate_stream(u0, dn0, w.dx, w.dz, w.lam, w.n0, nref=nref[:1])          # warm-up (thread pool, caches)
    t0 = time.perf_counter()
    oracle.propagate_stream(u0, dn0, w.dx, w.dz, w.lam, w.n0, nref=nref[:1])
    t1 = max(time.perf_counter() - t0, 1e-4)
    if slices is None:
        slices = int(min(w.Nz, max(4, budget_s / t1)))
    dns = dn[:slices].cpu().numpy()
    t0 = time.perf_counter()
    oracle.propagate_stream(u0, dns, w.dx, w.dz, w.lam, w.n0, nref=nref[:slices])
    dt = time.perf_counter() - t0
    return {"value": w.Nx * w.Ny * slices / dt / 1e6, "unit": "Mvox/s", "cores": oracle.num_threads(), "kind": "oracle",
            "sample": "first %d of %d z-slices of %s, one field, double precision, %.1f s" % (slices, w.Nz, w.name, dt),
            "seconds": dt, "slices": slices}


# --------------------------------------------------------------------------------------------
def run_reference(args):
    """The reference arm for this tier is the oracle (there is no reference code): rank 0 only."""
    rank, _, world = replicas.env_world()
    if rank != 0:
        return
    import oracle
    oracle.build()
    w = wl.config(args.workload)
    if args.nz:
        w = w.with_nz(args.nz)
    # bounded sample: S slices per step such that warmup + steps stay within ~2 minutes
    total_steps = args.steps + args.warmup
    probe = w.with_nz(2)
    dn_p, f0, em = make_inputs(probe, "cpu")
    nref_p = oracle.nref_from_dn(dn_p.numpy(), w.n0, w.nref_slab)
    r = oracle_sample(probe, dn_p, f0, em, nref_p, slices=2)
    per_slice = r["seconds"] / 2
    S = int(min(w.Nz, max(2, (100.0 / total_steps) / per_slice)))
    ws = w.with_nz(S)
    dn, f0, em = make_inputs(ws, "cpu")
    nref = oracle.nref_from_dn(dn.numpy(), w.n0, w.nref_slab)
    times = []
    for i in range(total_steps):
        r = oracle_sample(ws, dn, f0, em, nref, slices=S)
        if i >= args.warmup:
            times.append(r["seconds"])
    dt = sum(times)
    value = w.Nx * w.Ny * S * len(times) / dt / 1e6
    sample = "each step = first %d of %d z-slices of %s (bounded sample), one field" % (S, w.Nz, w.name)
    print(json.dumps({
        "impl": "reference",
        "metric": "pixel-slices per second through the split-step BPM (ms per full propagation = ms_per_step)",
        "value": value, "unit": "Mvox/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / len(times) * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s (oracle, CPU): %s" % (w.name, sample), "baseline_config": "BASELINE.json configs[%d]" % w.index},
        "cpu_baseline": {"value": value, "unit": "Mvox/s", "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "Mvox/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--workload", default="C4", choices=sorted(wl.CONFIGS))
    ap.add_argument("--nz", type=int, default=0, help="use only the first NZ slices (profiling; not the headline number)")
    ap.add_argument("--per-phase", action="store_true", help="one kernel launch per half-step (diagnostic)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-probe", action="store_true")
    ap.add_argument("--no-batch", "--no-configs", dest="no_configs", action="store_true",
                    help="skip the timing of the other BASELINE.json configurations (C1-C3, C5 summed and per-field)")
    ap.add_argument("--trace", type=int, default=0, metavar="N",
                    help="print the per-phase timeline of the persistent kernel over the first N z-steps and exit")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours" and not args.nz:
        args.warmup = 3                                   # timing rule: at least 3 warm-up steps
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` without a launcher: start the N ranks ourselves (one process per GPU)
        import socket
        with socket.socket() as so:
            so.bind(("127.0.0.1", 0))
            port = so.getsockname()[1]
        os.execvp(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
                                   "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    if args.trace:
        run_trace(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
