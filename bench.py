#!/usr/bin/env python
"""bench.py -- narrow-band SDF throughput of the CSC hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C4] [--impl ours|reference]

A "step" is one pass of the whole hot path over one mesh+grid: sdf_create (A0-A4: weld,
edge table, pseudonormals, classes) + sdf_compute (A5-A8: extrude, scan-convert, evaluate +
min-combine, sign + emit) through the C ABI.  Default workload: BASELINE.json config C4
(3,996,000-triangle star surface, 1024^3 grid, band 2h), the one north_star quotes the
target on.  `value` = populated band cells / step time with the soup and both output grids
resident in HBM; `e2e` = same metric with HOST buffers (pinned soup in, pinned grids out).

The path does not shard (north_star: one GPU): --gpus N under torchrun runs N independent
replicas, no collective on the data path ("replicas only").

--impl reference times the CPU oracle (oracle/) on the host cores on a bounded z-slab
sample of the same workload.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1903_00353_b200 import workloads as W  # noqa: E402

METRIC = "narrow_band_sdf_cells_per_s"
UNIT = "band cells/s"
L2_BYTES = 126 * 1024 * 1024
# dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed `ncu --set full` captures:
# rows "config,kernel,dram_bytes_read,dram_bytes_write,source" (profiles/kernel_traffic.md names the commands)
TRAFFIC_CSV = os.path.join("profiles", "kernel_traffic.csv")
FLOP_PER_PAIR = 40.0          # <= 5 half-plane tests + one feature distance per (cell, polyhedron) pair

# stage -> (the kernel that dominates it, what its algorithmic bytes are); F triangles, N cells, E edges, V vertices
STAGE_KERNEL = {
    "fill": ("fill_tma_kernel", "A8a dense write of both grids, cp.async.bulk shared->global: 8 B per cell"),
    "evaluate": ("evaluate_small_kernel", "A5-A7: every feature record read once (36 B per face, 64 B per edge, 32 B per vertex)"),
    "emit": ("emit_bricks_kernel", "A8b: 8 B of packed scratch read + 8 B written per cell of an active brick"),
    "ingest_weld": ("ingest_weld_kernel", "A0/A1: the soup read once and written once in the internal order, 72 B per triangle"),
    "edges": ("tri_geom_kernel", "A2/A3: the soup read once, 36 B per triangle"),
    "vertices": ("vertex_cone_kernel", "A3/A4: the soup read once, 36 B per triangle"),
    "clip_scan": ("brick_mark_kernel", "A6a: the soup read once, 36 B per triangle"),
    "clear": ("cudaMemsetAsync", "scratch reset: 8 B per cell of an active brick"),
}


# --------------------------------------------------------------------------------------- #
# helpers
# --------------------------------------------------------------------------------------- #
def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", os.environ.get("BENCH_SMI_MS", "20")],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is not None:
            self.p.terminate()
            try:
                self.p.wait(timeout=5)
            except Exception:
                self.p.kill()
        try:
            self.f.flush()
            with open(self.f.name) as f:
                rows = [r.strip().split(", ") for r in f if r.strip()]
            os.unlink(self.f.name)
        except Exception:
            rows = []
        sm, smax, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1]))
                smax.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(n)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(smax)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def kernel_traffic(config, kernel):
    """(dram bytes per launch, where from) out of the committed ncu summary, or (None, None)."""
    path = os.path.join(ROOT, TRAFFIC_CSV)
    if not os.path.exists(path):
        return None, None
    with open(path) as f:
        for line in f:
            r = [c.strip() for c in line.split(",")]
            if len(r) >= 5 and r[0] == config and r[1] == kernel:
                try:
                    return float(r[2]) + float(r[3]), "%s (%s)" % (TRAFFIC_CSV, r[4])
                except ValueError:
                    continue
    return None, None


def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def sample_slab(w, nslices):
    """Bounded sample of the workload for the oracle: `nslices` z-slices starting one brick below the lowest slice
    the band reaches -- at C4 that slab holds the south pole (a valence-2000 fan of slivers, the expensive part for
    the oracle) and the surface up to the equator's neighbourhood, not just the easy middle of the mesh."""
    nx, ny, nz = w.dims
    ns = min(nslices, nz)
    zmin = float(w.soup[:, :, 2].min())
    k0 = int(np.floor((zmin - w.band - w.origin[2]) / w.h)) - 8
    k0 = max(0, min(k0, nz - ns))
    return w.crop((0, 0, k0), (nx, ny, ns)), "z-slab k in [%d,%d) of %d slices (from the lowest slice of the band upwards), full mesh" % (k0, k0 + ns, nz)


# --------------------------------------------------------------------------------------- #
# reference arm: the CPU oracle, as it stands, on the host cores
# --------------------------------------------------------------------------------------- #
def time_oracle(w, nslices, steps, warmup, threads=None):
    import oracle
    oracle.build()
    cores = threads or oracle.default_threads()
    t0 = time.perf_counter()
    om = oracle.Mesh(w.soup)
    build_s = time.perf_counter() - t0
    c, what = sample_slab(w, nslices)
    cells = 0
    for _ in range(warmup):
        om.sdf(c.origin, c.h, c.dims, c.band, cores)
    t0 = time.perf_counter()
    for _ in range(steps):
        d, _t = om.sdf(c.origin, c.h, c.dims, c.band, cores)
    dt = (time.perf_counter() - t0) / max(steps, 1)
    cells = int(np.isfinite(d).sum())
    return {"value": cells / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": what + "; %d band cells per step in %.2f s; one-off connectivity build %.1f s not included"
                      % (cells, dt, build_s),
            "build_s": build_s, "s_per_step": dt, "band_cells": cells}


def run_reference(args):
    rank, _lr, world = dist_env()
    if rank != 0:
        return
    w = load_workload(args)
    r = time_oracle(w, args.ref_slices, args.steps, args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["s_per_step"] * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, args),
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def load_workload(args):
    """BASELINE.json config, optionally with another band width (exploration only: the headline
    numbers are the configs as BASELINE.json states them)."""
    import dataclasses
    w = W.config(args.config)
    if args.band_cells:
        w = dataclasses.replace(w, band=float(args.band_cells) * w.h)
    return w


def workload_config(w, args):
    nx, ny, nz = w.dims
    return {"workload": "%s: %d triangles, grid %dx%dx%d, h=%g, band %gh (BASELINE.json configs[%d])"
                        % (w.name, w.ntri, nx, ny, nz, w.h, w.band / w.h, W.CONFIG_NAMES.index(w.name)),
            "triangles": w.ntri, "grid": [nx, ny, nz], "band_cells": w.band / w.h,
            "parallelism": ("z-slabs: every rank builds the mesh and computes 1/%d of the grid, no exchange"
                            % (args.zslab_parts or args.gpus)) if (args.zslab or args.zslab_parts) else
                           "replicas only (the path does not shard)" if args.gpus > 1 else "1 GPU",
            "call": "sdf_transform (= sdf_create + sdf_compute in one call)"
                    if not (getattr(args, "split_calls", False) or args.zslab or args.zslab_parts) else "sdf_create + sdf_compute",
            "l2": "no flush needed: each step streams %.2f GB of output > %d MB L2"
                  % (8.0 * w.ncells / 1e9, L2_BYTES >> 20)}


# --------------------------------------------------------------------------------------- #
# our arm: the CUDA path through the C ABI
# --------------------------------------------------------------------------------------- #
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1903_00353_b200 import binding as B

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank % torch.cuda.device_count())
    dev = torch.device("cuda", torch.cuda.current_device())
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    w = load_workload(args)
    nx, ny, nz = w.dims
    # --zslab: every rank builds the whole mesh and computes one
    # z-slab of the grid (strong scaling, no data-path collective); --zslab-parts / --zslab-part time
    # one slab of a P-way split on a single GPU
    zslab = None
    if args.zslab or args.zslab_parts:
        parts = args.zslab_parts or world
        part = args.zslab_part if args.zslab_parts else rank
        k0, nk = B.sdf_zslab(nz, part, parts)
        if nk == 0:
            raise SystemExit("z-slab %d of %d of %d slices is empty" % (part, parts, nz))
        zslab = {"part": part, "parts": parts, "k0": k0, "nk": nk}
        full_dims, full_origin = w.dims, w.origin
        # the slab as a grid of its own (include/sdf.h, sdf_compute_zslab: origin_z + k0*h in double, rounded once)
        oz = float(np.float32(np.float64(np.float32(w.origin[2])) + k0 * np.float64(np.float32(w.h))))
        w = W.Workload(w.name, w.soup, (w.origin[0], w.origin[1], oz), w.h, (nx, ny, nk), w.band, dict(w.meta))
        nx, ny, nz = w.dims
    N = w.ncells
    soup_host = torch.from_numpy(np.ascontiguousarray(w.soup)).pin_memory()
    soup_dev = soup_host.to(dev)
    dist_out = torch.empty((nz, ny, nx), dtype=torch.float32, device=dev)
    tri_out = torch.empty((nz, ny, nx), dtype=torch.int32, device=dev)
    need_flush = 8 * N < 2 * L2_BYTES
    flush_buf = torch.empty(2 * L2_BYTES, dtype=torch.uint8, device=dev) if need_flush else None
    stream = torch.cuda.current_stream()

    def step_device():
        if not zslab and not args.split_calls:
            # one call for the whole path (SDF_PREFILL_AT picks where the sentinel fill starts: DESIGN.md 9b)
            return B.sdf_transform(soup_dev, w.origin, w.h, w.dims, w.band, dist_out, tri_out, stream=stream)[0]
        m = B.sdf_create(soup_dev, stream=stream)
        if zslab:
            B.sdf_compute_zslab(m, full_origin, w.h, full_dims, w.band, zslab["part"], zslab["parts"], dist_out, tri_out,
                                stream=stream)
        else:
            B.sdf_compute(m, w.origin, w.h, w.dims, w.band, dist_out, tri_out, stream=stream)
        return m

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- warm-up (also sizes torch's caching allocator pools)
    for _ in range(max(args.warmup, 0)):
        step_device().destroy()
    # ---- timed: K steps, device-resident inputs and outputs
    # only the dense writer (the kernel `roofline` is quoted on) is instrumented inside the timed steps: two event
    # records on the library's side stream; the full stage breakdown comes from a separate pass below
    B.sdf_enable_timing(2)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    fill_sum, stats = 0.0, None
    clocks = ClockSampler(torch.cuda.current_device())
    barrier()
    clocks.start()
    l0 = B.sdf_launch_count()
    for i in range(args.steps):
        if flush_buf is not None:
            flush_buf.zero_()
        ev[i][0].record(stream)
        m = step_device()
        ev[i][1].record(stream)
        fill_sum += B.sdf_get_timings(m)["fill"]         # synchronises the stream
        if i == args.steps - 1:
            stats = B.sdf_stats(m)
        m.destroy()
    barrier()
    launches = B.sdf_launch_count() - l0
    clk = clocks.stop()
    # ---- stage breakdown (not part of the timed region): a few more steps with every stage instrumented
    B.sdf_enable_timing(1)
    stage_sum, nbr = {}, max(1, min(args.steps, args.breakdown_steps))
    for _ in range(nbr):
        if flush_buf is not None:
            flush_buf.zero_()
        m = step_device()
        for k, v in B.sdf_get_timings(m).items():
            stage_sum[k] = stage_sum.get(k, 0.0) + v
        m.destroy()
    B.sdf_enable_timing(0)
    # ---- host wall clock per step: K more steps back to back, nothing instrumented, one synchronisation at the end
    # (the timed loop above reads the fill's events after every step, which drains the stream each time)
    barrier()
    t_wall = time.perf_counter()
    for _ in range(args.steps):
        if flush_buf is not None:
            flush_buf.zero_()
        step_device().destroy()
    barrier()
    t_wall = time.perf_counter() - t_wall
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    ms_per_step = total_ms / args.steps
    band_cells = int(stats["band_cells"])
    total_cells = world * band_cells
    if zslab and world > 1:                       # the slabs differ: sum what the ranks computed
        t = torch.tensor([band_cells], dtype=torch.int64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        total_cells = int(t.item())
    value = total_cells / (ms_per_step * 1e-3)

    # ---- end to end: HOST buffers through the C ABI (H2D of the soup, D2H of both grids)
    e2e = None
    if not args.no_e2e:
        dist_host = torch.empty((nz, ny, nx), dtype=torch.float32, pin_memory=True)
        tri_host = torch.empty((nz, ny, nx), dtype=torch.int32, pin_memory=True)
        soup_np = soup_host.numpy()

        def step_host():
            m = B.sdf_create(soup_np, stream=stream)                 # host pointer: copied by the library
            B.sdf_compute_host(m, w.origin, w.h, w.dims, w.band, dist_host, tri_host, stream=stream)
            m.destroy()

        step_host()
        ne = max(1, min(args.steps, args.e2e_steps))
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(ne):
            step_host()
        e1.record(stream)
        barrier()
        e_ms = e0.elapsed_time(e1) / ne
        if world > 1:
            t = torch.tensor([e_ms], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e_ms = float(t.item())
        assert int(torch.isfinite(dist_host).sum()) == band_cells
        e2e = {"value": total_cells / (e_ms * 1e-3), "unit": UNIT, "ms_per_step": e_ms, "steps": ne,
               "h2d_bytes_per_step": int(soup_host.numel() * 4), "d2h_bytes_per_step": int(8 * N),
               "note": "dense grids to the host: the 8 B per cell over PCIe are the floor of this contract"}
        del dist_host, tri_host
        # the same band in band-sparse storage (sdf_compute_sparse_host): only the bricks the band reaches cross PCIe,
        # no dense grid is filled or copied -- what a consumer that keeps a narrow band anyway would call
        if not zslab:
            m = B.sdf_create(soup_np, stream=stream)
            nb = B.sdf_brick_count(m, w.origin, w.h, w.dims, w.band, stream=stream)
            m.destroy()
            hi = torch.empty((nb + 64,), dtype=torch.int32).pin_memory()
            hd = torch.empty((nb + 64, 512), dtype=torch.float32).pin_memory()
            ht = torch.empty((nb + 64, 512), dtype=torch.int32).pin_memory()

            def step_sparse():
                m = B.sdf_create(soup_np, stream=stream)
                n = B.sdf_compute_sparse(m, w.origin, w.h, w.dims, w.band, hi, hd, ht, stream=stream)[0]
                m.destroy()
                return n

            step_sparse()
            barrier()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(max(ne, 5)):
                nbr_s = step_sparse()
            e1.record(stream)
            barrier()
            s_ms = e0.elapsed_time(e1) / max(ne, 5)
            assert int(torch.isfinite(hd[:nbr_s]).sum()) == band_cells
            e2e["sparse"] = {"value": total_cells / (s_ms * 1e-3), "unit": UNIT, "ms_per_step": s_ms, "bricks": int(nbr_s),
                             "h2d_bytes_per_step": int(soup_host.numel() * 4), "d2h_bytes_per_step": int(nbr_s) * (4 + 2 * 2048),
                             "call": "sdf_create(host soup) + sdf_compute_sparse_host(pinned brick buffers)"}
            del hi, hd, ht

    # ---- SURVEY.md 8(f) NEXT-1 (not part of the step): interior fill by axis sweeps on the last result
    fill_int = None
    if args.fill_interior and rank == 0:
        keep = dist_out.clone()
        tms = []
        for _ in range(3):
            dist_out.copy_(keep)
            torch.cuda.synchronize()
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record(stream)
            B.sdf_fill_interior(dist_out, w.band, stream=stream)
            f1.record(stream)
            torch.cuda.synchronize()
            tms.append(f0.elapsed_time(f1))
        filled = int((torch.isfinite(dist_out) & ~torch.isfinite(keep)).sum())
        fb = 4.0 * N + 4.0 * filled                       # read every cell once, write the interior once
        fill_int = {"ms": min(tms), "cells_filled": filled, "algorithmic_bytes": fb,
                    "achieved_gbs": fb / (min(tms) * 1e-3) / 1e9, "bound": "hbm",
                    "note": "three in-place sweeps: x reads the grid, y and z skip the 32-cell segments x left blank"}
        del keep

    # ---- SURVEY.md 8(f) NEXT-2 (not part of the step): closest points of the last result
    cpt = None
    if args.closest_points and rank == 0:
        m = step_device()
        cp_out = torch.empty((nz, ny, nx, 3), dtype=torch.float32, device=dev)
        tms = []
        for _ in range(3):
            torch.cuda.synchronize()
            f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            f0.record(stream)
            B.sdf_closest_points(m, w.origin, w.h, w.dims, tri_out, cp_out, stream=stream)
            f1.record(stream)
            torch.cuda.synchronize()
            tms.append(f0.elapsed_time(f1))
        m.destroy()
        cb = 16.0 * N                                      # 4 B of id read + 12 B of point written per cell
        cpt = {"ms": min(tms), "algorithmic_bytes": cb, "achieved_gbs": cb / (min(tms) * 1e-3) / 1e9, "bound": "hbm"}
        del cp_out

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel
    peak, peak_src = measured_peaks()
    stage_ms = {k: v / nbr for k, v in stage_sum.items()}
    dom = max(stage_ms, key=stage_ms.get)
    F_, E_, V_ = w.ntri, 3 * w.ntri // 2, int(stats["V"])
    bricks = int(stats["bricks_active"])
    alg_bytes = {"fill": 8.0 * N, "evaluate": 36.0 * F_ + 64.0 * E_ + 32.0 * V_, "emit": 16.0 * 512 * bricks,
                 "ingest_weld": 72.0 * F_, "edges": 36.0 * F_, "vertices": 36.0 * F_, "clip_scan": 36.0 * F_,
                 "clear": 8.0 * 512 * bricks}
    kern, what = STAGE_KERNEL[dom]
    # the dense writer is timed live in every timed step (CUDA events on the library's side stream, where it runs
    # beside the evaluate kernels: the in-step, contended figure); any other stage by the breakdown pass
    dom_ms = (fill_sum / args.steps) if dom == "fill" else stage_ms[dom]
    dom_gbs = alg_bytes[dom] / (dom_ms * 1e-3) / 1e9 if dom_ms else 0.0
    traffic, traffic_src = kernel_traffic(w.name, kern) if not zslab else (None, None)
    if args.traffic is not None:
        traffic, traffic_src = args.traffic, "--traffic"
    roofline = {"bound": "hbm", "kernel": "%s (%s)" % (kern, what), "achieved": dom_gbs, "peak": peak, "unit": "GB/s",
                "frac": dom_gbs / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": alg_bytes[dom], "ms_per_launch": dom_ms, "dominant_stage": dom,
                "timed": "live in the %d timed steps" % args.steps if dom == "fill" else "breakdown pass of %d steps" % nbr}
    if dom != "fill" and stage_ms.get("fill"):
        fg = 8.0 * N / (fill_sum / args.steps * 1e-3) / 1e9
        roofline["dense_writer"] = {"kernel": "fill_tma_kernel", "achieved": fg, "frac": fg / peak,
                                    "ms_per_launch": fill_sum / args.steps, "algorithmic_bytes_per_launch": 8.0 * N}
    # north_star: the slower of (grid + feature bytes at HBM peak) and (pair evaluations at FP32 peak)
    fp32_tf, sms = B.sdf_measure_fp32_peak(stream=stream)
    step_bytes = 8.0 * N + 36.0 * w.ntri
    hbm_ms = step_bytes / (peak * 1e9) * 1e3
    fp32_ms = float(stats["pairs_accepted"]) * FLOP_PER_PAIR / (fp32_tf * 1e12) * 1e3
    ideal_ms = max(hbm_ms, fp32_ms)
    roofline_step = {"bound": "hbm" if hbm_ms >= fp32_ms else "fp32", "algorithmic_bytes": step_bytes, "hbm_ms": hbm_ms,
                     "fp32_peak_tflops": fp32_tf, "fp32_peak_source": "measured: sdf_measure_fp32_peak, FMA loop on %d SMs" % sms,
                     "algorithmic_flop": float(stats["pairs_accepted"]) * FLOP_PER_PAIR, "fp32_ms": fp32_ms,
                     "ideal_ms": ideal_ms, "frac": ideal_ms / ms_per_step}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        r = time_oracle(w, args.cpu_slices, 1, 0)
        cpu = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
        # "plus a 1-thread time on C1-C3" -- bounded samples of each, one thread
        one = {}
        for cn, sl in (("C1", 64), ("C2", 24), ("C3", 12)):
            r1 = time_oracle(W.config(cn), sl, 1, 0, threads=1)
            one[cn] = {"value": r1["value"], "s": r1["s_per_step"], "band_cells": r1["band_cells"], "sample": r1["sample"].split(";")[0]}
        cpu["one_thread"] = one

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong" if zslab and world > 1 else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": workload_config(w, args),
            "band_cells": band_cells, "stage_ms": stage_ms, "step_ms_min": min(step_ms), "step_ms_median": float(np.median(step_ms)),
            "step_ms_max": max(step_ms), "wall_ms_per_step":
            t_wall * 1e3 / args.steps, "roofline": roofline, "roofline_step": roofline_step, "cpu_baseline": cpu,
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clk, "zslab": zslab, "fill_interior": fill_int, "closest_points": cpt,
            "stats": {k: stats[k] for k in ("polyhedra", "work_items", "pairs_tested", "pairs_accepted",
                                            "bricks_active", "fp64_rechecks", "cdp_fallbacks")}}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4", choices=list(W.CONFIG_NAMES))
    ap.add_argument("--band-cells", type=float, default=0.0, help="override the band width (cells); 0 = the config's")
    ap.add_argument("--fill-interior", action="store_true", help="also time sdf_fill_interior (NEXT-1) on the result")
    ap.add_argument("--closest-points", action="store_true", help="also time sdf_closest_points (NEXT-2) on the result")
    ap.add_argument("--zslab", action="store_true", help="strong scaling: rank r computes z-slab r of WORLD_SIZE (NEXT-4)")
    ap.add_argument("--zslab-parts", type=int, default=0, help="time one slab of a P-way z split on this GPU")
    ap.add_argument("--zslab-part", type=int, default=0)
    ap.add_argument("--split-calls", action="store_true",
                    help="step = sdf_create + sdf_compute (two calls) instead of sdf_transform (the same path in one call)")
    ap.add_argument("--breakdown-steps", type=int, default=3, help="extra untimed steps with every stage instrumented (stage_ms)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-slices", type=int, default=256, help="z-slices of the oracle sample (cpu_baseline)")
    ap.add_argument("--ref-slices", type=int, default=64, help="z-slices per step of --impl reference")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes (read + write) per launch of the dominant kernel; default: read from "
                         "profiles/kernel_traffic.csv (the committed ncu --set full captures)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
