#!/usr/bin/env python
"""bench.py -- BASELINE.json metric: fp64 TDMA grid cells/s (+ achieved HBM GB/s vs peak) on the
1024^3 y-systems workload (cfg3_weak: 1024 x 1024 x 1024, P = 16), one B200 per rank.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg3_weak] [--variant fused|pipelined] [--batch BZ] [--nstreams S]
                    [--sweep]           # S7 batch / stream sweep, JSON lines to stdout

A "step" is one pass of the whole hot path (partition reduce -> gather -> reduced solve ->
back-substitution, all batches) over the slab, inputs resident in HBM.  Timing: CUDA events on the
stream the solve is launched on, bracketed by barrier + synchronize, max over ranks.  The slab
(5 x 8 GiB) is far larger than L2 (126 MB), so no explicit L2 flush is needed between steps.
Multi-GPU: the path shards by lines with no exchange step, so every rank solves its own slab of the
same shape (weak scaling, no data-path collective); torch.distributed (NCCL) is used only for the
barrier and the max-over-ranks reduction.

Rank 0 prints ONE JSON line.  Extra keys: "roofline" (dominant kernel against the measured HBM
copy bandwidth in MEASURED_PEAKS.json), "cpu_baseline" (the oracle, as it stands, on the host
cores for a bounded sample), "e2e" (same metric through tdma_solve_host with pinned HOST buffers,
H2D/D2H inside the timed region), "clocks", "gpu_launches", "variants".
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64_tdma_grid_cells_per_s"
UNIT = "cells/s"
ALG_BYTES_PER_CELL = 40.0        # read a, b, c, d (32 B) + write x (8 B): SURVEY.md 8(d)
FALLBACK_HBM_GBS = 6650.0        # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(alg_bytes_per_launch, fused_cfg):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the
    committed `ncu --set full` capture (profiles/traffic.json; a profiler cannot run inside the
    timed region, so this is a STATIC capture: `source` says of what).  The capture is of a shorter
    slab; traffic is proportional to cells, so it is rescaled to this launch's algorithmic bytes.
    (None, why) when there is no capture or it was taken with another tiling of the kernel."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            t = json.load(f)
    except Exception:
        return None, "no profiles/traffic.json"
    cap = t.get("fused", {})
    for key in ("lines", "cluster", "leaf_rows", "threads"):
        if cap.get(key) != fused_cfg.get(key):
            return None, "capture is of another tiling (%s: captured %r, running %r)" % (key, cap.get(key), fused_cfg.get(key))
    src = {"static_capture": t.get("source"), "captured_cells": t.get("cells"), "commit": t.get("commit"),
           "bytes_per_cell": (t["dram_bytes_read"] + t["dram_bytes_write"]) / t["cells"]}
    return (t["dram_bytes_read"] + t["dram_bytes_write"]) / t["alg_bytes"] * alg_bytes_per_launch, src


class RankGroup:
    """One process per GPU.  The path shards by lines with no exchange step, so every rank solves
    its own slab of the same shape (weak scaling); torch.distributed is used for the barrier and
    the max-over-ranks of the device time only.  backend None = single process."""

    def __init__(self, backend, device=None):
        self.dist = None
        self.device = device
        self.world = int(os.environ.get("WORLD_SIZE", "1")) if backend else 1
        self.rank = int(os.environ.get("RANK", "0")) if backend else 0
        if backend:
            import torch.distributed as dist_mod
            self.dist = dist_mod
            kw = {"device_id": device} if backend == "nccl" else {}
            dist_mod.init_process_group(backend, **kw)

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max(self, v: float) -> float:
        if self.dist is None:
            return v
        import torch
        t = torch.tensor([v], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate(self, cells_per_rank: int, max_seconds: float) -> float:
        """Whole-job throughput: the cells all ranks processed / the slowest rank's time."""
        return cells_per_rank * self.world / max_seconds

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons every 200 ms while the timed region runs."""
    QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
             "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu_index = gpu_index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.gpu_index), "--query-gpu=" + self.QUERY,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[1])); smax.append(float(r[2]))
            except Exception:
                continue
            for name, val in zip(names, r[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None,
                "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def cpu_oracle_rate(w_host, min_seconds=10.0, max_repeats=64):
    """The oracle as it stands (OpenMP over lines, all host cores) on the given host sample."""
    import oracle
    arrs = [t.numpy() for t in w_host]
    cells = arrs[0].size
    oracle.solve_y(*arrs)                                   # warm-up (page faults, thread pool)
    t0 = time.perf_counter()
    reps = 0
    while True:
        oracle.solve_y(*arrs)
        reps += 1
        el = time.perf_counter() - t0
        if el >= min_seconds or reps >= max_repeats:
            break
    return cells * reps / el, reps, el, oracle.max_threads()


def run_reference(args):
    """--impl reference: the CPU oracle on the box's host cores, same metric / config keys."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import torch
    import tdma_inputs
    spec = tdma_inputs.config_spec(args.workload)
    nzs = min(spec["nz"], args.ref_slices)
    w = tdma_inputs.make_workload(args.workload, device="cpu", nz=nzs)
    host = (w.a, w.b, w.c, w.d)
    import oracle
    arrs = [t.numpy() for t in host]
    for _ in range(max(1, args.warmup if args.warmup <= 2 else 2)):
        oracle.solve_y(*arrs)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.solve_y(*arrs)
    el = time.perf_counter() - t0
    value = w.cells * args.steps / el
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": args.workload, "nx": w.nx, "ny": w.ny, "nz": spec["nz"], "P": w.P,
                   "sample": "each step = oracle Thomas solve of %d of the %d z-slices" % (nzs, spec["nz"])},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
                         "sample": "%d z-slices (%d cells) per step" % (nzs, w.cells)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def time_solve(torch, plan, w, x, steps, warmup, barrier, per_step=None):
    """Returns seconds per step (device time, CUDA events on the launching stream).  per_step: a list
    that receives every step's own duration in ms (an event between consecutive steps; SURVEY 8(d):
    "report median and best")."""
    stream = torch.cuda.current_stream()
    for _ in range(warmup):
        plan.solve(w.a, w.b, w.c, w.d, x, stream)
    torch.cuda.synchronize()
    barrier()
    marks = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1 if per_step is not None else 2)]
    marks[0].record(stream)
    for i in range(steps):
        plan.solve(w.a, w.b, w.c, w.d, x, stream)
        if per_step is not None and i + 1 < steps:
            marks[i + 1].record(stream)
    marks[-1].record(stream)
    torch.cuda.synchronize()
    barrier()
    if per_step is not None:
        per_step.extend(marks[i].elapsed_time(marks[i + 1]) for i in range(steps))
    return marks[0].elapsed_time(marks[-1]) * 1e-3 / steps


def stage_times(torch, tdma, plan, w, x, reps=3):
    """Stage-isolated mean time per batch, PIPELINED plans."""
    nb = plan.get(tdma.TDMA_GET_NB)
    stream = torch.cuda.current_stream()
    out = {}
    for name, st in (("A", tdma.TDMA_STAGE_A), ("B", tdma.TDMA_STAGE_B), ("C", tdma.TDMA_STAGE_C)):
        nbt = min(nb, 64)
        for n in range(min(nbt, 4)):
            plan.stage(st, n, w.a, w.b, w.c, w.d, x, stream)
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            for n in range(nbt):
                plan.stage(st, n, w.a, w.b, w.c, w.d, x, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        out[name] = e0.elapsed_time(e1) * 1e-3 / (reps * nbt)
    return out


def parity_check(torch, w, x, slices):
    """Checker leg, outside every timed region: sampled z-slices of the x the timed solves left
    behind, against the CPU oracle (long double on the weakly dominant Poisson workloads), with the
    metric and tolerance of the parity tests (normwise per line)."""
    import numpy as np
    import oracle
    prec = "f64" if w.strictly_dominant else "ld"
    worst, finite = 0.0, True
    for k in slices:
        arrs = [t[k:k + 1].cpu().numpy() for t in (w.a, w.b, w.c, w.d, x)]
        finite = finite and bool(np.isfinite(arrs[4]).all())
        ref = oracle.solve_y(*arrs[:4], prec)
        worst = max(worst, float(oracle.normwise_error(arrs[4], ref).max()))
    return {"slices": list(slices), "E_max": worst, "tol": 1e-11, "oracle": prec,
            "ok": bool(finite and worst <= 1e-11)}


def pick_slices(nz, fill):
    """First / interior / last slices of the main launch's range and of the fill launch's."""
    main_last = nz - fill - 1
    picks = {0, min(1, nz - 1), nz // 2 + 1 if nz // 2 + 1 <= main_last else 0, max(0, main_last)}
    if fill > 0:
        picks |= {nz - fill, nz - 1}
    return sorted(p for p in picks if 0 <= p < nz)


def fused_config(tdma, plan):
    impl = plan.get(tdma.TDMA_GET_FUSED_IMPL)
    return {"impl": "tma" if impl == 2 else "reg", "lines": plan.get(tdma.TDMA_GET_FUSED_LINES),
            "cluster": plan.get(tdma.TDMA_GET_FUSED_CLUSTER), "leaf_rows": plan.get(tdma.TDMA_GET_FUSED_LEAF_ROWS),
            "threads": plan.get(tdma.TDMA_GET_FUSED_THREADS), "smem": plan.get(tdma.TDMA_GET_FUSED_SMEM)}


def pipelined_report(torch, tdma, plan, w, x, sec):
    """Stage-isolated times and how much of stage B is hidden behind A / C."""
    st = stage_times(torch, tdma, plan, w, x)
    nb = plan.get(tdma.TDMA_GET_NB)
    tot_b = st["B"] * nb
    exposed = sec - (st["A"] + st["C"]) * nb
    return {"stage_ms_per_batch": {k: v * 1e3 for k, v in st.items()},
            "stage_b_hidden_frac": (1.0 - max(0.0, exposed) / tot_b) if tot_b > 0 else None,
            "sum_of_stages_ms": (st["A"] + st["B"] + st["C"]) * nb * 1e3}, st


def second_workload(torch, tdma, tdma_inputs, name, dev, steps, warmup, barrier, peak):
    """A further BASELINE config timed the same way (FUSED, one launch), with its parity check."""
    w = tdma_inputs.make_workload(name, device=dev)
    x = torch.empty_like(w.d)
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, 0, variant=tdma.TDMA_VARIANT_FUSED) as plan:
        sec = time_solve(torch, plan, w, x, steps, warmup, barrier)
        fill = plan.get(tdma.TDMA_GET_FUSED_FILL)
        rec = {"ms_per_step": sec * 1e3, "value": w.cells / sec, "unit": UNIT, "steps": steps,
               "hbm_gbs_40B": ALG_BYTES_PER_CELL * w.cells / sec / 1e9,
               "hbm_frac_of_8TBs": ALG_BYTES_PER_CELL * w.cells / sec / 8e12,
               "frac_of_measured_peak": ALG_BYTES_PER_CELL * w.cells / sec / 1e9 / peak,
               "config": {"workload": name, "nx": w.nx, "ny": w.ny, "nz": w.nz, "P": w.P, "variant": "fused",
                          "fill_slices": fill, "fused": fused_config(tdma, plan)}}
    rec["parity_check"] = parity_check(torch, w, x, pick_slices(w.nz, fill))
    return rec


def shared_workload(torch, tdma, tdma_inputs, base, cplx, dev, steps, warmup, barrier, peak, nz=None,
                    cpu_seconds=5.0):
    """SURVEY 8(f) f3 / the paper's own benchmark form: the Poisson config with
    its coefficients passed as 1-D arrays and a real or complex right-hand side, through
    tdma_solve_shared.  Algorithmic bytes: d read + x written = 16 B per real cell, 32 B per complex
    cell.  Own roofline, parity check (long-double reference on sampled slices) and CPU baseline."""
    import numpy as np
    import oracle
    w = tdma_inputs.make_shared_workload(base, cplx, device=dev, nz=nz)
    x = torch.empty_like(w.d)
    stream = torch.cuda.current_stream()
    args = (w.a_y, w.b0_y, w.c_y, w.sx, w.sz, w.d, x)
    with tdma.Plan(w.nx, w.ny, w.nz, 1, 0) as plan:
        for _ in range(warmup):
            plan.solve_shared(*args, pin00=w.pin00, stream=stream)
        torch.cuda.synchronize()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            plan.solve_shared(*args, pin00=w.pin00, stream=stream)
        e1.record(stream)
        torch.cuda.synchronize()
        barrier()
        sec = e0.elapsed_time(e1) * 1e-3 / steps
        tiling = {k: plan.get(getattr(tdma, "TDMA_GET_SHARED_" + k.upper()))
                  for k in ("lines", "cluster", "leaf_rows", "threads", "slots", "smem", "fill")}
    bpc = 16.0 * w.ncomp
    fill = tiling["fill"]
    main_bytes = bpc * w.nx * w.ny * (w.nz - fill)
    rec = {"ms_per_step": sec * 1e3, "value": w.cells / sec, "unit": "complex cells/s" if cplx else UNIT, "steps": steps,
           "dtype": "c128 (f64 arithmetic)" if cplx else "f64", "alg_bytes_per_cell": bpc,
           "hbm_gbs": bpc * w.cells / sec / 1e9, "frac_of_measured_peak": bpc * w.cells / sec / 1e9 / peak,
           "hbm_frac_of_8TBs": bpc * w.cells / sec / 8e12,
           "roofline": {"bound": "hbm", "kernel": "shared_tma_kernel", "achieved": main_bytes / sec / 1e9, "peak": peak,
                        "unit": "GB/s", "frac": main_bytes / sec / 1e9 / peak, "traffic": None,
                        "alg_bytes_per_launch": main_bytes, "launch_ms": sec * 1e3},
           "config": {"workload": w.name, "nx": w.nx, "ny": w.ny, "nz": w.nz, "ncomp": w.ncomp, "pin00": w.pin00,
                      "tiling": tiling}}
    # parity of what was just timed: sampled slices against the long-double reference
    picks = pick_slices(w.nz, fill)
    worst = 0.0
    host = [t.cpu().numpy() for t in (w.a_y, w.b0_y, w.c_y, w.sx)]
    def lines(v):
        return v.view(np.float64).reshape(v.shape[0], v.shape[1], -1) if np.iscomplexobj(v) else v
    for k in picks:
        dk, xk = w.d[k:k + 1].cpu().numpy(), x[k:k + 1].cpu().numpy()
        ref = oracle.solve_y_shared(*host, w.sz[k:k + 1].cpu().numpy(), dk, pin00=(w.pin00 and k == 0), precision="ld")
        worst = max(worst, float(oracle.normwise_error(lines(np.ascontiguousarray(xk)), lines(ref)).max()))
    rec["parity_check"] = {"slices": picks, "E_max": worst, "tol": 1e-11, "oracle": "ld", "ok": bool(worst <= 1e-11)}
    # the CPU reference as it stands on a bounded sample (first slices), all host cores
    nzc = min(w.nz, 16)
    dh = w.d[:nzc].cpu().numpy()
    szh = w.sz[:nzc].cpu().numpy()
    oracle.solve_y_shared(*host, szh, dh, pin00=w.pin00)
    t0, reps = time.perf_counter(), 0
    while True:
        oracle.solve_y_shared(*host, szh, dh, pin00=w.pin00)
        reps += 1
        el = time.perf_counter() - t0
        if el >= cpu_seconds or reps >= 64:
            break
    rec["cpu_baseline"] = {"value": w.nx * w.ny * nzc * reps / el, "unit": rec["unit"], "cores": oracle.max_threads(),
                           "kind": "oracle", "sample": "%d z-slices x %d repeats, %.1f s" % (nzc, reps, el)}
    return rec


def general_shapes(torch, tdma, tdma_inputs, dev, steps, warmup):
    """The general-shape paths next to the tiled kernels on neighbouring shapes (not headline numbers: they
    exist so that every nx, line length, axis and wrap is solved).  Every timed solve is checked against the
    oracle on two sampled slices, outside the timed region."""
    import numpy as np
    import oracle

    def timed(fn):
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps

    def err_axis(a, b, c, d, x, axis, periodic, slices):
        ax = {"y": 1, "z": 0, "x": 2}[axis]
        worst = 0.0
        for k in slices:
            sl = (slice(None), slice(k, k + 1)) if axis == "z" else (slice(k, k + 1),)
            arrs = [t[sl].cpu().numpy() for t in (a, b, c, d, x)]
            ref = oracle.solve_axis(*arrs[:4], axis, bool(periodic))
            worst = max(worst, float((np.max(np.abs(arrs[4] - ref), axis=ax) / np.max(np.abs(ref), axis=ax)).max()))
        return worst

    out = {"general_shapes": True, "steps": steps, "tol": 1e-11, "records": []}
    V = {"pipelined": tdma.TDMA_VARIANT_PIPELINED, "staged": tdma.TDMA_VARIANT_STAGED, "fused": tdma.TDMA_VARIANT_FUSED}
    # general form: cyclic y lines on all three variants, x sweeps on the TMA kernel and on the stage pipeline
    for name, (nz, ny, nx), P, batch, opts, axis in [
            ("y cyclic, fused", (64, 1024, 1024), 16, 0, dict(variant=V["fused"], periodic=1), "y"),
            ("y cyclic, pipelined", (64, 1024, 1024), 16, 16, dict(variant=V["pipelined"], periodic=1), "y"),
            ("y plain, pipelined", (64, 1024, 1024), 16, 16, dict(variant=V["pipelined"]), "y"),
            ("y cyclic, staged", (64, 1024, 1024), 16, 16, dict(variant=V["staged"], periodic=1), "y"),
            ("y cyclic, 1000 rows x 1023 (auto -> pipelined)", (64, 1000, 1023), 8, 16, dict(periodic=1), "y"),
            ("y sweep, ny = 768 (auto: clusters of 3, 16-row leaves)", (256, 768, 1024), 16, 0, dict(variant=V["fused"]), "y"),
            ("y sweep, ny = 768, clusters of 4, 12-row leaves", (256, 768, 1024), 16, 0, dict(variant=V["fused"], fused_cluster=4), "y"),
            ("y sweep, ny = 1280 (auto: clusters of 5, 16-row leaves)", (128, 1280, 1024), 16, 0, dict(variant=V["fused"]), "y"),
            ("y sweep, ny = 1280, clusters of 8, 10-row leaves", (128, 1280, 1024), 16, 0, dict(variant=V["fused"], fused_cluster=8), "y"),
            ("z sweep, nz = 640 (auto: clusters of 5)", (640, 256, 1024), 16, 0, dict(variant=V["fused"], axis=tdma.TDMA_AXIS_Z), "z"),
            ("z sweep, nz = 640, clusters of 4, 10-row leaves", (640, 256, 1024), 16, 0, dict(variant=V["fused"], axis=tdma.TDMA_AXIS_Z, fused_cluster=4), "z"),
            ("x sweep, nx = 1024 (auto -> fused)", (64, 512, 1024), 8, 8, dict(axis=tdma.TDMA_AXIS_X), "x"),
            ("x sweep, nx = 768 (auto -> fused, clusters of 3)", (64, 512, 768), 8, 8, dict(axis=tdma.TDMA_AXIS_X), "x"),
            ("x sweep, nx = 1000 (auto -> pipelined)", (64, 512, 1000), 8, 8, dict(axis=tdma.TDMA_AXIS_X), "x")]:
        a, b, c, d = tdma_inputs.dominant_random(nx, ny, nz, 7, dev)
        x = torch.full_like(d, float("nan"))
        with tdma.Plan(nx, ny, nz, P, batch, **opts) as plan:
            ms = timed(lambda: plan.solve(a, b, c, d, x))
            variant = plan.get(tdma.TDMA_GET_VARIANT)
        E = err_axis(a, b, c, d, x, axis, opts.get("periodic", 0), [0, (ny if axis == "z" else nz) - 1])
        out["records"].append({"case": name, "shape": [nz, ny, nx], "variant": {1: "pipelined", 2: "fused", 3: "staged"}[variant],
                               "ms": ms, "gbs_40B": 40.0 * nz * ny * nx / ms / 1e6, "E_max": E, "ok": bool(E <= 1e-11)})
        del a, b, c, d, x
    # shared form: the tiled kernel and the one-thread-per-line kernel on neighbouring shapes
    g = torch.Generator().manual_seed(5)
    u = lambda n, lo, hi: (lo + (hi - lo) * torch.rand(n, dtype=torch.float64, generator=g)).to(dev)
    for name, (nz, ny, nx), cplx in [("shared, ny = 1024", (128, 1024, 1024), False), ("shared, ny = 768 (24-row leaves)", (128, 768, 1024), False),
                                     ("shared, ny = 640 (20-row leaves)", (128, 640, 1024), False),
                                     ("shared complex, ny = 768 (12-row leaves)", (128, 768, 1024), True),
                                     ("shared, ny = 1000", (128, 1000, 1024), False),
                                     ("shared, nx = 1023", (128, 1024, 1023), False), ("shared complex, ny = 1000", (128, 1000, 1024), True)]:
        a_y, b0_y, c_y, sx, sz = u(ny, -1, 1), u(ny, 2.5, 3.5), u(ny, -1, 1), -u(nx, 0, 2), -u(nz, 0, 2)
        d = torch.randn((nz, ny, nx), dtype=torch.float64, device=dev)
        if cplx:
            d = torch.complex(d, torch.randn((nz, ny, nx), dtype=torch.float64, device=dev))
        x = torch.full_like(d, float("nan"))
        with tdma.Plan(nx, ny, nz, 1, 0) as plan:
            ms = timed(lambda: plan.solve_shared(a_y, b0_y, c_y, sx, sz, d, x))
            line_kernel = plan.get(tdma.TDMA_GET_SHARED_LINE_KERNEL)
        worst = 0.0
        for k in (0, nz - 1):
            ref = oracle.solve_y_shared(*[t.cpu().numpy() for t in (a_y, b0_y, c_y, sx)], sz[k:k + 1].cpu().numpy(),
                                        d[k:k + 1].cpu().numpy(), pin00=False, precision="f64")
            xr, rr = x[k:k + 1].cpu().numpy(), ref
            if cplx:
                xr, rr = xr.view(np.float64).reshape(1, ny, -1), np.ascontiguousarray(rr).view(np.float64).reshape(1, ny, -1)
            worst = max(worst, float(oracle.normwise_error(xr, rr).max()))
        bpc = 32.0 if cplx else 16.0
        out["records"].append({"case": name, "shape": [nz, ny, nx], "kernel": "one thread per line" if line_kernel else "tiled TMA",
                               "ms": ms, "gbs_alg": bpc * nz * ny * nx / ms / 1e6, "alg_bytes_per_cell": bpc, "E_max": worst,
                               "ok": bool(worst <= 1e-11)})
        del d, x
    out["ok"] = all(r["ok"] for r in out["records"])
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3_weak")
    ap.add_argument("--variant", default="auto", choices=["auto", "fused", "pipelined", "staged"])
    ap.add_argument("--batch", type=int, default=-1, help="z-slices per batch (-1: workload default)")
    ap.add_argument("--nstreams", type=int, default=0)
    ap.add_argument("--nz", type=int, default=0, help="restrict the slab to the first NZ slices")
    ap.add_argument("--ref-slices", type=int, default=16)
    ap.add_argument("--e2e-slices", type=int, default=128)
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    ap.add_argument("--sustained-seconds", type=float, default=2.5,
                    help="length of the second, power-steady timed leg (0 = skip)")
    ap.add_argument("--also", default="cfg5_stress",
                    help="further workload timed after the headline one at N = 1 ('' = none)")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip sustained / e2e / cpu_baseline / stage / second-workload legs")
    ap.add_argument("--shared", default="", choices=["", "f64", "c128"],
                    help="time only the shared-coefficient form of --workload (real / complex RHS) and print its record")
    ap.add_argument("--sweep", action="store_true", help="S7 batch x stream sweep (JSON lines)")
    ap.add_argument("--timeline", action="store_true",
                    help="S6 evidence without nsys: per-launch start/end of the PIPELINED stages of one solve "
                         "(CUDA events on the plan's streams), overlap statistics as one JSON line")
    ap.add_argument("--yslab", type=int, default=0,
                    help="NEXT row f4: time the rank-local stages of an N-rank y-slab job on this GPU (one JSON line)")
    ap.add_argument("--adi", action="store_true",
                    help="NEXT row f1 / BASELINE cfg 4: three successive FUSED solves along x (periodic), "
                         "y (Dirichlet) and z (periodic); use with --workload cfg4_adi_y")
    ap.add_argument("--general-shapes", action="store_true",
                    help="time the paths that take what the TMA kernels cannot tile (cyclic lines / x sweeps on the "
                         "stage pipeline, the one-thread-per-line kernel of the shared form), each checked against "
                         "the oracle on sampled slices; one JSON line")
    args = ap.parse_args()

    if args.impl == "reference":
        return run_reference(args)

    import torch
    import tdma_inputs
    import paper_2509_03933_b200 as tdma

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    group = RankGroup("nccl" if world > 1 else None, dev)
    barrier, max_over_ranks = group.barrier, group.max
    peak, peak_src = measured_peak()

    if args.general_shapes:
        rec = general_shapes(torch, tdma, tdma_inputs, dev, args.steps, max(3, args.warmup))
        if rank == 0:
            print(json.dumps(rec))
        group.close()
        return 0
    spec = tdma_inputs.config_spec(args.workload)
    nz = args.nz if args.nz > 0 else spec["nz"]
    if args.shared:
        rec = shared_workload(torch, tdma, tdma_inputs, args.workload, args.shared == "c128", dev, args.steps,
                              max(3, args.warmup), group.barrier, peak, nz=nz,
                              cpu_seconds=0.0 if args.no_extras else args.cpu_seconds / 2)
        if rank == 0:
            print(json.dumps(rec))
        group.close()
        return 0
    w = tdma_inputs.make_workload(args.workload, device=dev, nz=nz)
    x = torch.empty_like(w.d)
    batch = spec["batch"] if args.batch < 0 else args.batch
    cells = w.cells
    vmap = {"fused": tdma.TDMA_VARIANT_FUSED, "pipelined": tdma.TDMA_VARIANT_PIPELINED,
            "staged": tdma.TDMA_VARIANT_STAGED}
    warmup = max(3, args.warmup)

    if args.sweep:
        return sweep(torch, tdma, w, x, args, barrier, rank)
    if args.adi:
        return adi(torch, tdma, w, x, args, barrier, rank, peak)
    if args.yslab:
        return yslab(torch, tdma, w, args, rank, peak)
    if args.timeline:
        return timeline(torch, tdma, w, x, args, batch, rank)

    # ---- candidate variants: the headline is the faster one; both are reported ---------------
    names = ["fused", "pipelined", "staged"] if args.variant == "auto" else [args.variant]
    results = {}
    for name in names:
        opts = dict(variant=vmap[name])
        bz = batch
        if name == "fused":
            bz = 0 if args.batch < 0 else args.batch      # one launch covers the slab by default
        if args.nstreams:
            opts["nstreams"] = args.nstreams
        try:
            plan = tdma.Plan(w.nx, w.ny, w.nz, w.P, bz, **opts)
        except tdma.TdmaError as exc:
            results[name] = {"error": str(exc)}
            continue
        quick = time_solve(torch, plan, w, x, max(2, args.steps // 4), warmup, barrier)
        results[name] = {"plan": plan, "quick_s": quick, "batch": plan.get(tdma.TDMA_GET_BATCH),
                         "launches": plan.get(tdma.TDMA_GET_LAUNCHES),
                         "nstreams": plan.get(tdma.TDMA_GET_NSTREAMS)}
    ok = {k: v for k, v in results.items() if "plan" in v}
    if not ok:
        raise SystemExit("no variant could be planned: %r" % results)
    best = min(ok, key=lambda k: ok[k]["quick_s"])
    plan = ok[best]["plan"]

    # ---- timed region (K steps) --------------------------------------------------------------
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    step_ms = []
    sec = time_solve(torch, plan, w, x, args.steps, warmup, barrier, per_step=step_ms)
    clocks = sampler.stop() if rank == 0 else None
    sec = max_over_ranks(sec)
    value = group.aggregate(cells, sec)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "nx": w.nx, "ny": w.ny, "nz": w.nz, "P": w.P,
                   "variant": best, "batch": ok[best]["batch"], "nstreams": ok[best]["nstreams"],
                   "cells_per_gpu": cells, "l2": "inputs (5 x %.1f GiB) far larger than L2" % (cells * 8 / 2 ** 30),
                   "parallelism": "lines sharded, one slab per rank, no collective"},
        "gpu_launches": ok[best]["launches"] * args.steps,
        "hbm_gbs_40B": ALG_BYTES_PER_CELL * cells / sec / 1e9,
        "hbm_frac_of_8TBs": ALG_BYTES_PER_CELL * cells / sec / 8e12,
    }
    if clocks is not None:
        out["clocks"] = clocks
    out["step_ms"] = {"median": sorted(step_ms)[len(step_ms) // 2], "best": min(step_ms), "worst": max(step_ms),
                      "note": "rank 0, per-step CUDA events inside the timed region"}
    out["variants"] = {k: ({"ms_per_step": v["quick_s"] * 1e3, "batch": v["batch"], "launches": v["launches"]}
                           if "plan" in v else v) for k, v in results.items()}

    # ---- sustained leg: long enough to reach power steady state ------------------------------
    if args.sustained_seconds > 0 and not args.no_extras:
        n_sus = max(args.steps, int(args.sustained_seconds / sec) + 1)
        sampler = ClockSampler(local_rank)
        if rank == 0:
            sampler.start()
        sec_s = max_over_ranks(time_solve(torch, plan, w, x, n_sus, 1, barrier))
        ck = sampler.stop() if rank == 0 else {}
        out["sustained"] = {"ms_per_step": sec_s * 1e3, "steps": n_sus, "seconds": sec_s * n_sus,
                            "value": group.aggregate(cells, sec_s),
                            "hbm_gbs_40B": ALG_BYTES_PER_CELL * cells / sec_s / 1e9,
                            "hbm_frac_of_8TBs": ALG_BYTES_PER_CELL * cells / sec_s / 8e12,
                            "frac_of_measured_peak": ALG_BYTES_PER_CELL * cells / sec_s / 1e9 / peak,
                            "sm_mhz": ck.get("sm_mhz"), "reasons": ck.get("reasons"), "samples": ck.get("samples")}

    # ---- parity of what was just timed (rank 0; checker leg, untimed) ------------------------
    fill = plan.get(tdma.TDMA_GET_FUSED_FILL) if best == "fused" else 0
    if rank == 0:
        out["parity_check"] = parity_check(torch, w, x, pick_slices(w.nz, fill))

    # ---- roofline of the dominant kernel -----------------------------------------------------
    if best == "fused":
        # Persistent launches back to back do the whole step.  When clusters of >= 4 CTAs leave SMs
        # empty, a concurrent fill launch (clusters of 2) solves the last `fill` z-slices of each
        # launch's range on them; the dominant kernel is the main launch: together the main launches
        # span the step (CUDA events around the step on the launching stream).
        # the slab is solved in nb_f persistent launches of bz_f slices (default: ~2^27 cells each),
        # every one with its own fill launch over its last `fill` slices
        nb_f = max(1, plan.get(tdma.TDMA_GET_NB))
        bz_f = plan.get(tdma.TDMA_GET_BATCH)
        alg_bytes = ALG_BYTES_PER_CELL * w.nx * w.ny * (bz_f - fill)
        dur = sec * bz_f / w.nz
        achieved = alg_bytes / dur / 1e9
        out["config"]["fill_slices"] = fill
        out["config"]["launches_per_step"] = ok[best]["launches"]
        fcfg = fused_config(tdma, plan)
        out["config"]["fused"] = fcfg
        traffic, tsrc = ncu_traffic(alg_bytes, fcfg)
        out["roofline"] = {"bound": "hbm", "kernel": "fused_tma_kernel" if fcfg["impl"] == "tma" else "fused_kernel",
                           "achieved": achieved, "peak": peak,
                           "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": tsrc,
                           "alg_bytes_per_launch": alg_bytes, "launch_ms": dur * 1e3, "peak_source": peak_src,
                           "whole_step_frac": ALG_BYTES_PER_CELL * cells / sec / 1e9 / peak}
    # the paper's pipeline (S6): stage times and the hidden share of stage B, whichever variant won
    # (PIPELINED: a', c', d' through HBM, 88 B/cell; STAGED: TMA-staged stage A / C, 72 B/cell)
    for pname in ("pipelined", "staged"):
        if pname not in ok or args.no_extras:
            continue
        pplan = ok[pname]["plan"]
        psec = sec if best == pname else ok[pname]["quick_s"]
        rep, st = pipelined_report(torch, tdma, pplan, w, x, psec)
        out["variants"][pname].update(rep)
        out["variants"][pname]["hbm_bytes_per_cell"] = 88.0 if pname == "pipelined" else 72.0
        try:        # the overlap itself, from per-launch events on the plan's streams (one untimed solve)
            tl, _ = timeline_overlap(torch, tdma, w, x, vmap[pname], ok[pname]["batch"], ok[pname]["nstreams"])
            out["variants"][pname]["timeline"] = tl
        except tdma.TdmaError as exc:
            out["variants"][pname]["timeline"] = {"error": str(exc)}
        if best == "pipelined" and pname == "pipelined":
            bz = ok[best]["batch"]
            bcells = w.nx * w.ny * bz
            alg_bytes = (32.0 + 24.0) * bcells + 48.0 * w.P * w.nx * bz   # read a,b,c,d; write a',c',d' + reduced rows
            achieved = alg_bytes / st["A"] / 1e9
            out["roofline"] = {"bound": "hbm", "kernel": "stage_a_kernel", "achieved": achieved, "peak": peak,
                               "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                               "alg_bytes_per_launch": alg_bytes, "launch_ms": st["A"] * 1e3,
                               "peak_source": peak_src}
            out["stage_ms_per_batch"] = rep["stage_ms_per_batch"]
            out["stage_b_hidden_frac"] = rep["stage_b_hidden_frac"]
        if best == "staged" and pname == "staged":
            bz = ok[best]["batch"]
            bcells = w.nx * w.ny * bz
            alg_bytes = 40.0 * bcells                   # stage C: read a, b, c, d again, write x
            achieved = alg_bytes / st["C"] / 1e9
            out["roofline"] = {"bound": "hbm", "kernel": "fused_tma_kernel<kStage = 2> (stage C)", "achieved": achieved,
                               "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                               "alg_bytes_per_launch": alg_bytes, "launch_ms": st["C"] * 1e3, "peak_source": peak_src}
            out["stage_ms_per_batch"] = rep["stage_ms_per_batch"]
            out["stage_b_hidden_frac"] = rep["stage_b_hidden_frac"]

    # ---- extras on rank 0, N = 1 only --------------------------------------------------------
    if rank == 0 and world == 1 and not args.no_extras:
        for v in ok.values():
            if v["plan"] is not plan:
                v["plan"].close()
        # e2e: C ABI with pinned HOST buffers, copies inside the timed region
        nze = min(w.nz, args.e2e_slices)
        try:
            host = [t[:nze].cpu().pin_memory() for t in (w.a, w.b, w.c, w.d)]
            xh = torch.empty_like(host[3]).pin_memory()
            bze = min(ok[best]["batch"], nze) if ok[best]["batch"] < w.nz else 0
            with tdma.Plan(w.nx, w.ny, nze, w.P, bze, variant=vmap[best]) as hplan:
                for _ in range(2):
                    hplan.solve_host(*host, xh)
                t0 = time.perf_counter()
                reps = 3
                for _ in range(reps):
                    hplan.solve_host(*host, xh)
                el = (time.perf_counter() - t0) / reps
            ecells = w.nx * w.ny * nze
            out["e2e"] = {"value": ecells / el, "unit": UNIT, "h2d_bytes_per_step": 32 * ecells,
                          "d2h_bytes_per_step": 8 * ecells, "ms_per_step": el * 1e3,
                          "pcie_gbs": 40.0 * ecells / el / 1e9,
                          "sample": "first %d of %d z-slices through tdma_solve_host (pinned host buffers, "
                                    "chunks of ~16 Mi cells, H2D / solve / D2H overlapped)" % (nze, w.nz)}
            # cpu baseline on the same host sample (bounded)
            nzc = min(nze, 64)
            rate, reps, el, cores = cpu_oracle_rate([t[:nzc] for t in host], args.cpu_seconds)
            out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                   "sample": "%d z-slices (%d cells) x %d repeats, %.1f s" % (nzc, w.nx * w.ny * nzc, reps, el)}
            del host, xh
        except Exception as exc:                      # report, never hide
            out["e2e_error"] = repr(exc)
        # a second BASELINE workload (cfg 5, pipeline stress), same harness
        if args.also and args.also != args.workload and args.nz == 0:
            plan.close()
            del w, x
            torch.cuda.empty_cache()
            try:
                out["workloads"] = {args.also: second_workload(torch, tdma, tdma_inputs, args.also, dev,
                                                               args.steps, warmup, barrier, peak)}
            except Exception as exc:
                out["workloads"] = {args.also: {"error": repr(exc)}}
            # NEXT row f3: the headline config in the paper's own form (shared 1-D coefficients,
            # complex and real right-hand sides), each with its own 32 / 16 B per cell roofline
            for tag, cplx in (("c128", True), ("f64", False)):
                torch.cuda.empty_cache()
                key = "%s_shared_%s" % (args.workload, tag)
                try:
                    out["workloads"][key] = shared_workload(torch, tdma, tdma_inputs, args.workload, cplx, dev,
                                                            args.steps, warmup, barrier, peak,
                                                            cpu_seconds=args.cpu_seconds / 2)
                except Exception as exc:
                    out["workloads"][key] = {"error": repr(exc)}
            # NEXT row f1: BASELINE cfg 4, the ADI step (x periodic, y Dirichlet, z periodic) in the general
            # form, the matrix-sharing form and the uniform-matrix form, each sweep checked against the oracle
            torch.cuda.empty_cache()
            try:
                w4 = tdma_inputs.make_workload("cfg4_adi_y", device=dev)
                x4 = torch.empty_like(w4.d)
                a4 = argparse.Namespace(steps=args.steps, warmup=warmup, workload="cfg4_adi_y")
                out["workloads"]["cfg4_adi"] = adi(torch, tdma, w4, x4, a4, barrier, rank, peak, emit=False)
                del w4, x4
            except Exception as exc:
                out["workloads"]["cfg4_adi"] = {"error": repr(exc)}
    if rank == 0:
        print(json.dumps(out))
    group.close()
    return 0


def timeline_overlap(torch, tdma, w, x, variant, batch, ns, warmup=3):
    """One solve of a stage-pipeline plan with per-launch timing events (options.timeline): how much
    of stage B's time lies inside the union of the stage A / C intervals of other batches."""
    with tdma.Plan(w.nx, w.ny, w.nz, w.P, batch, variant=variant, nstreams=ns, timeline=1) as plan:
        for _ in range(warmup):
            plan.solve(w.a, w.b, w.c, w.d, x)
        torch.cuda.synchronize()
        plan.solve(w.a, w.b, w.c, w.d, x)
        recs = plan.timeline()
    names = {0: "A", 1: "G", 2: "B", 3: "C"}
    t0 = min(r[2] for r in recs)
    recs = sorted(((names[r[0]], r[1], r[2] - t0, r[3] - t0) for r in recs), key=lambda r: r[2])
    ac = sorted((r[2], r[3]) for r in recs if r[0] in "AC")
    def covered(lo, hi):                       # length of [lo, hi] covered by the union of A/C intervals
        tot, cur = 0.0, lo
        for s0, s1 in ac:
            s0, s1 = max(s0, cur), min(s1, hi)
            if s1 > s0:
                tot += s1 - s0
                cur = s1
        return tot
    tb = sum(r[3] - r[2] for r in recs if r[0] == "B")
    tb_hidden = sum(covered(r[2], r[3]) for r in recs if r[0] == "B")
    return {"launches": len(recs), "span_ms": max(r[3] for r in recs),
            "sum_ms": {k: sum(r[3] - r[2] for r in recs if r[0] == k) for k in "ABC"},
            "stage_b_overlapped_frac": tb_hidden / tb if tb > 0 else None}, recs


def timeline(torch, tdma, w, x, args, batch, rank):
    """Stream-overlap timeline of a stage pipeline (Alg. 2): how much of stage B's time runs while a
    stage A or C kernel of another batch is running.  Plain stream launches (no graph)."""
    ns = args.nstreams or 2
    var = tdma.TDMA_VARIANT_STAGED if args.variant == "staged" else tdma.TDMA_VARIANT_PIPELINED
    stats, recs = timeline_overlap(torch, tdma, w, x, var, batch, ns, max(3, args.warmup))
    rec = {"timeline": True, "workload": args.workload, "variant": "staged" if var == tdma.TDMA_VARIANT_STAGED else "pipelined",
           "batch": batch, "nstreams": ns, **stats,
           "note": "events bracket each launch on its stream: an interval includes the time the kernel "
                   "waits for SM slots, so overlapped_frac is an upper bound of true co-execution"}
    if rank == 0:
        rec["first_launches"] = [{"stage": r[0], "batch": r[1], "start_ms": round(r[2], 4), "end_ms": round(r[3], 4)}
                                 for r in recs[:60]]
        print(json.dumps(rec))
    return 0


def yslab(torch, tdma, w, args, rank, peak):
    """SURVEY 8(f) f4, what ONE B200 can measure of it: the rank-local stages of the y-slab
    decomposition (tdma_slab_stage_a / _b / _c) for one interior rank of an --yslab N job whose
    global slab is the workload (rank-local slab: nx x ny/N x nz), timed stage by stage, plus the
    per-batch exchange sizes and what they would take at the profiling guide's 770 GB/s peer-copy
    rate.  The all-to-alls themselves are NOT measured (one GPU): the record says so."""
    from paper_2509_03933_b200.yslab import CudaSlabStages
    n, r = args.yslab, args.yslab // 2
    nyl = w.ny // n
    batch = 32 if args.batch < 0 else args.batch
    loc = [t[:, r * nyl:(r + 1) * nyl, :].contiguous() for t in (w.a, w.b, w.c, w.d)]
    x = torch.empty_like(loc[3])
    st = CudaSlabStages(w.nx, nyl, w.nz, 1, batch, r, n)
    tma, pl = st.tma, st.P
    lb, ls = st.batch_lines(0)
    send = torch.zeros((n, pl, 6, ls), dtype=torch.float64, device=loc[0].device)
    yout = torch.zeros((n, 2 * pl, ls), dtype=torch.float64, device=loc[0].device)
    stream = torch.cuda.current_stream()
    nbf = w.nz // st.bz                                  # full batches only
    def timed(fn):
        for q in range(min(nbf, 3)):
            fn(q)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(args.steps):
            for q in range(nbf):
                fn(q)
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / (args.steps * nbf)
    t_a = timed(lambda q: st.stage_a(q, *loc, send, stream))
    # a stand-in for the exchange, so that stage B sees a consistent system: every source rank
    # contributes this rank's rows for the receiver's share of the lines
    recv = send[r].unsqueeze(0).expand(n, pl, 6, ls).contiguous()
    t_b = timed(lambda q: st.stage_b(q, recv, yout, stream))
    yrecv = yout[r].unsqueeze(0).expand(n, 2 * pl, ls).contiguous()
    t_c = timed(lambda q: st.stage_c(q, yrecv, x, stream))
    # the stages fused with their exchange (peer stores): every block goes straight into a receiver's
    # ring -- here n separate buffers on this GPU standing in for the n ranks' memory
    rings = [[torch.zeros(n * pl * 6 * ls, dtype=torch.float64, device=loc[0].device) for _ in range(n)] for _ in range(3)]
    yrings = [[torch.zeros(n * 2 * pl * ls, dtype=torch.float64, device=loc[0].device) for _ in range(n)] for _ in range(3)]
    for slot in range(3):
        st.set_peers(slot, rings[slot], yrings[slot])
    t_ap = timed(lambda q: st.stage_a_peer(q, *loc, stream))
    t_bp = timed(lambda q: st.stage_b_peer(q, recv, stream))
    st.close()
    cells = w.nx * nyl * st.bz
    out_b, back_b = 48 * pl * lb, 16 * pl * lb
    rec = {"yslab": True, "workload": args.workload, "nranks": n, "rank_timed": r, "nx": w.nx, "ny_local": nyl, "nz": w.nz,
           "batch": st.bz, "stage_ms_per_batch": {"A": t_a, "B": t_b, "C": t_c},
           "peer_store_stage_ms_per_batch": {"A": t_ap, "B": t_bp,
                                             "note": "stage A / B storing straight into n receive rings (all on this GPU): "
                                                     "no send / yout buffer and no all-to-all; what a real job adds is "
                                                     "NVLink store latency and one barrier per exchange"},
           "stage_kernels": "tma-staged (stage A 32 B/cell, stage C 40 B/cell, nothing spilled)" if tma else
                            "one thread per (line, partition) (stage A 56 B/cell, stage C 32 B/cell, a', c', d' through HBM)",
           "stage_gbs": {"A": (32.0 if tma else 56.0) * cells / t_a / 1e6, "C": (40.0 if tma else 32.0) * cells / t_c / 1e6},
           "exchange_bytes_per_batch": {"A2B": out_b, "B2C": back_b},
           "exchange_ms_at_770GBs": {"A2B": out_b / 770e6, "B2C": back_b / 770e6},
           "rank_cells_per_s_if_exchange_hidden": w.nx * nyl * w.nz / ((t_a + t_c) * (w.nz / st.bz) * 1e-3),
           "measured": "rank-local stages on one B200; the two all-to-alls per batch are unmeasured (one GPU)"}
    if rank == 0:
        print(json.dumps(rec))
    return 0


def adi(torch, tdma, w, x, args, barrier, rank, peak, emit=True):
    """BASELINE cfg 4: ADI implicit viscous sweeps, three batched solves per step (x and z periodic,
    y Dirichlet with P partitions), each a FUSED plan of its own; x1 -> x2 -> x3 chained as in an
    ADI step.  One JSON line: time per sweep and for the whole step (emit = False: the record is
    returned instead, for the default line's `workloads`)."""
    F = tdma.TDMA_VARIANT_FUSED
    plans = [("x", tdma.Plan(w.nx, w.ny, w.nz, w.P, 0, variant=F, axis=tdma.TDMA_AXIS_X, periodic=1)),
             ("y", tdma.Plan(w.nx, w.ny, w.nz, w.P, 0, variant=F)),
             ("z", tdma.Plan(w.nx, w.ny, w.nz, w.P, 0, variant=F, axis=tdma.TDMA_AXIS_Z, periodic=1))]
    y = torch.empty_like(x)
    stream = torch.cuda.current_stream()
    bufs = [(w.d, x), (x, y), (y, x)]
    def step():
        for (name, plan), (src, dst) in zip(plans, bufs):
            plan.solve(w.a, w.b, w.c, src, dst, stream)
    for _ in range(max(3, args.warmup)):
        step()
    torch.cuda.synchronize()
    barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    tot = [0.0, 0.0, 0.0]
    for _ in range(args.steps):
        ev[0].record(stream)
        for i, ((name, plan), (src, dst)) in enumerate(zip(plans, bufs)):
            plan.solve(w.a, w.b, w.c, src, dst, stream)
            ev[i + 1].record(stream)
        torch.cuda.synchronize()
        for i in range(3):
            tot[i] += ev[i].elapsed_time(ev[i + 1])
    ms = [t / args.steps for t in tot]
    rec = {"adi": True, "workload": args.workload, "nx": w.nx, "ny": w.ny, "nz": w.nz, "P": w.P,
           "ms_x_periodic": ms[0], "ms_y": ms[1], "ms_z_periodic": ms[2], "ms_step": sum(ms),
           "cells_per_s_step": 3 * w.cells / (sum(ms) * 1e-3),
           "gbs_40B": {n: 40.0 * w.cells / (m * 1e-3) / 1e9 for n, m in zip("xyz", ms)},
           "frac_of_measured_peak": {n: 40.0 * w.cells / (m * 1e-3) / 1e9 / peak for n, m in zip("xyz", ms)}}
    if rank == 0:
        # checker leg (untimed): every sweep of the last step against the oracle on sampled
        # z-slices (x, y sweeps) / y-planes (z sweep); chain: d -x-> x -y-> y -z-> x, so the x
        # sweep's output was overwritten by the z sweep and is re-solved once for the check
        import numpy as np
        import oracle
        def err(src, dst, axis, periodic, picks):
            worst = 0.0
            for q in picks:
                sl = (slice(None), slice(q, q + 1)) if axis == "z" else (slice(q, q + 1),)
                an, bn, cn, dn, xn = [t[sl].cpu().numpy() for t in (w.a, w.b, w.c, src, dst)]
                ref = oracle.solve_axis(an, bn, cn, dn, axis, periodic)
                ax = {"y": 1, "z": 0, "x": 2}[axis]
                worst = max(worst, float((np.max(np.abs(xn - ref), axis=ax) / np.max(np.abs(ref), axis=ax)).max()))
            return worst
        picks_z = sorted({0, 1, w.nz // 2 + 1, w.nz - 1})
        picks_y = sorted({0, 1, w.ny // 2 + 1, w.ny - 1})
        e_z = err(y, x, "z", True, picks_y)
        x1 = torch.empty_like(x)
        plans[0][1].solve(w.a, w.b, w.c, w.d, x1, stream)
        torch.cuda.synchronize()
        e_x = err(w.d, x1, "x", True, picks_z)
        e_y = err(x1, y, "y", False, picks_z)
        rec["parity_check"] = {"E_max": {"x": e_x, "y": e_y, "z": e_z}, "tol": 1e-11,
                               "slices": {"x": picks_z, "y": picks_z, "z_planes": picks_y},
                               "ok": bool(max(e_x, e_y, e_z) <= 1e-11)}
        # The same three sweeps in the matrix-sharing form (tdma_solve_shared): the
        # ADI matrix is the same for every line, so only d and x travel (16 B/cell).  d -> xs -> y -> x
        # as above; checked against the same oracle on the same sampled slices / planes.
        dev_ = x.device
        alpha = float(-w.a[0, 1, 0].item())
        def coef(n):
            return (torch.full((n,), -alpha, dtype=torch.float64, device=dev_),
                    torch.full((n,), 1.0 + 2.0 * alpha, dtype=torch.float64, device=dev_),
                    torch.full((n,), -alpha, dtype=torch.float64, device=dev_))
        zero = lambda n: torch.zeros(n, dtype=torch.float64, device=dev_)
        sxp = tdma.Plan(w.nx, w.ny, w.nz, 1, 0, axis=tdma.TDMA_AXIS_X, periodic=1)
        sy = tdma.Plan(w.nx, w.ny, w.nz, 1, 0)
        sz_ = tdma.Plan(w.nx, w.ny, w.nz, 1, 0, axis=tdma.TDMA_AXIS_Z, periodic=1)
        ax_, bx_, cx_ = coef(w.nx)
        ay, by, cy = coef(w.ny)
        az, bz_, cz = coef(w.nz)
        zx, zz, zyy = zero(w.nx), zero(w.nz), zero(w.ny)
        xs = torch.empty_like(x)
        def shared_leg(uniform):
            """zero shift arrays (general matrix-sharing form) or no shift arrays (uniform matrix)"""
            def sstep(evs=None):
                for i, (pl_, co, sh, src, dst) in enumerate(((sxp, (ax_, bx_, cx_), (zyy, zz), w.d, xs),
                                                             (sy, (ay, by, cy), (zx, zz), xs, y),
                                                             (sz_, (az, bz_, cz), (zx, zyy), y, x))):
                    pl_.solve_shared(*co, *((None, None) if uniform else sh), src, dst, stream=stream)
                    if evs is not None:
                        evs[i + 1].record(stream)
            for _ in range(3):
                sstep()
            torch.cuda.synchronize()
            ev2 = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            ts = [0.0, 0.0, 0.0]
            for _ in range(args.steps):
                ev2[0].record(stream)
                sstep(ev2)
                torch.cuda.synchronize()
                for i in range(3):
                    ts[i] += ev2[i].elapsed_time(ev2[i + 1])
            ms_s = [t / args.steps for t in ts]
            out = {"ms_x_periodic": ms_s[0], "ms_y": ms_s[1], "ms_z_periodic": ms_s[2], "ms_step": sum(ms_s),
                   "gbs_16B": {n: 16.0 * w.cells / (m * 1e-3) / 1e9 for n, m in zip("xyz", ms_s)},
                   "frac_of_measured_peak_16B": {n: 16.0 * w.cells / (m * 1e-3) / 1e9 / peak for n, m in zip("xyz", ms_s)},
                   "E_max": {"x": err(w.d, xs, "x", True, picks_z), "y": err(xs, y, "y", False, picks_z),
                             "z": err(y, x, "z", True, picks_y)}, "tol": 1e-11}
            out["ok"] = bool(max(out["E_max"].values()) <= 1e-11)
            return out
        rec["shared_form"] = shared_leg(False)
        # sx = sz = NULL: the matrix work hoisted out of the tile loop (every line has the same matrix)
        rec["uniform_matrix_form"] = shared_leg(True)
        sxp.close()
        sy.close(); sz_.close()
        if emit:
            print(json.dumps(rec))
    for _, plan in plans:
        plan.close()
    return 0 if emit else rec


def sweep(torch, tdma, w, x, args, barrier, rank):
    """S7: batch x stream sweep; one JSON line per point."""
    nz = w.nz
    batches = [b for b in (1, 2, 4, 8, 16, 32, 64, 128) if b <= nz]
    points = []
    vm = {"fused": tdma.TDMA_VARIANT_FUSED, "pipelined": tdma.TDMA_VARIANT_PIPELINED, "staged": tdma.TDMA_VARIANT_STAGED}
    for variant, streams_list in (("pipelined", (1, 2, 3, 4)), ("staged", (1, 2, 3, 4)), ("fused", (1,))):
        for ns in streams_list:
            for bz in batches + ([0] if variant == "fused" else []):
                opts = dict(variant=vm[variant])
                if variant != "fused":
                    opts["nstreams"] = ns
                try:
                    with tdma.Plan(w.nx, w.ny, nz, w.P, bz, **opts) as plan:
                        sec = time_solve(torch, plan, w, x, args.steps, max(3, args.warmup), barrier)
                        rec = {"sweep": True, "workload": args.workload, "variant": variant, "nstreams": ns,
                               "batch": plan.get(tdma.TDMA_GET_BATCH), "nb": plan.get(tdma.TDMA_GET_NB),
                               "ms": sec * 1e3, "cells_per_s": w.cells / sec,
                               "gbs_40B": 40.0 * w.cells / sec / 1e9,
                               "workspace_MiB": plan.workspace_bytes / 2 ** 20}
                except tdma.TdmaError as exc:
                    rec = {"sweep": True, "variant": variant, "nstreams": ns, "batch": bz, "error": str(exc)}
                points.append(rec)
                if rank == 0:
                    print(json.dumps(rec), flush=True)
    return 0


if __name__ == "__main__":
    sys.exit(main())
