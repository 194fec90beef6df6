#!/usr/bin/env python
"""bench.py -- Yee cell-updates/s of the FDTD hot path on B200 (BASELINE.json metric).

One "step" = one whole pass of the hot path over one synthetic problem: fdtd_forward with interface
recording (F1..F8) + the caller's loss cotangent + fdtd_backward (B0..B5) + the rho chain rule (B6).
Default workload: the graded config C3 (200^3, 12-cell CPML, 2000 time steps, 864k design voxels).

    value  = cells * n_time_steps * K / (time of K steps), summed over ranks, with record=1: the recorder on
             the PML / interior interface, the whole interior reconstructed (t_fwd(record=1) +
             t_bwd, 161 B/cell/step on C3);
    fwd    = cells * n_time_steps / t_fwd(record=0);
    n1_design_box_recorder = the same gradient with record=2 (faces of the design box
             recorded, only that box reconstructed; 135 B/cell/step on C3), a named extra beside `value`.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload c3|c4|c5] [--grid N] [--time-steps T] [--record 1|2|both]

N > 1 (torchrun): every rank runs an independent problem (seed + rank), no data-path collective
("weak" scaling over independent inverse-design problems).
--impl reference times the CPU oracle (oracle/, fp32 build, all host cores) on a bounded sample.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

METRIC = "Yee cell-updates/s, forward(record=1) + time-reversed backward (gradient)"
UNIT = "Mcells/s"
KERNEL_SOURCES = ("kernels_step.cu", "kernels_generic.cu", "fused_common.cuh", "fdtd_internal.h")


def kernel_source_hash() -> str:
    """sha256 over the kernel sources: profiles/traffic.json records the hash of the build its ncu capture was taken on."""
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        h.update((ROOT / "paper_2412_12360_b200" / "csrc" / name).read_bytes())
    return h.hexdigest()


# ------------------------------------------------------------------------------------------------
# algorithmic bytes: what one launch of each kernel class must move
# ------------------------------------------------------------------------------------------------
def algorithmic_bytes(w, grad_cells: int, recording: bool, has_mu: bool = False, rbox=None) -> dict:
    """rbox = (bx, by, bz): the reconstruction box (record=2: the design box; default: the interior I)."""
    nx, ny, nz, d = w.nx, w.ny, w.nz, w.pml_cells
    cells = nx * ny * nz
    bx, by, bz = rbox if rbox else (nx - 2 * d, ny - 2 * d, nz - 2 * d)
    inter = bx * by * bz
    slab = 2 * d * (ny * nz + nx * nz + nx * ny)            # slab cells summed over the three axes
    face = 4 * (by * bz + bx * bz + bx * by) if d else 0
    mu = 4 if has_mu else 0
    rec = 4 * face if recording else 0                      # 2 comps x 2 sides per face cell, fp32
    return {
        # fused step: 6 R + 6 W fields + ie (+im); psi R/W: 4 arrays (2E+2H) per slab cell per axis; with the recorder
        # on, the face recorder runs beside the step kernel (side stream) and is timed with it
        "fused_forward_step": cells * (52 + mu) + slab * 32 + 2 * rec,
        # fused adjoint step (B2+B5): 6 R + 6 W cotangents + ie over the grid, adjoint psi R/W on slabs; the face
        # injection of the reverse sweep runs beside it and is timed with it
        "fused_adjoint_step": cells * (52 + mu) + slab * 32 + 2 * rec,
        # fused inverse step (B3+B4) over the box: R E',H' (6), ie, W E,H (6); on the grad box also R lamE' (3) and g R/W
        "fused_inverse_step": inter * (52 + mu) + grad_cells * 20,
        "update_E": cells * 40 + slab * 16,
        "update_H": cells * (36 + mu) + slab * 16,
        "adjoint_H": cells * (36 + mu) + slab * 16,
        "adjoint_E": cells * 40 + slab * 16,
        "inverse_H": inter * (36 + mu),
        "inverse_E_grad": inter * 52 + grad_cells * 8,
        "record_faces": 2 * 4 * face,
        "inject_faces": 2 * 4 * face,
    }


def whole_job_bytes_per_cell_step(w, grad_cells: int, rbox=None) -> dict:
    """SURVEY 8(d) whole-job figures per cell and time step: forward alone (6 R + 6 W + inv_eps + psi on the slabs), and
    forward + adjoint pass + inverse pass + g, where the inverse pass counts 12 floats per box cell (R E', H'; W E, H):
    inv_eps and lamE' are counted once, with the adjoint pass (13 + 12 + 2 floats; C3: 63.5 / 161.0).
    The per-kernel figure of k_inverse (algorithmic_bytes) is 13 floats per box cell and 16 on the gradient box because as a
    launch of its own it has to read inv_eps and (where the gradient is formed) lamE' again; the whole-job roofline is not
    credited with that re-read."""
    a0 = algorithmic_bytes(w, grad_cells, recording=False)
    d = w.pml_cells
    bx, by, bz = rbox if rbox else (w.nx - 2 * d, w.ny - 2 * d, w.nz - 2 * d)
    c = float(w.cells)
    return {"fwd": a0["fused_forward_step"] / c,
            "fwd_bwd": (2 * a0["fused_forward_step"] + bx * by * bz * 48 + grad_cells * 8) / c}


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.idx), "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 9:
                continue
            try:
                sm.append(float(parts[1])); mx.append(float(parts[2]))
            except ValueError:
                continue
            for nm, val in zip(names, parts[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
def make_workload(args, rank: int = 0):
    from paper_2412_12360_b200 import workloads as wl
    from paper_2412_12360_b200 import sharding
    if args.workload == "c4":
        w = wl.c4(n_steps=args.time_steps or 5000)
        w.meta.setdefault("delta_eps", 12.25 - 2.085)
    elif args.workload == "c5":
        w = wl.c5(args.grid or 256, n_steps=args.time_steps or 500)          # configs[4]: loss over I, gradient on all of I
    else:
        w = wl.c3(n=args.grid or 200, n_steps=args.time_steps or 2000, seed=sharding.problem_seed(3, rank))
    return w


def oracle_loss_cotangents(w, f, phasors):
    """The caller's loss on the oracle side (numpy), same definitions as the GPU leg."""
    import numpy as np
    if w.loss == "phasor_power":
        return [2.0 * P if i in w.loss_detectors else None for i, P in enumerate(phasors)], None
    dLf = np.zeros_like(f)
    d = w.pml_cells
    sl = (slice(0, 3), slice(d, w.nz - d), slice(d, w.ny - d), slice(d, w.nx - d))
    dLf[sl] = 2.0 * f[sl]
    return None, dLf


def cpu_oracle_rate(w, sample_steps: int, threads: int = 0):
    """Times the oracle as it stands (fp32 build, OpenMP, FTZ on) on the first `sample_steps` time steps of the
    workload: forward with recording + reversible backward.  threads = 0: all host cores."""
    import numpy as np
    from oracle.oracle import Oracle
    o = Oracle(**w.grid_kwargs(), dtype=np.float32)
    all_cores = os.cpu_count() or 1
    o.set_num_threads(threads if threads > 0 else all_cores)
    o.set_ftz(True)
    f = np.zeros((6, w.nz, w.ny, w.nx), dtype=np.float32)
    t0 = time.perf_counter()
    out = o.forward(f, w.inv_eps, None, w.sources, w.detectors, sample_steps, record=w.pml_cells > 0)
    t1 = time.perf_counter()
    dLp, dLf = oracle_loss_cotangents(w, f, out["phasors"])
    o.backward(f, w.inv_eps, None, w.sources, w.detectors, dLp, dLf, sample_steps, out["rec"])
    t2 = time.perf_counter()
    cells = w.cells * sample_steps
    res = {"value": cells / (t2 - t0) / 1e6, "fwd_value": cells / (t1 - t0) / 1e6, "unit": UNIT,
           "cores": o.num_threads(), "kind": "oracle",
           "sample": f"{w.name} {w.nx}x{w.ny}x{w.nz} grid, first {sample_steps} of {w.n_steps} time steps, "
                     f"forward(record)+reversible backward, fp32 build of oracle/fdtd_oracle.c, OpenMP, FTZ"}
    o.set_num_threads(all_cores)
    return res


def workload_config(w, extra=None):
    cfg = {"workload": f"{w.name}: {w.nx}x{w.ny}x{w.nz} fp32 Yee grid, {w.pml_cells}-cell CPML, {w.n_steps} time steps, "
                       f"forward(record=1: PML/interior interface)+reversible backward over the whole interior, "
                       + ("gradient on the design region" if w.design_lo else "gradient on the whole interior"),
           "time_steps": w.n_steps, "cells": w.cells,
           "l2": "inputs larger than L2 (working set > 0.5 GB vs 126 MB L2); no flush needed" if w.cells * 52 > 126e6
                 else "grid fits in L2: fractions of the HBM roofline may exceed 1 (SURVEY 8(d))"}
    if extra:
        cfg.update(extra)
    return cfg


def run_reference(args, rank):
    """--impl reference: the CPU oracle on the host cores (bounded sample per step)."""
    if rank != 0:
        return
    w = make_workload(args)
    sample = args.ref_sample_steps
    for _ in range(args.warmup):
        cpu_oracle_rate(w, max(1, sample // 4))
    t0 = time.perf_counter()
    rates = [cpu_oracle_rate(w, sample) for _ in range(args.steps)]
    dt = time.perf_counter() - t0
    val = w.cells * sample * args.steps / sum(w.cells * sample / (r["value"] * 1e6) for r in rates) / 1e6
    cb = dict(rates[-1]); cb["value"] = val
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                      "data": "synthetic", "config": workload_config(w, {"sample_time_steps": sample}),
                      "cpu_baseline": cb,
                      "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


# ------------------------------------------------------------------------------------------------
def run_decomposed(args, rank, world, local_rank, barrier):
    """--decompose z: one grid, `world` z slabs, one halo exchange per time step (include/fdtd.h "Domain decomposition").
    Forward pass and adjoint sweep of the whole grid; value = cells * time_steps / time, strong scaling."""
    import torch
    from paper_2412_12360_b200 import binding as B
    from paper_2412_12360_b200 import sharding
    w = make_workload(args)                                   # the same problem on every rank: each takes its slab
    T = args.time_steps or min(w.n_steps, 200)
    dev = torch.device("cuda", local_rank)
    seed = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32, device=dev)
    seed[1, w.nz // 2] = 1.0                                  # a fixed cotangent seed for the adjoint sweep
    if world == 1 and args.slabs > 1:
        # one process, one device: the slabs in lock step on one stream (what the exchange costs in launches and copies,
        # not a scaling figure: the slabs run one after the other)
        runners = [sharding.SlabRunner(B, w, s, T, record=0) for s in sharding.z_slabs(w.nz, args.slabs, w.pml_cells)]
        peer = args.halo in ("peer", "flags") and all(q.grid.info().path == B.FDTD_PATH_FUSED for q in runners)
        if peer and args.halo == "flags":
            peer = "flags"                                    # + the wait / signal kernels (met at once on one stream)

        def fwd1():
            for q in runners:
                q.fields.zero_()
                for P in q.phasors:
                    P.zero_()
            sharding.run_slabs_lockstep(runners, T, "forward", peer=peer)

        def adj1():
            for q in runners:
                q.want_grad = False
                q.set_cotangents(None, seed)
            sharding.run_slabs_lockstep(runners, T, "backward", peer=peer)

        def timed1(fn, reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1)

        for _ in range(args.warmup):
            fwd1()
        ms_f = timed1(fwd1, args.steps)
        adj1()
        ms_a = timed1(adj1, max(1, min(args.steps, 3)))
        cs = w.cells * T
        print(json.dumps({"metric": "Yee cell-updates/s, forward pass of ONE grid cut into z slabs run in lock step on ONE device",
                          "value": cs * args.steps / (ms_f * 1e-3) / 1e6, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms_f / args.steps, "higher_is_better": True, "scaling": "none (one device)",
                          "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": workload_config(w, {"time_steps": T, "parallelism": f"{args.slabs} z slabs on one device, " + (
                                                            ("peer stores + device-side ordering kernels" if peer == "flags" else "peer stores (no exchange launches)") if peer else "plane copies between the steps (fdtd_halo_export / _import)"),
                                                        "slab_planes": [q.slab.nz for q in runners]}),
                          "us_per_time_step": {"forward": 1e3 * ms_f / args.steps / T, "adjoint": 1e3 * ms_a / max(1, min(args.steps, 3)) / T},
                          "adjoint_sweep": {"value": cs * max(1, min(args.steps, 3)) / (ms_a * 1e-3) / 1e6, "unit": UNIT},
                          "gpu_launches": int(sum(q.grid.info().kernel_launches for q in runners))}))
        for q in runners:
            q.close()
        return
    slab = sharding.z_slabs(w.nz, world, w.pml_cells)[rank]
    r = sharding.SlabRunner(B, w, slab, T, record=0)

    # --halo peer: the fused step kernels store the halo planes into the neighbours' volumes (CUDA IPC mappings, opened
    # once per direction outside the timed region); --halo nccl: plane copies + NCCL point-to-point between the launches
    # --halo flags: peer stores + the device-side ordering kernels (no token either; ranges of 64 steps per call)
    peer = args.halo in ("peer", "flags") and r.grid.info().path == B.FDTD_PATH_FUSED
    use_flags = args.halo == "flags"
    links = {0: sharding.PeerLinks(r, 0, flags=use_flags) if peer else False}

    def fwd():
        r.fields.zero_()
        for P in r.phasors:
            P.zero_()
        sharding.run_slab_distributed(r, T, "forward", peer=links[0])

    def adj():
        r.set_cotangents(None, seed)
        if 1 not in links:
            links[1] = sharding.PeerLinks(r, 1, flags=use_flags) if peer else False
        sharding.run_slab_distributed(r, T, "backward", peer=links[1])

    def timed(fn, reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        barrier()
        return sharding.max_over_ranks(e0.elapsed_time(e1), device=dev)

    for _ in range(args.warmup):
        fwd()
    ms_f = timed(fwd, args.steps)
    r.want_grad = False                                       # adjoint sweep only (dL_dinv_eps = NULL)
    adj()
    ms_a = timed(adj, max(1, min(args.steps, 3)))
    info = r.grid.info()
    if rank == 0:
        cs = w.cells * T
        print(json.dumps({"metric": "Yee cell-updates/s, forward pass of ONE grid cut into z slabs (strong scaling)",
                          "value": cs * args.steps / (ms_f * 1e-3) / 1e6, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms_f / args.steps, "higher_is_better": True, "scaling": "strong",
                          "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                          "config": workload_config(w, {"time_steps": T, "parallelism": f"z slabs x{world}, " + (
                                                            "halo planes stored by the step kernels into the neighbours' volumes (peer stores), " + ("ordered by flags on the device" if use_flags else "one token per neighbour and step")
                                                            if peer else "one halo exchange per time step (3 planes of nx*ny floats per neighbour and direction, NCCL point-to-point)"),
                                                        "slab_planes": slab.nz, "path": {1: "generic", 2: "fused"}[info.path]}),
                          "adjoint_sweep": {"value": cs * max(1, min(args.steps, 3)) / (ms_a * 1e-3) / 1e6, "unit": UNIT},
                          "gpu_launches": int(info.kernel_launches)}))
    for l in links.values():
        if l:
            l.close()
    r.close()


def run_n4(args):
    """bench.py --n4: the SURVEY 8(f) N4 variants on C3's grid and recipe, timed like `value` (CUDA events around whole gradient
    passes, inputs resident): per-component inv_eps, dL/d inv_mu, the checkpointed reverse sweep and a lossy medium.  One JSON line."""
    import math
    import numpy as np
    import torch
    from paper_2412_12360_b200 import binding as B
    args.time_steps = args.time_steps or 600
    w = make_workload(args, 0)
    T = w.n_steps
    dev = torch.device("cuda", 0)
    stream = torch.cuda.Stream()
    shape = (w.nz, w.ny, w.nx)
    rng = np.random.default_rng(5)
    ie = torch.as_tensor(w.inv_eps).to(dev)
    ie3 = torch.stack([ie * float(a) for a in (1.0, 0.95, 1.05)]).contiguous()
    im = torch.as_tensor((1.0 / (1.0 + 0.2 * rng.random(shape, dtype=np.float32))).astype(np.float32)).to(dev)
    sig = torch.as_tensor((0.02 * rng.random(shape, dtype=np.float32)).astype(np.float32)).to(dev)
    for q in w.sources:
        q.waveform = torch.as_tensor(q.waveform).to(dev)
        q.profile = None if q.profile is None else torch.as_tensor(q.profile).to(dev)
    K = max(1, int(round(math.sqrt(T))))
    fields = torch.zeros((6,) + shape, dtype=torch.float32, device=dev)
    phasors = [torch.zeros(dt.phasor_shape, dtype=torch.float32, device=dev) for dt in w.detectors]
    reps = max(1, min(args.steps, 3))
    rows = {}

    def case(name, record, flags=0, eps=ie, mu=None, sigma=None, grad_mu=False, ck=0):
        kw = w.grid_kwargs()
        kw.update(max_steps=T, record=record, flags=flags, checkpoint_every=ck, grad_lo=w.design_lo, grad_hi=w.design_hi)   # gradient on the design region, as `value`
        g = B.Grid(**kw)
        if sigma is not None:
            g.set_conductivity(sigma)
        gm = torch.empty(shape, dtype=torch.float32, device=dev) if grad_mu else None

        def fwd():
            fields.zero_()
            for P in phasors:
                P.zero_()
            g.forward(fields, eps, mu, w.sources, w.detectors, T, phasors=phasors)

        def grad():
            fwd()
            dLp = [2.0 * P if i in w.loss_detectors else None for i, P in enumerate(phasors)]
            return g.backward(fields, eps, mu, w.sources, w.detectors, dLp, None, T, grad_mu=gm)[0]

        def timed(fn):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            fn()
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(reps):
                out = fn()
            e1.record(stream)
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / reps, out

        with torch.cuda.stream(stream):
            ms_f, _ = timed(fwd)
            ms_g, gr = timed(grad)
            info = g.info()
            rows[name] = {"path": {B.FDTD_PATH_FUSED: "fused", B.FDTD_PATH_GENERIC: "generic"}[info.path],
                          "forward_Mcells_s": round(w.cells * T / ms_f / 1e3, 1), "forward_us_per_time_step": round(1e3 * ms_f / T, 1),
                          "gradient_Mcells_s": round(w.cells * T / ms_g / 1e3, 1), "gradient_us_per_time_step": round(1e3 * ms_g / T, 1),
                          "recorder_GB": round(info.recorder_bytes / 1e9, 2), "max_abs_grad": float(gr.double().abs().max())}
        g.close()

    case("isotropic, time-reversed (record=1): the contract's path", 1)
    case("inv_mu volume + dL/d inv_mu (fdtd_backward_mu)", 1, mu=im, grad_mu=True)
    case("per-component inv_eps (FDTD_FLAG_ANISO_EPS), time-reversed", 1, flags=B.FDTD_FLAG_ANISO_EPS, eps=ie3)
    case(f"isotropic, checkpointed reverse sweep (record=3, every {K} steps)", 3, ck=K)
    case(f"lossy medium (fdtd_set_conductivity), checkpointed reverse sweep (record=3, every {K} steps)", 3, sigma=sig, ck=K)
    print(json.dumps({"n4": "SURVEY 8(f) N4 variants on C3's grid and recipe", "grid": list(shape[::-1]), "time_steps": T,
                      "passes_timed": reps, "unit": "Mcells/s = cells * time steps / time of forward (or forward + backward)", "rows": rows}))


def run_probe(args):
    """bench.py --probe: what the memory system gives for the step kernel's bytes and traversal, without its arithmetic."""
    import torch
    from paper_2412_12360_b200 import binding as B
    N = args.grid or 200
    vin = torch.rand((7, N, N, N), device="cuda")
    vout = torch.empty((6, N, N, N), device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    peaks_file = ROOT / "MEASURED_PEAKS.json"
    if peaks_file.exists():
        peaks = {"hbm_gbs": float(json.loads(peaks_file.read_text())["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json hbm_gbs)"}
    else:
        peaks = {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)"}
    rows = []

    def one(label, pattern, tile_y=0, runs=1, unroll=1, blocks=0, threads=256):
        gbs = B.fdtd_probe_bandwidth(pattern, N, N, N, tile_y, runs, unroll, blocks, threads, 20, vin, vout, st)
        us = 13 * 4 * N ** 3 * (runs if pattern == 0 else 1) / gbs / 1e3
        rows.append({"probe": label, "GB/s": round(gbs, 1), "us": round(us, 1), "frac_of_peak": round(gbs / peaks["hbm_gbs"], 3)})

    for b in (4, 8, 16):
        one(f"stream {sms * b}x256", 0, blocks=sms * b, threads=256)
    if 13 * 4 * N ** 3 < 60e6:                  # fits in L2: many passes per launch = the L2 <-> SM rate of this mix
        one(f"stream {sms * 8}x256, 20 passes per launch (L2 resident)", 0, runs=20, blocks=sms * 8, threads=256)
        one(f"stream {sms * 8}x512, 20 passes per launch (L2 resident)", 0, runs=20, blocks=sms * 8, threads=512)
    for ty, runs, u, th in ((7, 5, 1, 384), (7, 5, 2, 384), (7, 5, 4, 384), (7, 10, 1, 384), (7, 10, 2, 384), (7, 20, 2, 384),
                            (14, 10, 2, 512), (28, 20, 2, 512)):
        nb = (N + ty - 1) // ty * runs
        one(f"tile {N}x{ty} runs={runs} unroll={u} ({nb} blocks x {th}, {nb / sms:.2f}/SM)", 1, ty, runs, u, threads=th)
    # the hand-over from one time step to the next: ping-pong volumes, marching upwards every time (2) or alternating (3)
    for ty, runs, u, th in ((7, 5, 2, 384), (7, 10, 2, 384)):
        nb = (N + ty - 1) // ty * runs
        one(f"tile {N}x{ty} runs={runs} unroll={u}, ping-pong volumes, every launch marches upwards ({nb} blocks)", 2, ty, runs, u, threads=th)
        one(f"tile {N}x{ty} runs={runs} unroll={u}, ping-pong volumes, marching direction alternates ({nb} blocks)", 3, ty, runs, u, threads=th)
    print(json.dumps({"probe": "7 volumes read + 6 written, float4 per thread, no arithmetic (fdtd_probe_bandwidth)",
                      "grid": [N, N, N], "bytes_per_launch": 13 * 4 * N ** 3, "peak_hbm_gbs": peaks["hbm_gbs"],
                      "peak_source": peaks["source"], "rows": rows}))


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--time-steps", type=int, default=0, help="FDTD time steps per gradient (default: the config's: C3 2000, C4 5000, C5 500)")
    ap.add_argument("--grid", type=int, default=0, help="grid size per axis: C3 recipe scaled to N^3 (default 200), C5 N (default 256)")
    ap.add_argument("--workload", default="c3", choices=["c3", "c4", "c5"],
                    help="c3: the graded config (default); c4: configs[3], 800x800x600 memory-scale run; c5: configs[4], the size sweep")
    ap.add_argument("--path", default="auto", choices=["auto", "generic", "fused"])
    ap.add_argument("--ref-sample-steps", type=int, default=12)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--lean", action="store_true",
                    help="memory-scale runs: no second (forward-only) grid, hence no forward-only and adjoint-only passes")
    ap.add_argument("--decompose", default="", choices=["", "z"],
                    help="z: ONE grid cut into z slabs, one per rank (SURVEY 8(e) / 8(f) N3; sharding.run_slab_distributed, NCCL "
                         "point-to-point halo exchange once per time step); times the forward pass and the adjoint sweep of the whole "
                         "grid (strong scaling).  Not measured on more than one GPU in this build: see DESIGN.md section 10")
    ap.add_argument("--slabs", type=int, default=0,
                    help="--decompose z on ONE rank: cut the grid into this many z slabs and run them in lock step on the one device "
                         "(sharding.run_slabs_lockstep): the cost of the exchange in launches and copies, with --halo peer | nccl (= plane copies)")
    ap.add_argument("--halo", default="peer", choices=["peer", "flags", "nccl"],
                    help="--decompose z: peer = the fused step kernels store the halo planes into the neighbours' volumes (include/fdtd.h "
                         "\"Peer stores\"; falls back to nccl on a grid that runs the generic kernels), one token per neighbour and step; "
                         "flags = peer stores ordered on the device (wait / signal kernels beside the step kernel, no token; one GPU per rank only); "
                         "nccl = plane copies + NCCL point-to-point")
    ap.add_argument("--recorder-fp16", action="store_true",
                    help="SURVEY 8(f) N1: store the interface record as fp16 (FDTD_FLAG_RECORDER_FP16; an approximation, off by default)")
    ap.add_argument("--record", default="", choices=["", "1", "2", "both"],
                    help="1: `value` only (record the PML/interior interface, reconstruct the interior); 2: `value` on the "
                         "design-box recorder instead (labelled); both (default where there is a design box and memory allows): "
                         "`value` on record=1 and the record=2 figure beside it")
    ap.add_argument("--n4", action="store_true",
                    help="SURVEY 8(f) N4 variants on C3 (per-component inv_eps, dL/d inv_mu, checkpointed sweep, lossy medium): forward "
                         "and gradient rates, one JSON line (--time-steps, default 600)")
    ap.add_argument("--probe", action="store_true",
                    help="no FDTD: the bandwidth probes of fdtd_probe_bandwidth (the step kernel's 7 volumes read + 6 written "
                         "without its arithmetic, streaming and in the step kernel's tile-column traversal) on the --grid size "
                         "(default 200), one JSON line; DESIGN.md section 8")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2412_12360_b200 import binding as B
    from paper_2412_12360_b200 import workloads as wl
    from paper_2412_12360_b200 import sharding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.probe or args.n4:
        if rank == 0:
            (run_probe if args.probe else run_n4)(args)
        if world > 1:
            dist.destroy_process_group()
        return

    if args.decompose == "z":
        run_decomposed(args, rank, world, local_rank, barrier)
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- workload (seed + rank: every rank an independent problem) ---------------------------------
    w = make_workload(args, rank)
    T = w.n_steps
    has_box = w.design_lo is not None
    rec_arg = args.record or ("both" if has_box and args.workload != "c4" else ("2" if args.workload == "c4" else "1"))
    if not has_box:
        rec_arg = "1"
    main_record = 2 if rec_arg == "2" else 1
    path = {"auto": B.FDTD_PATH_AUTO, "generic": B.FDTD_PATH_GENERIC, "fused": B.FDTD_PATH_FUSED}[args.path]
    d = w.pml_cells
    dlo, dhi = (w.design_lo, w.design_hi) if has_box else ((d, d, d), (w.nx - d, w.ny - d, w.nz - d))

    def make_grid(record, staging=False):
        kw = w.grid_kwargs()
        kw.update(max_steps=T, record=record, path=path,
                  flags=(B.FDTD_FLAG_HOST_STAGING if staging else 0) | (B.FDTD_FLAG_RECORDER_FP16 if args.recorder_fp16 else 0))
        if has_box:
            kw.update(grad_lo=dlo, grad_hi=dhi)
        return B.Grid(**kw)

    grid = make_grid(main_record, staging=not args.no_e2e)          # the `value` grid
    grid2 = make_grid(2) if rec_arg == "both" else None             # N1 extra: design-box recorder
    grid_f = None if args.lean else make_grid(0)                    # forward-only grid (no recorder)
    stream = torch.cuda.Stream()
    dev = torch.device("cuda", local_rank)
    ie = torch.as_tensor(w.inv_eps).to(dev)
    fields = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32, device=dev)
    for s in w.sources:                                        # resident descriptors
        s.waveform = torch.as_tensor(s.waveform).to(dev)
        s.profile = None if s.profile is None else torch.as_tensor(s.profile).to(dev)
    phasors = [torch.zeros(dt.phasor_shape, dtype=torch.float32, device=dev) for dt in w.detectors]
    grad = torch.empty((w.nz, w.ny, w.nx), dtype=torch.float32, device=dev)
    drho = torch.empty((dhi[2] - dlo[2], dhi[1] - dlo[1], dhi[0] - dlo[0]), dtype=torch.float32, device=dev) if has_box else None
    grad_cells = (dhi[0] - dlo[0]) * (dhi[1] - dlo[1]) * (dhi[2] - dlo[2])
    delta_eps = float(w.meta.get("delta_eps", 0.0))
    dLf_buf = torch.zeros_like(fields) if w.loss != "phasor_power" else None
    inter = (slice(0, 3), slice(d, w.nz - d), slice(d, w.ny - d), slice(d, w.nx - d))

    def loss_cotangents():
        """The caller's loss (torch ops on the caller's side of the ABI): phasor power or sum E^2 over I."""
        if w.loss == "phasor_power":
            return [2.0 * P if i in w.loss_detectors else None for i, P in enumerate(phasors)], None
        dLf_buf[inter] = 2.0 * fields[inter]
        return None, dLf_buf

    def gradient_step(g):
        """One pass of the whole hot path, inputs resident in HBM."""
        fields.zero_()
        for P in phasors:
            P.zero_()
        g.forward(fields, ie, None, w.sources, w.detectors, T, phasors=phasors)
        dLp, dLf = loss_cotangents()
        g.backward(fields, ie, None, w.sources, w.detectors, dLp, dLf, T, out=grad)
        if has_box:
            B.fdtd_grad_rho(g.h, grad, ie, delta_eps, dlo, dhi, drho, g.stream())

    def forward_only(g):
        fields.zero_()
        for P in phasors:
            P.zero_()
        g.forward(fields, ie, None, w.sources, w.detectors, T, phasors=phasors)

    def timed(fn, reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        barrier()
        return sharding.max_over_ranks(e0.elapsed_time(e1), device=dev)

    def loss_value():
        if w.loss == "phasor_power":
            return float(sum((P.double() ** 2).sum() for i, P in enumerate(phasors) if i in w.loss_detectors))
        return None

    with torch.cuda.stream(stream):
        for _ in range(args.warmup):
            gradient_step(grid)
        l0 = grid.info().kernel_launches
        sampler = ClockSampler(local_rank)
        sampler.start()
        ms_total = timed(lambda: gradient_step(grid), args.steps)
        clocks = sampler.stop()
        launches = grid.info().kernel_launches - l0
        loss = loss_value()
        gnorm = float((drho if has_box else grad).double().abs().max())

        # N1 extra: the same gradient with the design-box recorder (record=2)
        n1 = None
        if grid2 is not None:
            reps2 = max(1, min(args.steps, 3))
            for _ in range(min(args.warmup, 2)):
                gradient_step(grid2)
            ms2 = timed(lambda: gradient_step(grid2), reps2)
            n1 = {"value": sharding.whole_job_rate(w.cells * T, reps2, ms2, world), "unit": UNIT, "ms_per_step": ms2 / reps2,
                  "max_abs_dL_drho": float(drho.double().abs().max()), "loss": loss_value()}

        # the recorded forward pass of the same grid alone: splits `ms_per_step` into forward(record) and reverse sweep
        reps_fr = max(1, min(args.steps, 3))
        ms_fwd_rec = timed(lambda: forward_only(grid), reps_fr) / reps_fr

        ms_fwd = ms_adj = None
        reps_adj = max(1, min(args.steps, 3))
        if grid_f is not None:
            # forward-only (record=0) rate, same workload
            for _ in range(min(args.warmup, 2)):
                forward_only(grid_f)
            ms_fwd = timed(lambda: forward_only(grid_f), max(1, args.steps))

            # adjoint sweep only (dL_dinv_eps = NULL: one k_step<adjoint> launch per time step), same cotangent seed
            dLp_t, dLf_t = loss_cotangents()

            def adjoint_only(g):
                g.backward(fields, ie, None, w.sources, w.detectors, dLp_t, dLf_t, T, want_grad=False)

            adjoint_only(grid_f)
            ms_adj = timed(lambda: adjoint_only(grid_f), reps_adj)

        # ---- per-kernel roofline: one more pass with every step kernel bracketed by CUDA events --------
        B.fdtd_set_profiling(grid.h, True)
        B.fdtd_get_profile(grid.h)
        gradient_step(grid)
        torch.cuda.synchronize()
        prof = B.fdtd_get_profile(grid.h)
        B.fdtd_set_profiling(grid.h, False)

    cells_steps = w.cells * T
    value = sharding.whole_job_rate(cells_steps, args.steps, ms_total, world)
    fwd_value = sharding.whole_job_rate(cells_steps, max(1, args.steps), ms_fwd, world) if ms_fwd else None

    peaks_file = ROOT / "MEASURED_PEAKS.json"
    if peaks_file.exists():
        peak, peak_src = float(json.loads(peaks_file.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    else:
        peak, peak_src = 6650.0, "fallback (B200_PROFILING.md)"
    dbox = tuple(dhi[a] - dlo[a] for a in range(3))
    rbox_main = dbox if (main_record == 2 and has_box) else None
    alg = algorithmic_bytes(w, grad_cells, recording=True, rbox=rbox_main)
    kernels = {}
    for name, (n, ms) in prof.items():
        if name in alg and n:
            gbs = alg[name] * n / (ms * 1e-3) / 1e9
            kernels[name] = {"launches": n, "avg_us": ms / n * 1e3, "alg_bytes_per_launch": alg[name],
                             "achieved_gbs": gbs, "frac": gbs / peak, "share_of_step": None}
        else:
            kernels[name] = {"launches": n, "avg_us": ms / n * 1e3 if n else None}
    tot_ms = sum(ms for _, ms in prof.values()) or 1.0
    for name, (n, ms) in prof.items():
        kernels[name]["share_of_step"] = ms / tot_ms
    info = grid.info()
    info_path_fused = info.path == 2
    dom = max((k for k in kernels if "achieved_gbs" in kernels[k]), key=lambda k: prof[k][1], default=None)
    # the two instances of k_step take the same share of the step to within a percent, so which one is "largest" flips
    # from run to run: report the adjoint instance (the slower one; round 1 reported it too), the forward instance beside it
    if dom == "fused_forward_step" and "fused_adjoint_step" in kernels and prof["fused_adjoint_step"][1] > 0.9 * prof[dom][1]:
        dom = "fused_adjoint_step"
    roofline = None
    if dom:
        # dram bytes per launch from the committed ncu --set full capture; refused when the kernel sources changed since
        traffic, traffic_note = None, "no profiles/traffic.json"
        tf = ROOT / "profiles" / "traffic.json"
        if tf.exists():
            tj = json.loads(tf.read_text())
            if tj.get("kernel_source_sha256") != kernel_source_hash():
                traffic_note = "profiles/traffic.json was captured on other kernel sources (hash mismatch): not reported"
            elif tj.get("workload") not in (None, w.name) or (tj.get("grid") not in (None, [w.nx, w.ny, w.nz])):
                traffic_note = "profiles/traffic.json was captured on another workload: not reported"
            else:
                traffic, traffic_note = tj.get(dom), tj.get("how", "ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum per launch")
        roofline = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["achieved_gbs"], "peak": peak,
                    "peak_source": peak_src, "unit": "GB/s", "frac": kernels[dom]["frac"], "traffic": traffic,
                    "traffic_note": traffic_note,
                    "alg_bytes_per_launch": alg[dom], "avg_launch_us": kernels[dom]["avg_us"],
                    "frac_of_8000": kernels[dom]["achieved_gbs"] / 8000.0}
        # the same kernel template inside the replayed CUDA graph (no events between launches): the forward-only
        # pass is one k_step launch per time step, so its time / launches is that kernel's launch-to-launch period
        if info_path_fused and ms_fwd:
            fb = algorithmic_bytes(w, grad_cells, recording=False)["fused_forward_step"]
            us = ms_fwd / max(1, args.steps) / T * 1e3
            roofline["forward_step_in_graph"] = {"avg_launch_us": us, "alg_bytes_per_launch": fb,
                                                 "achieved": fb / us / 1e3, "frac": fb / us / 1e3 / peak}
            # likewise the adjoint-sweep-only pass: one k_step<adjoint> launch per time step (its time also holds the
            # cotangent seed and the copy of the result: 6 volumes each, once per T launches)
            ab = algorithmic_bytes(w, grad_cells, recording=False)["fused_adjoint_step"]
            us = ms_adj / reps_adj / T * 1e3
            roofline["adjoint_step_in_graph"] = {"avg_launch_us": us, "alg_bytes_per_launch": ab,
                                                 "achieved": ab / us / 1e3, "frac": ab / us / 1e3 / peak}
            # headline = the dominant kernel as it runs in the job (replayed graph, back-to-back launches, CUDA events
            # around the timed region / launches); the figure with events around every single launch stays beside it
            ing = {"fused_adjoint_step": "adjoint_step_in_graph", "fused_forward_step": "forward_step_in_graph"}.get(dom)
            if ing:
                roofline["events_around_every_launch"] = {k: roofline[k] for k in ("achieved", "frac", "avg_launch_us", "frac_of_8000")}
                g_ = roofline[ing]
                roofline.update(achieved=g_["achieved"], frac=g_["frac"], avg_launch_us=g_["avg_launch_us"],
                                alg_bytes_per_launch=g_["alg_bytes_per_launch"], frac_of_8000=g_["achieved"] / 8000.0,
                                method=f"{ing}: CUDA events around a pass of {T} back-to-back launches of this kernel "
                                       "in the replayed graph, time / launches")
        # the reverse sweep as it runs in the job (grouped launches): ms_per_step minus the recorded forward pass; what it
        # takes beyond the adjoint-sweep-only pass is the inverse step (+ face injection) inside the job, without the launch
        # latency that "events around every launch" adds to it
        rev_us = (ms_total / args.steps - ms_fwd_rec) / T * 1e3
        rs = {"forward_with_recorder_us_per_time_step": ms_fwd_rec / T * 1e3, "reverse_sweep_us_per_time_step": rev_us}
        if ms_adj and "fused_inverse_step" in kernels:
            inv_us = rev_us - ms_adj / reps_adj / T * 1e3
            ib = kernels["fused_inverse_step"]["alg_bytes_per_launch"]
            rs["inverse_step_in_job"] = {"avg_launch_us": inv_us, "alg_bytes_per_launch": ib, "achieved": ib / inv_us / 1e3,
                                         "frac": ib / inv_us / 1e3 / peak,
                                         "how": "reverse sweep per time step minus the adjoint-sweep-only pass per time step"}
        roofline["in_job"] = rs
        # whole-job fractions: algorithmic B/cell/step x rate against the measured peak and the 8000 GB/s bar
        bpc = whole_job_bytes_per_cell_step(w, grad_cells, rbox=rbox_main)
        wj = {f"fwd_bwd_record{main_record}": {"bytes_per_cell_step": bpc["fwd_bwd"], "achieved": bpc["fwd_bwd"] * value / world / 1e3}}
        if fwd_value:
            wj["fwd"] = {"bytes_per_cell_step": bpc["fwd"], "achieved": bpc["fwd"] * fwd_value / world / 1e3}
        if n1 is not None:
            b2 = whole_job_bytes_per_cell_step(w, grad_cells, rbox=dbox)["fwd_bwd"]
            wj["fwd_bwd_record2"] = {"bytes_per_cell_step": b2, "achieved": b2 * n1["value"] / world / 1e3}
            n1["bytes_per_cell_step"] = b2
        for v in wj.values():
            v["frac"] = v["achieved"] / peak
            v["frac_of_8000"] = v["achieved"] / 8000.0
        roofline["whole_job"] = wj

    # ---- end to end through the host-buffer C ABI (pinned host memory, H2D/D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        h_ie = torch.as_tensor(w.inv_eps).pin_memory()
        h_grad = torch.empty((w.nz, w.ny, w.nx), dtype=torch.float32).pin_memory()
        h_ph = [torch.zeros(dt.phasor_shape, dtype=torch.float32).pin_memory() for dt in w.detectors]
        h_cot = [torch.zeros(dt.phasor_shape, dtype=torch.float32).pin_memory() for dt in w.detectors]
        field_loss = w.loss != "phasor_power"
        h_fields = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32).pin_memory() if field_loss else None
        h_dLf = torch.zeros((6, w.nz, w.ny, w.nx), dtype=torch.float32).pin_memory() if field_loss else None
        host_src = [wl.Source(s.component, s.lo, s.hi, s.waveform.cpu().numpy(),
                              None if s.profile is None else s.profile.cpu().numpy()) for s in w.sources]
        sarr, ns, k1 = grid.marshal_sources(host_src, host=True)
        darr, nd, k2 = grid.marshal_detectors(w.detectors, h_ph)
        import ctypes as C
        cot = (C.c_void_p * max(nd, 1))()
        for i in range(nd):
            cot[i] = h_cot[i].data_ptr() if i in w.loss_detectors else None
        sp = C.c_void_p(stream.cuda_stream)
        vol = h_ie.numel() * 4
        h2d = vol * 2 + sum(p.numel() * 4 for p in h_ph) + sum(h_cot[i].numel() * 4 for i in w.loss_detectors)
        h2d += sum(s.waveform.size * 4 + (0 if s.profile is None else s.profile.size * 4) for s in host_src) * 2
        d2h = vol + sum(p.numel() * 4 for p in h_ph)
        if field_loss:            # the final state goes to the host for the caller's loss, its cotangent comes back
            h2d += 6 * vol * 2
            d2h += 6 * vol

        def e2e_step():
            for P in h_ph:
                P.zero_()
            if field_loss:
                h_fields.zero_()
            B.fdtd_forward_host(grid.h, h_fields, h_ie, None, sarr, ns, darr, nd, T, sp)
            for i in w.loss_detectors:
                torch.mul(h_ph[i], 2.0, out=h_cot[i])                      # caller's loss cotangent on the host
            if field_loss:
                h_dLf[inter] = 2.0 * h_fields[inter]
            B.fdtd_backward_host(grid.h, None, h_ie, None, sarr, ns, darr, nd, cot if nd else None, h_dLf, T, h_grad, None, sp)

        with torch.cuda.stream(stream):
            e2e_step()
            reps = max(1, min(args.steps, 3))
            ms_e2e = timed(e2e_step, reps)
        e2e = {"value": world * cells_steps * reps / (ms_e2e * 1e-3) / 1e6, "unit": UNIT,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "ms_per_step": ms_e2e / reps,
               "api": "fdtd_forward_host + fdtd_backward_host (pinned host buffers, staging allocated by fdtd_create_grid)"}

    info = grid.info()
    if rank == 0:
        cpu = None
        if not args.no_cpu_baseline and world == 1:
            wc = make_workload(args)
            cpu = cpu_oracle_rate(wc, args.ref_sample_steps)
            one = cpu_oracle_rate(wc, max(2, args.ref_sample_steps // 4), threads=1)
            cpu["one_thread"] = {"value": one["value"], "fwd_value": one["fwd_value"], "unit": UNIT, "cores": 1,
                                 "sample_time_steps": max(2, args.ref_sample_steps // 4)}
        rec_names = {1: "PML/interior interface, record=1 (SURVEY 8(d))", 2: "faces of the design box, record=2 (SURVEY 8(f) N1)"}
        out = {"metric": METRIC if main_record == 1 else METRIC.replace("record=1", "record=2"),
               "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
               "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
               "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
               "config": workload_config(w, {"path": {1: "generic", 2: "fused"}[info.path],
                                             "tile": [info.tile_x, info.tile_y, info.tile_z],
                                             "parallelism": f"independent problems x{world}",
                                             "partition": B.PARTITION_NAMES.get(int(info.partition), str(info.partition)),
                                             "reverse_sweep": "grouped launches" if info.pipelined_inverse_ctas else "sequential",
                                             "recorder": rec_names[main_record] + (", fp16 (FDTD_FLAG_RECORDER_FP16)" if args.recorder_fp16 else ""),
                                             "recorder_bytes": int(info.recorder_bytes), "scratch_bytes": int(info.scratch_bytes)}),
               "fwd": {"value": fwd_value, "unit": UNIT, "ms_per_pass": ms_fwd / max(1, args.steps),
                       "what": "forward only, record=0, same workload"} if ms_fwd else None,
               "n1_design_box_recorder": n1,
               "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
               "roofline": roofline, "kernels": kernels, "cpu_baseline": cpu,
               "check": {"loss": loss, "max_abs_grad": gnorm,
                         "device_bytes": {"caller_torch_peak": int(torch.cuda.max_memory_allocated()),
                                          "grid_recorder": int(info.recorder_bytes), "grid_scratch": int(info.scratch_bytes)}}}
        print(json.dumps(out))
    grid.close()
    if grid_f is not None:
        grid_f.close()
    if grid2 is not None:
        grid2.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
