#!/usr/bin/env python
"""bench.py -- coupled LBM-IBM MLUPS and fraction of the HBM roofline versus marker density on one B200
(BASELINE.json metric), ONE JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload W4] [--impl ours|reference]

A "step" is one pass of the whole hot path: one time step of the coupled scheme (kinematics, marker sort + chunks +
tiles + collect plan, moments on active cells, mdf_iters x (tile pass = interpolate + correct + sweep, collect), fused
stream-collide-force), replayed as one CUDA graph.

`value` is measured on W4 (BASELINE.json configs[3]: 256^3 periodic, 64 three-blade propellers, 1,179,648 markers,
5 MDF iterations): the coupled configuration on the SAME 256^3 lattice as the pure-LBM bandwidth case configs[1] (W2),
so that coupled / pure is like for like.  The metric is a curve, not a point: `density_sweep` carries the same
measurement for W3, W3x4 (the propeller of W3 with four times the markers), W4lit, W4, W5lit, W5 (the largest single-GPU
configuration, configs[4]) and the paper-shaped cases P1 / P6 / P18 (P:231-237's own sweep over 1 -> 6 -> 18 propellers).  All inputs are seeded synthetic
(paper_1904_02108_b200/workloads.py).

N > 1: "replicas only": every rank runs the same workload on its own GPU, no data-path collective;
value = units of all ranks / max-over-ranks time.

--impl reference times the fp64 CPU oracle (oracle/) on the host cores on the same workload at full size.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "coupled LBM-IBM MLUPS"
UNIT = "MLUPS"
NOMINAL_HBM_GBS = 8000.0       # north_star's denominator
# B200 fp32 FMA peak for the ALU-bound tile pass: 148 SMs x 128 fp32 lanes x 2 flop x 1.965 GHz
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
SWEEP = ["W3", "W3x4", "W4lit", "W4", "W5lit", "W5", "P1", "P6", "P18"]
PAPER_MLUPS = {"P1": 893.0, "P6": 650.0, "P18": 344.2}
ORACLE_FULL_MAX_CELLS = 1 << 25      # the fp64 oracle at full size up to 256^3 x 2 (W5: 512^3 needs ~48 GB and minutes per step)


# ---- algorithmic bytes ---------------------------------------------------------------------------
def step_bytes(cells, n_active, n_markers, mdf, sort_passes):
    """What the method itself must move per time step, fp32: a8 152 B per cell + 12 B of G per active cell; a4
    (76 + 16) B per active cell; per MDF iteration 36 B per active cell + 88 B per marker; a2 + a3 40 B per marker +
    16 B per marker and radix pass."""
    if n_markers == 0 or mdf == 0:
        return 152.0 * cells
    return (152.0 * cells + (12.0 + 92.0 + 36.0 * mdf) * n_active
            + (88.0 * mdf + 40.0 + 16.0 * sort_passes) * n_markers)


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def traffic_from_profile(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the stream-collide kernel from the newest
    committed ncu --set full summary (profiles/traffic_rNN.csv), or (None, None).  NOT measured in this run."""
    try:
        pdir = os.path.join(ROOT, "profiles")
        files = sorted(f for f in os.listdir(pdir) if f.startswith("traffic_r") and f.endswith(".csv"))
        for name in reversed(files):
            with open(os.path.join(pdir, name)) as fh:
                for line in fh.read().splitlines()[1:]:
                    if line.split(",", 1)[0] == workload:
                        return float(line.rsplit(",", 1)[1]), f"profiles/{name} (ncu --set full, builder run; not measured in this run)"
    except Exception:
        pass
    return None, None


class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.QUERY}",
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1]))
            except ValueError:
                continue
            for n, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            # under load = the upper half of the samples (the sampler also sees idle gaps)
            s = sorted(sm)
            out["sm_mhz"] = float(np.median(s[len(s) // 2:]))
            out["sm_max_mhz"] = float(max(mx))
        out["reasons"] = sorted(reasons)
        return out


def time_steps(torch, sim, stream, steps, mdf):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        sim.step(steps, mdf)
        e1.record(stream)
    stream.synchronize()
    return e0.elapsed_time(e1)          # ms


def host_info():
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    ram = None
    try:
        with open("/proc/meminfo") as fh:
            for line in fh:
                if line.startswith("MemTotal"):
                    ram = round(int(line.split()[1]) / 1048576.0, 1)
                    break
    except OSError:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count() or 1, "ram_gb": ram}


# ---- the oracle on the host cores ----------------------------------------------------------------------------------
def oracle_case(workload_name, seed):
    """The oracle as it stands on the SAME workload at full size; W5 / W5lit (512^3: ~48 GB of fp64 populations and
    minutes per step) run their recipe in a 256^3 box with the same body density."""
    import oracle
    from paper_1904_02108_b200 import workloads
    wl = workloads.get(workload_name, seed)
    same = True
    what = f"{workload_name} at full size ({wl.nx}x{wl.ny}x{wl.nz}, {wl.n_markers} markers)"
    if wl.cells > ORACLE_FULL_MAX_CELLS:
        wl = workloads.w5(seed, 12 if workload_name == "W5" else 1, n=256)
        same = False
        what = f"{workload_name} recipe in a 256^3 box ({len(wl.bodies)} propellers, {wl.n_markers} markers)"
    return oracle.from_workload(wl), wl, what, same


def time_oracle(ref, wl, steps, warmup):
    if warmup:
        ref.step(warmup, wl.mdf_iters)
    t0 = time.perf_counter()
    ref.step(steps, wl.mdf_iters)
    dt = time.perf_counter() - t0
    return wl.cells * steps / dt / 1e6, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    info = host_info()
    ref, wl, what, same = oracle_case(args.workload, args.seed)
    # a step of the full-size oracle takes seconds: bound the run to a few minutes
    per_step_guess = wl.cells / 12e6
    steps = max(1, min(args.steps, int(150.0 / max(per_step_guess, 1e-3))))
    warm = min(args.warmup, 1)
    mlups, dt = time_oracle(ref, wl, steps, warm)
    sample = f"{what}, {steps} steps timed" + ("" if steps == args.steps else f" (of the {args.steps} asked for: bounded to minutes)")
    line = {
        "impl": "reference", "metric": METRIC, "value": mlups, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded)",
        "config": {"workload": args.workload, "lattice": [wl.nx, wl.ny, wl.nz], "markers": wl.n_markers,
                   "mdf_iters": wl.mdf_iters, "same_config_as_gpu_arm": same, "sample": sample, "host": info},
        "cpu_baseline": {"value": mlups, "unit": UNIT, "cores": info["nproc"], "kind": "oracle", "sample": sample},
        "e2e": {"value": mlups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---- one workload on the GPU: coupled step, pure LBM on the same lattice, sizes -----------------------------------
def gpu_case(torch, api, wl, stream, steps, warmup, opts=()):
    sim = api.from_workload(wl, stream=stream)
    for k, v in opts:
        sim.set_option(k, v)
    mdf = wl.mdf_iters
    sim.step(warmup, mdf)
    stream.synchronize()
    warm_until(torch, sim, stream, mdf)
    ms = time_steps(torch, sim, stream, steps, mdf) / steps
    sim.sync()
    out = {"sim": sim, "ms": ms}
    if wl.n_markers:
        out["active_cells"] = sim.get_info(api.INFO_ACTIVE_CELLS)
        out["active_words"] = sim.get_info(api.INFO_ACTIVE_WORDS)
        out["tiles"] = sim.get_info(api.INFO_TILES)
        out["tile_rows"] = sim.get_info(api.INFO_TILE_ROWS)
        out["layout"] = sim.get_info(api.INFO_LAYOUT)
        out["sort_passes"] = sim.get_info(api.INFO_SORT_PASSES)
    else:
        out.update(active_cells=0, active_words=0, tiles=0, tile_rows=0, layout=0, sort_passes=0)
    return out


def warm_until(torch, sim, stream, mdf, seconds=0.05):
    """Sweep entries: small workloads finish their few warm-up steps in well under a millisecond, before the clocks
    have settled; keep stepping (untimed) until `seconds` of device work have passed."""
    t0 = time.perf_counter()
    while time.perf_counter() - t0 < seconds:
        sim.step(10, mdf)
        stream.synchronize()


def pure_ms(torch, sim, stream, steps, settle=False):
    sim.step(3, 0)
    stream.synchronize()
    if settle:
        warm_until(torch, sim, stream, 0)
    return time_steps(torch, sim, stream, steps, 0) / steps


def sweep_entry(name, wl, case, ms_pure, peak):
    ms = case["ms"]
    nbytes = step_bytes(wl.cells, case["active_cells"], wl.n_markers, wl.mdf_iters, case["sort_passes"])
    gbs = nbytes / (ms * 1e-3) / 1e9
    e = {"workload": name, "lattice": [wl.nx, wl.ny, wl.nz], "markers": wl.n_markers, "bodies": len(wl.bodies),
         "mdf_iters": wl.mdf_iters, "active_cells": int(case["active_cells"]),
         "markers_per_lattice_cell": wl.n_markers / wl.cells,
         "markers_per_active_cell": wl.n_markers / max(1, case["active_cells"]),
         "active_cell_fraction": case["active_cells"] / wl.cells,
         "ms_per_step": ms, "mlups": wl.cells / (ms * 1e-3) / 1e6,
         "pure_ms_per_step": ms_pure, "pure_mlups": wl.cells / (ms_pure * 1e-3) / 1e6,
         "coupled_over_pure": ms_pure / ms, "ibm_share": max(0.0, 1.0 - ms_pure / ms),
         "step_algorithmic_bytes": nbytes, "step_gbs": gbs, "step_hbm_frac": gbs / peak,
         "step_hbm_frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS,
         "tiles": int(case["tiles"]), "tile_rows": int(case["tile_rows"]), "step_layout": int(case["layout"])}
    if name in PAPER_MLUPS:
        e["paper_context"] = {"mlups": PAPER_MLUPS[name], "hardware": "Tesla P100-PCIE (P:229-237)",
                              "note": "paper's Blender mesh replaced by a synthetic propeller of the same point count"}
    return e


def run_ours(args):
    import torch
    if not torch.cuda.is_available():
        print(json.dumps({"error": "no CUDA device: this library has no CPU fallback"}))
        return 2
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    from paper_1904_02108_b200 import replicas
    dist = replicas.init("nccl", rank, world, device=torch.device("cuda", local))

    from paper_1904_02108_b200 import api, workloads
    wl = workloads.get(args.workload, args.seed)
    mdf = wl.mdf_iters
    stream = torch.cuda.Stream()
    sim = api.from_workload(wl, stream=stream)
    user_opts = []
    if args.spread != "gather":
        user_opts.append((api.OPT_SPREAD, {"atomic": 1, "plain": 2}[args.spread]))
    if args.lbm_kernel != "auto":
        user_opts.append((api.OPT_LBM_KERNEL, {"scalar": 1, "vec4": 2}[args.lbm_kernel]))
    for kv in args.opt:
        name, val = kv.split("=")
        user_opts.append((getattr(api, "OPT_" + name.upper()), int(val)))
    for k, v in user_opts:
        sim.set_option(k, v)
    overlap_user = dict(user_opts).get(api.OPT_OVERLAP, 3)

    def barrier():
        torch.cuda.synchronize()
        replicas.barrier(dist)
        torch.cuda.synchronize()

    peak, how = measured_peak_gbs()

    # ---- device-resident timing (the headline `value`) ------------------------------------------
    sim.step(args.warmup, mdf)
    barrier()
    l0 = sim.get_info(api.INFO_LAUNCHES)
    sampler = ClockSampler(local) if rank == 0 else None
    ms = time_steps(torch, sim, stream, args.steps, mdf)
    barrier()
    launches = sim.get_info(api.INFO_LAUNCHES) - l0
    clocks = sampler.stop() if sampler else {}
    sim.sync()
    ms = replicas.max_over_ranks(ms, dist, device="cuda")
    value = replicas.whole_job_mlups(wl.cells, args.steps, world, ms)
    ms_step = ms / args.steps

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic (seeded)",
        "config": {"workload": wl.name, "lattice": [wl.nx, wl.ny, wl.nz], "tau": wl.tau, "markers": wl.n_markers,
                   "bodies": len(wl.bodies), "mdf_iters": mdf, "spread": args.spread, "lbm_kernel": args.lbm_kernel,
                   "parallelism": "replicas" if world > 1 else "single-gpu",
                   "why_this_workload": "configs[3]: the coupled case on the lattice of the pure-LBM case configs[1], so "
                                        "coupled / pure is like for like; the other densities incl. configs[4] (W5, the "
                                        "largest) are in density_sweep",
                   "l2": "inputs larger than L2 (populations %.0f MB per buffer)" % (wl.cells * 76 / 1e6)},
        "clocks": clocks, "gpu_launches": int(launches),
    }
    if wl.name in PAPER_MLUPS:
        # context, not a baseline: the paper's own MLUPS for the case this synthetic workload is shaped after
        line["config"]["paper_context"] = {"mlups": PAPER_MLUPS[wl.name], "hardware": "Tesla P100-PCIE (P:229-237)",
                                           "note": "paper's Blender mesh replaced by a synthetic propeller of the same point count"}
    if rank == 0:
        n_active = sim.get_info(api.INFO_ACTIVE_CELLS) if wl.n_markers else 0
        n_words = sim.get_info(api.INFO_ACTIVE_WORDS) if wl.n_markers else 0
        layout = sim.get_info(api.INFO_LAYOUT) if wl.n_markers else 0
        tile_rows = sim.get_info(api.INFO_TILE_ROWS) if wl.n_markers else 0
        sort_passes = sim.get_info(api.INFO_SORT_PASSES) if wl.n_markers else 0
        # ---- the same step as one serial chain with a single fused stream-collide pass (comparison) -----
        if wl.n_markers:
            sim.set_option(api.OPT_OVERLAP, 0)
            sim.step(3, mdf)
            ms_serial = time_steps(torch, sim, stream, args.steps, mdf)
            sim.set_option(api.OPT_OVERLAP, overlap_user)
            line["serial_chain"] = {"value": wl.cells * args.steps / (ms_serial * 1e-3) / 1e6, "unit": UNIT,
                                    "ms_per_step": ms_serial / args.steps,
                                    "what": "LBM_OPT_OVERLAP=0: one stream, one fused stream-collide pass"}
        # ---- the paper's own kernel designs on the same step, one option at a time ---------
        if wl.n_markers and args.compare:
            cmp_steps = max(3, min(args.steps, 20))
            variants = [("moments_box(P:209)", {api.OPT_MOMENTS: api.MOMENTS_BOX}),
                        ("moments_block_per_marker(P:215)", {api.OPT_MOMENTS: api.MOMENTS_PER_MARKER}),
                        ("round1_pipeline(interp kernel + TMA tile sweep + collect)", {api.OPT_FUSED: 0}),
                        ("interp_caller_order(ib_force1)", {api.OPT_INTERP: api.INTERP_CALLER_ORDER}),
                        ("interp_warp_per_marker(shuffle_reduce)", {api.OPT_INTERP: api.INTERP_WARP_PER_MARKER}),
                        ("interp_chunk_window_in_smem", {api.OPT_INTERP: api.INTERP_CHUNK_SMEM}),
                        ("spread_atomic_thread_per_marker", {api.OPT_SPREAD: api.SPREAD_ATOMIC}),
                        ("spread_block125_atomic(ib_force2)", {api.OPT_SPREAD: api.SPREAD_BLOCK125}),
                        ("paper_pipeline(box+ib_force1+ib_force2,serial)",
                         {api.OPT_MOMENTS: api.MOMENTS_BOX, api.OPT_INTERP: api.INTERP_CALLER_ORDER,
                          api.OPT_SPREAD: api.SPREAD_BLOCK125, api.OPT_OVERLAP: 0})]
            defaults = {api.OPT_MOMENTS: 0, api.OPT_INTERP: 0, api.OPT_SPREAD: 0, api.OPT_OVERLAP: overlap_user,
                        api.OPT_FUSED: 1}
            comp = {"default": ms_step}
            for name, opts in variants:
                for k, v in opts.items():
                    sim.set_option(k, v)
                sim.step(3, mdf)
                comp[name] = time_steps(torch, sim, stream, cmp_steps, mdf) / cmp_steps
                for k, v in defaults.items():
                    sim.set_option(k, v)
            sim.step(2, mdf)
            line["comparisons_ms_per_step"] = comp
        # ---- per-phase device time with CUDA events on the launching stream (phases run one after the other) --
        n_ph = max(3, min(args.steps, 20))
        sim.set_option(api.OPT_TIMING, 1)
        sim.step(n_ph, mdf)
        ph = {k: v / n_ph for k, v in sim.phase_ms().items()}
        sim.set_option(api.OPT_TIMING, 0)
        lbm_ms = ph["lbm"]
        # the stream-collide pass (a8).  Step layout 1: the bulk pass over every 32-cell word without an active cell
        # (the words pass follows); layout 2 / pure: one pass over all cells (+ 12 B of G per active cell).
        if wl.n_markers and layout == 1:
            lbm_cells = wl.cells - min(wl.cells, n_words * 32)
            alg_bytes = 152.0 * lbm_cells
            kname = "k_stream_collide_scalar<LBM_BULK> (a8, cells outside the marker stencils)"
        else:
            lbm_cells = wl.cells
            alg_bytes = 152.0 * lbm_cells + (12.0 * n_active if wl.n_markers else 0.0)
            kname = "k_stream_collide_scalar<%s> (a8, all cells)" % ("LBM_FUSED" if wl.n_markers else "LBM_PURE")
        achieved = alg_bytes / (lbm_ms * 1e-3) / 1e9
        traffic, traffic_src = traffic_from_profile(wl.name)
        line["roofline"] = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "GB/s",
                            "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                            "peak_source": how, "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                            "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": lbm_ms,
                            "cells_per_launch": int(lbm_cells),
                            "share_of_step": lbm_ms / max(1e-9, sum(ph[k] for k in ("moments", "interp", "spread", "lbm", "lbm_active"))),
                            "note": "the HBM-bound kernel of the path; the kernel with the largest time share of the "
                                    "coupled step is in roofline_ibm, the step as a whole in roofline_step"}
        # the step as a whole against the HBM roofline (the metric): algorithmic bytes of SURVEY 8(d) / step time
        sb = step_bytes(wl.cells, n_active, wl.n_markers, mdf, sort_passes)
        sgbs = sb / (ms_step * 1e-3) / 1e9
        line["roofline_step"] = {"bound": "hbm", "what": "whole coupled step: algorithmic bytes (SURVEY 8(d)) / ms_per_step",
                                 "achieved": sgbs, "peak": peak, "unit": "GB/s", "frac": sgbs / peak,
                                 "frac_of_nominal_8TBs": sgbs / NOMINAL_HBM_GBS, "algorithmic_bytes_per_step": sb,
                                 "traffic": None}
        if wl.n_markers and mdf:
            # the kernel with the largest summed time per step: the tile pass (a5 + a6 + a7 stage A), launched mdf times.
            # Bound by plain fp32 arithmetic and shared-memory traffic, not by HBM: 2 x 64 x 3 FMA per marker and pass
            # (interpolation + spreading) = 768 flop against 148 SMs x 128 lanes x 2 x 1.965 GHz.
            tile_ms = ph["interp"] / mdf
            tfl = 768.0 * wl.n_markers / (tile_ms * 1e-3) / 1e12
            line["roofline_ibm"] = {"bound": "alu", "kernel": "k_mdf_tiles<%d> (a5 + a6 + a7 stage A), %d launches per step" % (tile_rows, mdf),
                                    "achieved": tfl, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": tfl / FP32_PEAK_TFLOPS,
                                    "peak_source": "148 SMs x 128 fp32 lanes x 2 flop x 1.965 GHz (B200_PROFILING.md clocks)",
                                    "algorithmic_flop_per_launch": 768.0 * wl.n_markers, "kernel_ms": tile_ms,
                                    "summed_ms_per_step": ph["interp"],
                                    "share_of_step": ph["interp"] / max(1e-9, sum(ph[k] for k in ("moments", "interp", "spread", "lbm", "lbm_active"))),
                                    "traffic": None,
                                    "collect_kernel_ms": ph["spread"] / mdf,
                                    "note": "issue-slot and shared-memory figures of this kernel: profiles/top_kernels_r2.md"}
        line["phases_ms_per_step"] = ph
        line["phases_note"] = "phases timed one after the other (LBM_OPT_TIMING); in the timed step the binning of the next step runs beside the MDF loop"
        line["active_cells"] = int(n_active)
        line["active_word_cells"] = int(min(wl.cells, n_words * 32))
        line["step_layout"] = int(layout)
        if wl.n_markers:
            line["chunks"] = sim.get_info(api.INFO_RUNS)
            line["chunk_entries"] = sim.get_info(api.INFO_RUN_ENTRIES)
            line["tiles"] = sim.get_info(api.INFO_TILES)
            line["tile_rows"] = int(tile_rows)

        # ---- pure LBM on the same lattice and on configs[1] (W2) ---------------------------------
        ms_p = pure_ms(torch, sim, stream, args.steps)
        pure_same = wl.cells / (ms_p * 1e-3) / 1e6
        line["pure_lbm"] = {"same_lattice_mlups": pure_same,
                            "frac_of_measured": pure_same * 1e6 * 152.0 / 1e9 / peak,
                            "frac_of_nominal_8TBs": pure_same * 1e6 * 152.0 / 1e9 / NOMINAL_HBM_GBS,
                            "coupled_over_pure": value / world / pure_same}
        # share of the coupled step that the IBM adds on top of a pure-LBM step of the same lattice
        line["ibm_share"] = max(0.0, 1.0 - ms_p / ms_step)
        main_entry = None
        if wl.n_markers:
            main_entry = sweep_entry(args.workload, wl, {"ms": ms_step, "active_cells": n_active, "tiles": line["tiles"],
                                          "tile_rows": tile_rows, "layout": layout, "sort_passes": sort_passes}, ms_p, peak)

    # ---- end to end through the public API with host buffers (all ranks) ---------------------------
    # every step: H2D = the per-body kinematics table a host controller sets (ibm_update_kinematics),
    # D2H = the marker forces Delta u(k) into pinned host memory; the fields stay resident, as the method
    # intends ("fully performed within the GPU's memory"); one extra leg reads the fields every 10 steps.
    e2e_steps = max(3, min(args.steps, 20))

    def timed(fn, finish=None, n=e2e_steps):
        fn()
        if finish:
            finish()
        barrier()
        t0 = time.perf_counter()
        for _ in range(n):
            fn()
        if finish:
            finish()
        torch.cuda.synchronize()
        return replicas.max_over_ranks(time.perf_counter() - t0, dist, device="cuda")

    if wl.n_markers:
        nb = len(wl.bodies)
        om = np.array([b.omega for b in wl.bodies]); ax = np.stack([b.axis for b in wl.bodies])
        force_host = torch.empty((wl.n_markers, 3), dtype=torch.float32, pin_memory=True)
        out = {"force": force_host.numpy()}
        h2d, d2h = nb * 56, wl.n_markers * 12

        def e2e_blocking_step():
            sim.update_kinematics(0, om, ax)
            sim.step(1, mdf)
            sim.read_markers(pos=False, perm=False, cell=False, out=out)

        dt_b = timed(e2e_blocking_step)
        # the same loop with the asynchronous read-out of the public API (ibm_read_markers_async): the D2H copy of
        # step n overlaps step n+1; the host consumes the forces of step n-1 (two pinned buffers) every step
        bufs = [torch.empty((wl.n_markers, 3), dtype=torch.float32, pin_memory=True) for _ in range(2)]
        state = {"k": 0, "sum": 0.0, "om": om.copy()}

        def make_async(change_omega):
            def fn():
                if change_omega:
                    # a controller that changes the rotation rates every step: the set binned ahead for the next
                    # step is discarded and the step bins its markers in line (no binning overlap)
                    state["om"] = om * (1.0 + 1e-7 * ((state["k"] & 1) * 2 - 1))
                sim.update_kinematics(0, state["om"] if change_omega else om, ax)
                sim.step(1, mdf)                                     # step k is enqueued ...
                sim.wait_markers()                                   # ... while the forces of step k-1 finish landing on the host
                state["sum"] += float(bufs[(state["k"] + 1) & 1][0, 0])   # the host controller reads them
                sim.read_markers_async(bufs[state["k"] & 1])         # read-out of step k, ordered behind it on the device
                state["k"] += 1
            return fn

        dt = timed(make_async(False), sim.wait_markers)
        dt_c = timed(make_async(True), sim.wait_markers)
        sim.update_kinematics(0, om, ax)
        # fields leg: the same loop, plus rho + u of the whole lattice to pinned host memory every 10 steps
        rho_host = torch.empty((wl.nz, wl.ny, wl.nx), dtype=torch.float32, pin_memory=True)
        u_host = torch.empty((3, wl.nz, wl.ny, wl.nx), dtype=torch.float32, pin_memory=True)
        fout = {"rho": rho_host.numpy(), "u": u_host.numpy()}
        fstate = {"k": 0}
        step_async = make_async(False)

        def fields_step():
            step_async()
            fstate["k"] += 1
            if fstate["k"] % 10 == 0:
                sim.read_fields(force=False, out=fout)

        n_f = 20
        dt_f = timed(fields_step, sim.wait_markers, n=n_f)
        line["e2e"] = {"value": replicas.whole_job_mlups(wl.cells, e2e_steps, world, dt * 1e3), "unit": UNIT,
                       "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
                       "what": "per step: kinematics table H2D (ibm_update_kinematics, the workload's constant rates: "
                               "the table is unchanged, so the binning prepared ahead stays valid), one coupled step, "
                               "marker forces D2H (pinned) through ibm_read_markers_async (the copy of step n overlaps "
                               "step n+1, the host consumes the forces one step late); the fields stay resident (P:154)",
                       "blocking_read_value": replicas.whole_job_mlups(wl.cells, e2e_steps, world, dt_b * 1e3),
                       "changed_table_value": replicas.whole_job_mlups(wl.cells, e2e_steps, world, dt_c * 1e3),
                       "changed_table_what": "rotation rates perturbed every step: the set binned ahead is discarded, binning runs in line",
                       "with_fields_every_10_steps_value": replicas.whole_job_mlups(wl.cells, n_f, world, dt_f * 1e3),
                       "with_fields_d2h_bytes_per_step": int(d2h + wl.cells * 16 / 10)}
    else:
        rho_host = torch.empty((wl.nz, wl.ny, wl.nx), dtype=torch.float32, pin_memory=True)
        u_host = torch.empty((3, wl.nz, wl.ny, wl.nx), dtype=torch.float32, pin_memory=True)
        u_in = torch.zeros((3, wl.nz, wl.ny, wl.nx), dtype=torch.float32, pin_memory=True)
        out = {"rho": rho_host.numpy(), "u": u_host.numpy()}
        h2d, d2h = wl.cells * 12, wl.cells * 16

        def e2e_step():
            sim.set_fields(None, u_in.numpy())
            sim.step(1, 0)
            sim.read_fields(force=False, out=out)

        dt = timed(e2e_step)
        line["e2e"] = {"value": replicas.whole_job_mlups(wl.cells, e2e_steps, world, dt * 1e3), "unit": UNIT,
                       "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
                       "what": "per step: u field H2D (set_fields), one step, rho+u D2H (pinned)"}
    sim.close()
    del sim

    if rank == 0:
        # ---- configs[1] (W2): the pure-LBM bandwidth case ----------------------------------------------
        if wl.name != "W2" and not args.quick:
            w2 = workloads.get("W2", args.seed)
            s2 = api.from_workload(w2, stream=stream)
            if args.lbm_kernel != "auto":
                s2.set_option(api.OPT_LBM_KERNEL, {"scalar": 1, "vec4": 2}[args.lbm_kernel])
            s2.step(max(3, args.warmup), 0)
            stream.synchronize()
            ms2 = time_steps(torch, s2, stream, args.steps, 0)
            v2 = w2.cells * args.steps / (ms2 * 1e-3) / 1e6
            line["pure_lbm"].update({"W2_mlups": v2, "W2_frac_of_measured": v2 * 1e6 * 152.0 / 1e9 / peak,
                                     "W2_frac_of_nominal_8TBs": v2 * 1e6 * 152.0 / 1e9 / NOMINAL_HBM_GBS})
            s2.close()
            del s2
        # ---- the metric as a curve: coupled MLUPS, fraction of the HBM roofline and IBM share vs marker density ----
        if world == 1 and not args.no_sweep and (not args.quick or args.sweep != ",".join(SWEEP)):
            sweep = []
            n_sw = max(3, min(args.steps, 20))
            for name in [n for n in args.sweep.split(",") if n]:
                if main_entry is not None and name == args.workload:
                    sweep.append(main_entry)
                    continue
                swl = workloads.get(name, args.seed)
                case = gpu_case(torch, api, swl, stream, n_sw, max(3, min(args.warmup, 5)), user_opts)
                msp = pure_ms(torch, case["sim"], stream, n_sw, settle=True)
                case["sim"].close()
                del case["sim"]
                sweep.append(sweep_entry(name, swl, case, msp, peak))
                torch.cuda.empty_cache()
            line["density_sweep"] = sweep
            line["density_sweep_note"] = ("same measurement as `value` (device-resident, CUDA events on the library's stream, %d timed "
                                          "steps) per workload, each leg (coupled, pure) after its warm-up steps plus 50 ms of untimed steps; step_hbm_frac = SURVEY 8(d) algorithmic bytes per step / "
                                          "step time / measured copy peak; W*lit = single-layer (literal) marker sets, P* = the "
                                          "paper-shaped cases of P:231-237" % n_sw)

    # ---- the oracle on the host cores (rank 0, N = 1 only) ------------------------------------------
    if rank == 0 and world == 1 and not args.no_cpu:
        info = host_info()
        ref, swl, what, same = oracle_case(wl.name if wl.name in workloads_names() else args.workload, args.seed)
        mlups_c, _ = time_oracle(ref, swl, args.cpu_steps, 1)
        cb = {"value": mlups_c, "unit": UNIT, "cores": info["nproc"], "kind": "oracle",
              "sample": f"{what}, {args.cpu_steps} steps after 1 warm-up step", "same_config_as_gpu_arm": same, "host": info}
        # pure LBM (mdf_iters = 0) of the same oracle on the same lattice
        p_steps = max(1, min(3, args.cpu_steps))
        t0 = time.perf_counter()
        ref.step(p_steps, 0)
        cb["pure_lbm_value"] = swl.cells * p_steps / (time.perf_counter() - t0) / 1e6
        cb["pure_lbm_sample"] = f"{p_steps} steps with mdf_iters = 0 on the same lattice"
        line["cpu_baseline"] = cb
        ref.close()
    if rank == 0:
        print(json.dumps(line))
    replicas.finish(dist)
    return 0


def workloads_names():
    return ("W1", "W2", "W3", "W3lit", "W3x4", "W4", "W4lit", "W5", "W5lit", "P1", "P6", "P18")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="W4")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--spread", default="gather", choices=["gather", "atomic", "plain"])
    ap.add_argument("--lbm-kernel", default="auto", choices=["auto", "vec4", "scalar"])
    ap.add_argument("--cpu-steps", type=int, default=5)
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--quick", action="store_true", help="skip the extra W2 pure-LBM run and the density sweep")
    ap.add_argument("--no-sweep", action="store_true", help="skip the density sweep")
    ap.add_argument("--sweep", default=",".join(SWEEP), help="workloads of the density sweep (comma separated)")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="set a library option (lbm_set_option), e.g. --opt tile_rows=2 --opt persistent=1")
    ap.add_argument("--compare", action="store_true",
                    help="also time the paper's own kernel designs (box / per-marker U precompute, ib_force1, ib_force2)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else max(args.warmup, 0)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
