#!/usr/bin/env python
"""bench.py -- coupled LBM-IBM MLUPS on one B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload W4] [--impl ours|reference]

A "step" is one pass of the whole hot path: one time step of the coupled scheme (kinematics, marker
sort + chunks + tiles, moments on active cells, mdf_iters x (interpolate, correct, spread), fused
stream-collide-force), replayed as one CUDA graph whose branches overlap the MDF loop, the
stream-collide of the cells outside the marker stencils and the binning of the next step.  The default workload is W4 (BASELINE.json configs[3], 256^3 periodic, 64
three-blade propellers, ~1.18 M markers, 5 MDF iterations): the coupled configuration on the same
256^3 lattice as the pure-LBM bandwidth case configs[1] (W2), which is timed alongside and reported
under "pure_lbm".  All inputs are seeded synthetic (paper_1904_02108_b200/workloads.py).

N > 1: "replicas only": every rank runs the same workload on its own GPU, no data-path
collective; value = units of all ranks / max-over-ranks time.

--impl reference times the fp64 CPU oracle (oracle/) on the host cores on a bounded sample.
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
BYTES_PER_LUP = 152.0          # 19 fp32 loads + 19 fp32 stores per lattice update
G_BYTES_PER_ACTIVE = 12.0      # G read on active cells
NOMINAL_HBM_GBS = 8000.0       # north_star's denominator


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def traffic_from_profile(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the stream-collide kernel from the
    newest committed ncu --set full summary (profiles/traffic_rNN.csv), or None"""
    try:
        pdir = os.path.join(ROOT, "profiles")
        files = sorted(f for f in os.listdir(pdir) if f.startswith("traffic_r") and f.endswith(".csv"))
        for name in reversed(files):
            with open(os.path.join(pdir, name)) as fh:
                for line in fh.read().splitlines()[1:]:
                    w, _, b = line.rsplit(",", 2)[0].split(",", 1)[0], None, line.rsplit(",", 1)[1]
                    if w == workload:
                        return float(b)
    except Exception:
        pass
    return None


class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.QUERY}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
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


def oracle_sample(workload_name, seed, budget_steps):
    """The oracle as it stands on a bounded sample of the same workload (host cores)."""
    import oracle
    from paper_1904_02108_b200 import workloads
    if workload_name in ("W4", "W4lit"):
        wl = workloads.w4(seed, 8 if workload_name == "W4" else 1, n=128)
        sample = f"{workload_name} recipe on a 128^3 box (8 propellers, {wl.n_markers} markers), {budget_steps} steps"
    elif workload_name in ("W5", "W5lit"):
        wl = workloads.w5(seed, 12 if workload_name == "W5" else 1, n=128)
        sample = f"{workload_name} recipe on a 128^3 box ({len(wl.bodies)} propellers, {wl.n_markers} markers), {budget_steps} steps"
    elif workload_name == "W2":
        wl = workloads.w2(seed, n=128)
        sample = f"W2 recipe on a 128^3 channel, {budget_steps} steps"
    else:
        wl = workloads.get(workload_name, seed)
        sample = f"{workload_name} full size, {budget_steps} steps"
    ref = oracle.from_workload(wl)
    return ref, wl, sample


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = os.cpu_count() or 1
    ref, wl, sample = oracle_sample(args.workload, args.seed, args.steps)
    ref.step(args.warmup, wl.mdf_iters)
    t0 = time.perf_counter()
    ref.step(args.steps, wl.mdf_iters)
    dt = time.perf_counter() - t0
    mlups = wl.cells * args.steps / dt / 1e6
    line = {
        "impl": "reference", "metric": METRIC, "value": mlups, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded)",
        "config": {"workload": args.workload, "sample": sample, "mdf_iters": wl.mdf_iters, "markers": wl.n_markers},
        "cpu_baseline": {"value": mlups, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": mlups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


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
    sim.set_option(api.OPT_SPREAD, {"gather": 0, "atomic": 1, "plain": 2}[args.spread])
    sim.set_option(api.OPT_LBM_KERNEL, {"auto": 0, "scalar": 1, "vec4": 2}[args.lbm_kernel])
    for kv in args.opt:
        name, val = kv.split("=")
        sim.set_option(getattr(api, "OPT_" + name.upper()), int(val))

    def barrier():
        torch.cuda.synchronize()
        replicas.barrier(dist)
        torch.cuda.synchronize()

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

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic (seeded)",
        "config": {"workload": wl.name, "lattice": [wl.nx, wl.ny, wl.nz], "tau": wl.tau, "markers": wl.n_markers,
                   "bodies": len(wl.bodies), "mdf_iters": mdf, "spread": args.spread, "lbm_kernel": args.lbm_kernel,
                   "parallelism": "replicas" if world > 1 else "single-gpu",
                   "l2": "inputs larger than L2 (populations %.0f MB per buffer)" % (wl.cells * 76 / 1e6)},
        "clocks": clocks, "gpu_launches": int(launches),
    }

    paper = {"P1": 893.0, "P6": 650.0, "P18": 344.2}.get(wl.name)
    if paper is not None:
        # context, not a baseline: the paper's own MLUPS for the case this synthetic workload is shaped after
        line["config"]["paper_context"] = {"mlups": paper, "hardware": "Tesla P100-PCIE (P:229-237)",
                                           "note": "paper's Blender mesh replaced by a synthetic propeller of the same point count"}
    if rank == 0:
        # ---- the same step as one serial chain with a single fused stream-collide pass (comparison) -----
        if wl.n_markers:
            sim.set_option(api.OPT_OVERLAP, 0)
            sim.step(3, mdf)
            ms_serial = time_steps(torch, sim, stream, args.steps, mdf)
            sim.set_option(api.OPT_OVERLAP, 1)
            line["serial_chain"] = {"value": wl.cells * args.steps / (ms_serial * 1e-3) / 1e6, "unit": UNIT,
                                    "ms_per_step": ms_serial / args.steps,
                                    "what": "LBM_OPT_OVERLAP=0: one stream, one fused stream-collide pass"}
        # ---- the paper's own kernel designs on the same step, one option at a time ---------
        if wl.n_markers and args.compare:
            cmp_steps = max(3, min(args.steps, 20))
            variants = [("moments_box(P:209)", {api.OPT_MOMENTS: api.MOMENTS_BOX}),
                        ("moments_block_per_marker(P:215)", {api.OPT_MOMENTS: api.MOMENTS_PER_MARKER}),
                        ("interp_caller_order(ib_force1)", {api.OPT_INTERP: api.INTERP_CALLER_ORDER}),
                        ("interp_warp_per_marker(shuffle_reduce)", {api.OPT_INTERP: api.INTERP_WARP_PER_MARKER}),
                        ("interp_chunk_window_in_smem", {api.OPT_INTERP: api.INTERP_CHUNK_SMEM}),
                        ("spread_atomic_thread_per_marker", {api.OPT_SPREAD: api.SPREAD_ATOMIC}),
                        ("spread_block125_atomic(ib_force2)", {api.OPT_SPREAD: api.SPREAD_BLOCK125}),
                        ("paper_pipeline(box+ib_force1+ib_force2,serial)",
                         {api.OPT_MOMENTS: api.MOMENTS_BOX, api.OPT_INTERP: api.INTERP_CALLER_ORDER,
                          api.OPT_SPREAD: api.SPREAD_BLOCK125, api.OPT_OVERLAP: 0})]
            defaults = {api.OPT_MOMENTS: 0, api.OPT_INTERP: 0, api.OPT_SPREAD: 0, api.OPT_OVERLAP: 1}
            comp = {"default": ms / args.steps}
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
        ph = sim.phase_ms()
        sim.set_option(api.OPT_TIMING, 0)
        n_active = sim.get_info(api.INFO_ACTIVE_CELLS) if wl.n_markers else 0
        n_words = sim.get_info(api.INFO_ACTIVE_WORDS) if wl.n_markers else 0
        lbm_ms = ph["lbm"] / n_ph
        tot = sum(ph.values()) / n_ph
        peak, how = measured_peak_gbs()
        # the dominant kernel is the stream-collide pass over every 32-cell word without an active cell
        # (k_stream_collide_scalar<LBM_BULK>; with no markers: <LBM_PURE> over all cells): 152 B per cell it updates
        word_cells = min(wl.cells, n_words * 32)
        alg_bytes = BYTES_PER_LUP * (wl.cells - word_cells)
        achieved = alg_bytes / (lbm_ms * 1e-3) / 1e9
        line["roofline"] = {"bound": "hbm", "kernel": "k_stream_collide_scalar<%s> (a8)" % ("LBM_BULK" if wl.n_markers else "LBM_PURE"),
                            "achieved": achieved, "peak": peak,
                            "unit": "GB/s", "frac": achieved / peak, "traffic": traffic_from_profile(wl.name),
                            "peak_source": how, "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                            "algorithmic_bytes_per_launch": alg_bytes, "kernel_ms": lbm_ms,
                            "cells_per_launch": int(wl.cells - word_cells)}
        line["phases_ms_per_step"] = {k: v / n_ph for k, v in ph.items()}
        line["phases_note"] = "phases timed one after the other (LBM_OPT_TIMING); in the timed step they overlap"
        line["active_cells"] = int(n_active)
        line["active_word_cells"] = int(word_cells)
        if wl.n_markers:
            line["chunks"] = sim.get_info(api.INFO_RUNS)
            line["chunk_entries"] = sim.get_info(api.INFO_RUN_ENTRIES)
            line["tiles"] = sim.get_info(api.INFO_TILES)

        # ---- pure LBM on the same lattice and on configs[1] (W2) ---------------------------------
        sim.step(3, 0)
        ms_p = time_steps(torch, sim, stream, args.steps, 0)
        pure_same = wl.cells * args.steps / (ms_p * 1e-3) / 1e6
        line["pure_lbm"] = {"same_lattice_mlups": pure_same,
                            "frac_of_measured": pure_same * 1e6 * BYTES_PER_LUP / 1e9 / peak,
                            "frac_of_nominal_8TBs": pure_same * 1e6 * BYTES_PER_LUP / 1e9 / NOMINAL_HBM_GBS,
                            "coupled_over_pure": value / world / pure_same}
        # share of the coupled step that the IBM adds on top of a pure-LBM step of the same lattice
        line["ibm_share"] = max(0.0, 1.0 - (ms_p / args.steps) / (ms / args.steps))
        if wl.name != "W2" and not args.quick:
            w2 = workloads.get("W2", args.seed)
            s2 = api.from_workload(w2, stream=stream)
            s2.set_option(api.OPT_LBM_KERNEL, {"auto": 0, "scalar": 1, "vec4": 2}[args.lbm_kernel])
            s2.step(max(3, args.warmup), 0)
            stream.synchronize()
            ms2 = time_steps(torch, s2, stream, args.steps, 0)
            v2 = w2.cells * args.steps / (ms2 * 1e-3) / 1e6
            line["pure_lbm"].update({"W2_mlups": v2, "W2_frac_of_measured": v2 * 1e6 * BYTES_PER_LUP / 1e9 / peak,
                                     "W2_frac_of_nominal_8TBs": v2 * 1e6 * BYTES_PER_LUP / 1e9 / NOMINAL_HBM_GBS})
            s2.close()
            del s2

    # ---- end to end through the public API with host buffers (all ranks) ---------------------------
    # every step: H2D = the per-body kinematics table a host controller sets (ibm_update_kinematics),
    # D2H = the marker forces Delta u(k) into pinned host memory (ibm_read_markers); the fields stay
    # resident, as the method intends ("fully performed within the GPU's memory").
    e2e_steps = max(3, min(args.steps, 20))
    if wl.n_markers:
        nb = len(wl.bodies)
        om = np.array([b.omega for b in wl.bodies]); ax = np.stack([b.axis for b in wl.bodies])
        force_host = torch.empty((wl.n_markers, 3), dtype=torch.float32, pin_memory=True)
        out = {"force": force_host.numpy()}
        h2d, d2h = nb * 56, wl.n_markers * 12

        def e2e_step():
            sim.update_kinematics(0, om, ax)
            sim.step(1, mdf)
            sim.read_markers(pos=False, perm=False, cell=False, out=out)
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
    def timed(fn, finish=None):
        fn()
        if finish:
            finish()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            fn()
        if finish:
            finish()
        torch.cuda.synchronize()
        return replicas.max_over_ranks(time.perf_counter() - t0, dist, device="cuda")

    dt = timed(e2e_step)
    e2e_blocking = replicas.whole_job_mlups(wl.cells, e2e_steps, world, dt * 1e3)
    what = ("per step: kinematics table H2D, one coupled step, marker forces D2H (pinned)"
            if wl.n_markers else "per step: u field H2D (set_fields), one step, rho+u D2H (pinned)")
    if wl.n_markers:
        # the same loop with the asynchronous read-out of the public API (ibm_read_markers_async): the D2H copy of
        # step n overlaps step n+1; the host consumes the forces of step n-1 (two pinned buffers) every step
        bufs = [torch.empty((wl.n_markers, 3), dtype=torch.float32, pin_memory=True) for _ in range(2)]
        state = {"k": 0, "sum": 0.0}

        def e2e_step_async():
            sim.update_kinematics(0, om, ax)
            sim.step(1, mdf)                                     # step k is enqueued ...
            sim.wait_markers()                                   # ... while the forces of step k-1 finish landing on the host
            state["sum"] += float(bufs[(state["k"] + 1) & 1][0, 0])   # the host controller reads them
            sim.read_markers_async(bufs[state["k"] & 1])         # read-out of step k, ordered behind it on the device
            state["k"] += 1

        dt = timed(e2e_step_async, sim.wait_markers)
        line["e2e"] = {"value": replicas.whole_job_mlups(wl.cells, e2e_steps, world, dt * 1e3), "unit": UNIT,
                       "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h), "steps": e2e_steps,
                       "what": what + "; read-out through ibm_read_markers_async (copy of step n overlaps step n+1)",
                       "blocking_read_value": e2e_blocking}
    else:
        line["e2e"] = {"value": e2e_blocking, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                       "steps": e2e_steps, "what": what}
    sim.close()

    # ---- the oracle on the host cores (rank 0, N = 1 only) ------------------------------------------
    if rank == 0 and world == 1 and not args.no_cpu:
        ref, swl, sample = oracle_sample(wl.name if wl.name in ("W1", "W2", "W3") else args.workload, args.seed,
                                         args.cpu_steps)
        ref.step(1, swl.mdf_iters)
        t0 = time.perf_counter()
        ref.step(args.cpu_steps, swl.mdf_iters)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": swl.cells * args.cpu_steps / dt / 1e6, "unit": UNIT,
                                "cores": os.cpu_count() or 1, "kind": "oracle", "sample": sample}
    if rank == 0:
        print(json.dumps(line))
    replicas.finish(dist)
    return 0


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
    ap.add_argument("--cpu-steps", type=int, default=10)
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--quick", action="store_true", help="skip the extra W2 pure-LBM run")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="set a library option (lbm_set_option), e.g. --opt tile_rows=2 --opt persistent=2")
    ap.add_argument("--compare", action="store_true",
                    help="also time the paper's own kernel designs (box / per-marker U precompute, ib_force1, ib_force2)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else max(args.warmup, 0)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
