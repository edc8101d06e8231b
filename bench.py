#!/usr/bin/env python
"""bench.py -- cell-updates/s of the hot path (BASELINE.json `metric`) on BASELINE config 3.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--precision 64|32]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one full SSP-RK3 step (three stage evaluations of con2prim + wavespeed max, the three WENO7-LF
sweeps, the jet source and the stage combination) of the synthetic 256^3 ellipsoidal-flow + 1 jet grid
(config 3: PAPER.md:49 for grid/dx/dt, :37 for the IC family; numbers from BASELINE.json, DESIGN.md "Input
recipe").  The path is one-GPU (north_star); with N > 1 every rank advances its own replica of the grid
("replicas only") and the value is the aggregate.

One JSON line on stdout (rank 0).  Keys: the contract of the task statement + `roofline` (dominant kernel
class = the three sweep kernels, bound "alu": FP64 pipe) + `cpu_baseline` (the oracle, timed on the host cores
on a bounded slab of the same workload).

`--impl reference`: the oracle (oracle/hydro_oracle.cpp) as it stands on the host cores, each step one RK3
step of a 256 x 256 x NZ slab of the same initial condition (NZ chosen so the run stays within minutes).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1511_02137_b200 import synthetic as S  # noqa: E402

METRIC = "cell-updates/s (full RK3 steps x cells / s)"
UNIT = "cell-updates/s"
# Algorithmic flops per cell per stage evaluation, nf = 4 / 5: measured by running the oracle's per-cell routines
# on an operation-counting number type (oracle_count_flops): FMA = 2, + - * / sqrt = 1.
# Of these the sweep kernels carry interface_flux + divergence (+ the stage combination in the last sweep).
FLOPS_STAGE = {4: 3764.0, 5: 4691.0}
FLOPS_SWEEPS_STAGE = {4: 3 * (1208.0 + 12.0) + 20.0, 5: 3 * (1510.0 + 15.0) + 25.0}
# the WENO5 variant (--weno-order 5), same counting (oracle_count_flops_order)
FLOPS_STAGE_W5 = {4: 1820.0, 5: 2261.0}
FLOPS_SWEEPS_STAGE_W5 = {4: 3 * (560.0 + 12.0) + 20.0, 5: 3 * (700.0 + 15.0) + 25.0}
FP64_NOMINAL_TF = 148 * 64 * 2 * 1.965e9 / 1e12          # 148 SMs x 64 DFMA/clk x 2 x 1.965 GHz = 37.2
# Counters that only ncu can give (DRAM bytes, FP64 warp instructions, pipe utilisation, registers, occupancy) are READ from
# the committed summary of the `ncu --set full` captures, never typed in here; every row carries the sha of the CUDA
# sources it was taken at (paper_1511_02137_b200.build.source_sha) and the bench line says when that differs from HEAD.
NCU_TABLE = os.path.join(ROOT, "profiles", "r2_ncu_kernels.csv")


def variant_key(cfg, precision, order, nf, limiter):
    return "cfg%d_f%d_w%d_nf%d_lim%d" % (cfg, precision, order, nf, 1 if limiter else 0)


def ncu_rows(variant):
    """{kernel class: [row dicts]} of the committed ncu summary for this variant ({} if none).  A class has several rows
    when its passes were captured in several instantiations (x: COMBINE1 of stage 1 and COMBINE of stages 2, 3; 5-field
    states: the 4-field and the 1-field kernel of every pass)."""
    import csv
    out = {}
    if os.path.exists(NCU_TABLE):
        with open(NCU_TABLE) as f:
            for row in csv.DictReader(l for l in f if not l.startswith("#")):
                if row["variant"] == variant:
                    out.setdefault(row["kernel"], []).append(row)
    return out


def ncu_pass_mean(rows, key):
    """Mean over the nine directional passes of a step of an ncu counter: per direction, the kernels of one pass add up
    (nf4 + nf1 instantiations), and the x direction is COMBINE1 once and COMBINE twice per step."""
    tot, n = 0.0, 0
    for cls in ("sweep_x", "sweep_y", "sweep_z"):
        by_out = {}
        for r in rows.get(cls, []):
            by_out.setdefault(r["template"].split(";")[3], []).append(float(r[key]))
        if not by_out:
            return None
        if cls == "sweep_x" and "COMBINE1" in by_out and "COMBINE" in by_out:
            tot += sum(by_out["COMBINE1"]) + 2.0 * sum(by_out["COMBINE"])
        else:
            tot += 3.0 * sum(next(iter(by_out.values())))
        n += 3
    return tot / n


def max_over_ranks(values, world, device):
    """MAX over ranks of a list of floats (times): the contract's max-over-ranks timing.  world == 1: identity."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def job_value(world, cells, steps, seconds):
    """Whole-job cell-updates/s of `world` independent replicas ("replicas only")."""
    return world * cells * steps / seconds


class ClockSampler:
    """nvidia-smi clocks / throttle reasons of one GPU while the timed region runs (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.t = threading.Thread(target=self._read, daemon=True)
        self.t.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        inside = [r for (t, r) in self.rows if t0 <= t <= t1] or [r for (_, r) in self.rows[-3:]]
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in inside:
            c = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except (ValueError, IndexError):
                continue
            for k, nm in enumerate(names):
                if len(c) > 3 + k and c[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_slab_run(cfg, nzs, steps, warmup=0, order=7, sigma=0.0, limiter=False):
    """Oracle on the central nzs planes of config `cfg`'s initial condition; returns (cells, seconds, threads)."""
    from oracle import oracle as O
    c = S.CONFIGS[cfg]
    nx, ny, nz = c["n"]
    k0 = nz // 2 - nzs // 2
    U0 = S.make_state(cfg, z_range=(k0, k0 + nzs))
    o = O.Oracle(nx, ny, nzs, c["dx"], c["dt"], nfields=c["nf"], weno_order=order)
    o.set_state(U0)
    for pos, d in c["jets"]:
        o.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)
    o.set_deposit_width(sigma)
    o.set_limiter(limiter)
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    assert o.diag()["has_nan"] == 0
    o.close()
    return nx * ny * nzs, dt, O.num_threads()


def run_reference(args, rank):
    if rank != 0:
        return
    cfg = args.config
    c = S.CONFIGS[cfg]
    # size the slab so that (K + W) steps take about two minutes: calibrate on one step of 8 planes
    cells8, t8, threads = oracle_slab_run(cfg, 8, 1, order=args.weno_order, sigma=args.deposit_sigma, limiter=args.limiter)
    budget = 120.0
    nzs = int(min(c["n"][2], max(8, 8 * int(budget / (t8 * (args.steps + args.warmup)) + 1e-9))))
    cells, secs, threads = oracle_slab_run(cfg, nzs, args.steps, args.warmup, order=args.weno_order, sigma=args.deposit_sigma, limiter=args.limiter)
    value = cells * args.steps / secs
    sample = "%dx%dx%d central slab of config %d's IC + jet, %d RK3 steps" % (c["n"][0], c["n"][1], nzs, cfg,
                                                                              args.steps)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(args, cfg),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }), flush=True)


def workload_config(args, cfg):
    c = S.CONFIGS[cfg]
    return {"workload": "BASELINE config %d: %dx%dx%d, dx=%g fm, dt=%g fm/c, nf=%d, p=e/3, ellipsoidal flow + %d jet(s), "
                        "outflow ghosts" % (cfg, c["n"][0], c["n"][1], c["n"][2], c["dx"], c["dt"], c["nf"],
                                            len(c["jets"])),
            "cells": int(np.prod(c["n"])), "config_steps": c["steps"], "weno_order": getattr(args, "weno_order", 7), "deposit_sigma_fm": getattr(args, "deposit_sigma", 0.0), "limiter": bool(getattr(args, "limiter", False)),
            "parallelism": "replicas x%d" % args.gpus,
            "l2": "state (%.0f MiB per copy) exceeds L2; no flush needed" %
                  (np.prod(c["n"]) * c["nf"] * (args.precision // 8) / 2 ** 20)}


def run_decomposed(args, rank, world, local, barrier):
    """--decompose: ONE grid of config `args.config` split into `world` z-slabs (paper_1511_02137_b200/slab.py); every
    rank advances its slab, exchanging the Lax-Friedrichs speeds and 4 halo planes per face once per stage.  Strong
    scaling: value = cells x steps / max-over-ranks time.  Device-timed on the handle's stream (everything between the
    two events is host-synchronised per stage)."""
    import torch
    import torch.distributed as dist
    from paper_1511_02137_b200 import hydro as H, slab as SL
    cfg = args.config
    c = S.CONFIGS[cfg]
    cells = int(np.prod(c["n"]))
    U0 = S.make_state(cfg).astype(np.float64 if args.precision == 64 else np.float32)
    stream = torch.cuda.Stream()
    sl = SL.Slab(H, c["n"], c["dx"], c["dt"], rank, world, nfields=c["nf"], precision=args.precision, stream=stream,
                 weno_order=args.weno_order)
    for pos, d in c["jets"]:
        sl.g.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)
    sl.set_deposit_width(args.deposit_sigma)
    sl.set_limiter(args.limiter)
    d_ = dist if world > 1 else None
    sl.set_state(U0)
    SL.run_distributed(sl, args.warmup, d_)
    sl.set_state(U0)
    sl.g.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = sl.g.launch_count()
    barrier()
    e0.record(stream)
    SL.run_distributed(sl, args.steps, d_)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    ms_max = max_over_ranks([ms], world, "cuda")[0]
    dg = sl.g.diag()
    if dg["has_nan"]:
        raise SystemExit("bench.py: non-finite state after the timed run")
    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": cells * args.steps / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64" if args.precision == 64 else "f32",
            "data": "synthetic", "config": dict(workload_config(args, cfg), parallelism="z-slabs x%d" % world),
            "gpu_launches": int(sl.g.launch_count() - n0),
            "halo_bytes_per_stage_per_face": int(sl.g.halo_reals() * (args.precision // 8)),
        }), flush=True)
    sl.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=120)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32])
    ap.add_argument("--weno-order", type=int, default=7, choices=[7, 5])
    ap.add_argument("--deposit-sigma", type=float, default=0.0, help="Gaussian deposit width [fm] (R15); 0 = one cell")
    ap.add_argument("--decompose", action="store_true",
                    help="with --gpus N > 1: split ONE grid into N z-slabs (strong scaling, halo exchange + MAX all-reduce "
                         "over NCCL; DESIGN.md 9) instead of N independent replicas")
    ap.add_argument("--limiter", action="store_true", help="positivity-preserving flux limiter (R16, f-1); fp64 only")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_1511_02137_b200 import hydro as H

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    H.load()
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if args.decompose:
        run_decomposed(args, rank, world, local, barrier)
        if world > 1:
            dist.destroy_process_group()
        return

    cfg = args.config
    c = S.CONFIGS[cfg]
    cells = int(np.prod(c["n"]))
    tdt = torch.float64 if args.precision == 64 else torch.float32
    U0 = S.make_state(cfg)
    U0h = torch.from_numpy(U0).to(tdt).pin_memory()
    outh = torch.empty_like(U0h).pin_memory()
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        U0d = U0h.cuda(non_blocking=True)
    stream.synchronize()
    g = H.Hydro(*c["n"], c["dx"], c["dt"], nfields=c["nf"], precision=args.precision, stream=stream,
                weno_order=args.weno_order)
    for pos, d in c["jets"]:
        g.add_jet(pos, d, S.KAPPA_RAD, S.KAPPA_COLL, S.CR_OVER_CF)

    g.set_deposit_width(args.deposit_sigma)
    g.set_limiter(args.limiter)

    # ---- measured ALU peak of this GPU, same run
    peak_tf = H.measure_alu_peak(args.precision, 200.0, stream.cuda_stream)

    # ---- warm-up, then the device-resident timed region: K steps from the initial state, as a user runs them (hydro_step
    # replays one captured RK3 step as a CUDA graph; profiling off)
    g.set_state(U0d)
    g.step(args.warmup)
    g.set_state(U0d)
    g.synchronize()
    sampler = ClockSampler(local if "CUDA_VISIBLE_DEVICES" not in os.environ else
                           os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local])
    sampler.start()
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    n0 = g.launch_count()
    barrier()
    w0 = time.perf_counter()
    with torch.cuda.stream(stream):
        e0.record(stream)
        g.step(args.steps)
        e1.record(stream)
    barrier()
    w1 = time.perf_counter()
    ms = e0.elapsed_time(e1)
    launches = g.launch_count() - n0
    clocks = sampler.stop(w0, w1)
    dg = g.diag()
    if dg["has_nan"]:
        raise SystemExit("bench.py: non-finite state after the timed run")
    # ---- the same K steps again with one CUDA event after every launch (hydro_set_profiling): per-kernel-class device
    # times for the roofline of the dominant kernel; individual launches, so this pass is not the reported value
    g.set_state(U0d)
    g.synchronize()
    g.set_profiling(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        p0.record(stream)
        g.step(args.steps)
        p1.record(stream)
    kt = g.kernel_times()
    g.set_profiling(False)
    ms_profiled = p0.elapsed_time(p1)

    # ---- end to end through the C ABI with HOST buffers: upload, K steps, download, all inside the timed region
    e2e = None
    if not args.no_e2e:
        barrier()
        t0 = time.perf_counter()
        g.set_state(U0h)
        g.step(args.steps)
        g.get_fields(out=outh)
        torch.cuda.synchronize()
        t_e2e = time.perf_counter() - t0
        nbytes = U0h.numel() * U0h.element_size()
        e2e = (t_e2e, nbytes)

    ms_max, e2e_max = max_over_ranks([ms, e2e[0] if e2e else 0.0], world, "cuda")

    if rank == 0:
        value = job_value(world, cells, args.steps, ms_max * 1e-3)
        nf = c["nf"]
        sweeps = [kt[k] for k in ("sweep_x", "sweep_y", "sweep_z")]
        sw_ms = sum(k["ms"] for k in sweeps)
        sw_n = sum(k["launches"] for k in sweeps)
        all_ms = sum(k["ms"] for k in kt.values())
        # dominant kernel class: the WENO7-LF sweep kernels; flops per launch = (sweep flops per cell per stage / 3) * cells
        fl_sweeps = (FLOPS_SWEEPS_STAGE if args.weno_order == 7 else FLOPS_SWEEPS_STAGE_W5)[nf]
        fl_stage = (FLOPS_STAGE if args.weno_order == 7 else FLOPS_STAGE_W5)[nf]
        # one "launch" of the dominant kernel class = one directional pass over the grid (9 per RK3 step).  A 5-field fp64
        # state is swept by two kernels per pass (fields 0..3 + the baryon density): their times add up.
        passes = 9.0 * args.steps
        fl_launch = fl_sweeps / 3.0 * cells
        achieved = fl_launch / (sw_ms / passes * 1e-3) / 1e12 if sw_n else 0.0
        nominal = FP64_NOMINAL_TF * (1 if args.precision == 64 else 2)
        esz = args.precision // 8
        sweeps_per_step = 9.0
        rows = ncu_rows(variant_key(cfg, args.precision, args.weno_order, nf, args.limiter))
        from paper_1511_02137_b200 import build as B
        sha = B.source_sha()
        srows = [r for k in ("sweep_x", "sweep_y", "sweep_z") for r in rows.get(k, [])]
        traffic = inst64 = pipe = inst_all = None
        if srows and ncu_pass_mean(rows, "dram_read_B") is not None:
            traffic = ncu_pass_mean(rows, "dram_read_B") + ncu_pass_mean(rows, "dram_write_B")
            inst64 = ncu_pass_mean(rows, "inst_fp64")
            inst_all = ncu_pass_mean(rows, "inst_total")
            pipe = sum(float(r["pipe_fp64_pct"]) * float(r["duration_us"]) for r in srows) / \
                sum(float(r["duration_us"]) for r in srows) / 100.0
        avg_s = sw_ms / passes * 1e-3 if sw_n else None
        kernels_per_pass = sw_n / passes if sw_n else 1.0
        roof = {"bound": "alu", "kernel": "k_sweep_ring<x|y|z> (WENO%d-LF flux + divergence + RK3 combine)" % args.weno_order,
                "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s", "frac": achieved / peak_tf,
                "peak_kind": "measured in this run: register-resident %s chain on all SMs (hydro_measure_alu_peak)" %
                             ("DFMA" if args.precision == 64 else "FFMA"),
                "peak_nominal": nominal, "frac_of_nominal": achieved / nominal,
                "flops_per_launch": fl_launch, "avg_launch_ms": sw_ms / passes if sw_n else None,
                "kernels_per_launch": kernels_per_pass,
                "share_of_step": sw_ms / all_ms if all_ms else None,
                "kernel_ms_per_step": {k: v["ms"] / args.steps for k, v in kt.items()},
                "ms_per_step_profiled_pass": ms_profiled / args.steps,
                "whole_path_frac": (fl_stage * 3 * value) / (peak_tf * 1e12),
                # instruction-level fraction: FP64 warp instructions (ncu) x 32 lanes x 2 flops, as if every one were an
                # FMA, over the live launch time and the measured FMA peak: cannot exceed 1, unlike the textbook `frac`
                "inst_frac": (inst64 * 64.0 / avg_s / 1e12 / peak_tf) if (inst64 and avg_s and args.precision == 64) else None,
                "fp64_warp_inst_per_launch_ncu": inst64,
                "fp64_pipe_busy_ncu": pipe if args.precision == 64 else None,
                # the FP64 pipe takes a warp instruction every second issue cycle and nothing else issues in between
                # (DESIGN.md 7): with F FP64 and O other warp-instructions a pass needs 2F + O issue cycles per scheduler,
                # so the pipe cannot be busier than 2F / (2F + O); measured utilisation is 0.96-0.97 of this
                "issue_ceiling_ncu": (2.0 * inst64 / (inst64 + inst_all)) if (inst64 and inst_all and args.precision == 64) else None,
                "traffic": traffic,
                "traffic_source": "profiles/r2_ncu_kernels.csv (ncu --set full: dram__bytes_read.sum + dram__bytes_write.sum per "
                                  "directional pass, mean over the nine passes of a step)" if srows else None,
                "profile_csrc_sha": srows[0]["csrc_sha"] if srows else None, "csrc_sha": sha,
                "profile_stale": (srows[0]["csrc_sha"] != sha) if srows else None,
                # unique bytes of a fully fused stage, (2 + 3 + 3) x nf x sizeof(real) per cell-update, spread
                # over the step's sweep launches; traffic / this = how far the three-pass design is from that floor
                "algorithmic_bytes_per_launch": 8.0 * nf * esz * cells / sweeps_per_step,
                # what THIS design's sweep kernels must move per launch (U, W, P read; nf written or reduce-added; U^n
                # read by the COMBINE kernels of stages 2 and 3), mean over the step's launches
                "kernel_bytes_per_launch": (nf + 2 + nf + nf * 2.0 / 9.0 + 2.0 / 3.0 * nf) * esz * cells}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64" if args.precision == 64 else "f32",
            "data": "synthetic", "config": workload_config(args, cfg), "clocks": clocks,
            "gpu_launches": int(launches), "roofline": roof,
            "diag": {"limited_faces": g.limited_faces(), "ncap": dg["ncap"], "alpha": dg["alpha"].tolist(), "deposited_E_GeV": float(dg["deposited"][0])},
        }
        if e2e:
            line["e2e"] = {"value": job_value(world, cells, args.steps, e2e_max), "unit": UNIT,
                           "h2d_bytes_per_step": e2e[1] / args.steps, "d2h_bytes_per_step": e2e[1] / args.steps,
                           "what": "hydro_set_state(host) + hydro_step(K) + hydro_get_fields(host), pinned buffers; "
                                   "bytes are the one upload / one download spread over K steps"}
        if not args.no_cpu_baseline and world == 1:
            # bounded sample of the same workload: ~10-20 s of CPU work on the box's cores
            nzs, bsteps = min(64, c["n"][2]), 12
            cells_s, secs, threads = oracle_slab_run(cfg, nzs, bsteps, order=args.weno_order, sigma=args.deposit_sigma,
                                                     limiter=args.limiter)
            line["cpu_baseline"] = {"value": cells_s * bsteps / secs, "unit": UNIT, "cores": threads, "kind": "oracle",
                                    "sample": "%dx%dx%d central slab of config %d's IC + jet, %d RK3 steps (%.1f s)" %
                                              (c["n"][0], c["n"][1], nzs, cfg, bsteps, secs)}
        print(json.dumps(line), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
