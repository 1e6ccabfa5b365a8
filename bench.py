#!/usr/bin/env python
"""bench.py — particle updates/s of the GRPIC per-particle hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload large|...]

A "step" = one pass of the whole hot path (interp + GR push + BCs + deposit, both species; the counting sort
every `sort_every` steps as config 4 says: grpic_sort_into between two column sets, key of the cell predicted
sort_every/2 steps ahead) over the resident particle set.  N = 1 workload:
BASELINE.json configs[3] "Large" (2048x1024, a = 0.9375, Wald field, ~134M e+- with density ~ r^-2,
FP32, sort every 10 steps) — the >= 100M-particle configuration north_star's target is quoted on.
N > 1: the path does not shard (replicas only) -> every rank runs an independent
replica of the same workload (seed + rank), weak scaling, no data-path collective.

--impl reference times the oracle (oracle/, plain FP64 C, as it stands) on the host cores on a bounded
sample of the same workload; rank 0 only.
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
sys.path.insert(0, ROOT)

METRIC = "particle updates/sec (interp+GR push+deposit)"
UNIT = "updates/s"

# Algorithmic figures per particle update: what the method, as the paper states
# it with n_iter = 10, must compute and move.
FLOPS_PER_UPDATE_NITER10 = 2051.0          # DESIGN.md section 7 table: +,-,*,/,sqrt,exp,sin,cos,floor,min,max,compare each count 1
BYTES_PER_UPDATE = {"f32": 70.0, "f64": 122.0}   # fused step: read i,dx,u,phi,w,tag; write i,dx,u,phi,tag
# FP32 FMA peak from unit counts and clocks (B200_PROFILING.md: 148 SMs, 1965 MHz; 128 FP32 lanes/SM, FMA = 2)
ALU_PEAK_TFLOPS = {"f32": 148 * 128 * 2 * 1.965e9 / 1e12, "f64": 148 * 64 * 2 * 1.965e9 / 1e12}


def _ncu_traffic(prec, workload):
    """DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` capture
    (profiles/ncu_traffic.csv: kernel,precision,workload,particles,dram_read_bytes,dram_write_bytes,source)."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for line in f:
                t = line.strip().split(",")
                if len(t) >= 7 and t[1] == prec and t[2] == workload:
                    return {"bytes": float(t[4]) + float(t[5]), "particles": float(t[3]), "kernel": t[0], "source": t[6]}
    except Exception:
        pass
    return None


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def _workload(name, seed_offset=0, shrink=1):
    from paper_2511_17701_b200 import workloads as W
    if name == "large":
        return W.config_large(shrink=shrink, seed=4 + seed_offset)
    if name == "magnetosphere":
        return W.config_magnetosphere(shrink=shrink, seed=3 + seed_offset)
    if name == "two_species":
        return W.config_two_species(shrink=shrink, seed=5 + seed_offset)
    if name == "tiny":
        return W.config_tiny(shrink=shrink, seed=seed_offset)
    raise SystemExit(f"unknown workload {name}")


def _workload_desc(wl, shrink):
    d = wl.dom
    return (f"config '{wl.name}'" + (f" /{shrink}" if shrink > 1 else "") +
            f": Kerr a={d.a}, grid {d.n1}x{d.n2} log-r {d.r_min:.3f}..{d.r_max:g} r_g, "
            f"{wl.n_particles} particles in {len(wl.species)} species, {wl.dtype}, dt={wl.dt:.4g}, n_iter=10")


# ------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle on the host cores
# ------------------------------------------------------------------------------------------------
def _oracle_setup(name, shrink):
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from helpers import grid_from_domain, oracle_particles
    from oracle import oracle as O
    O.build()
    wl = _workload(name, shrink=shrink)
    rt = np.float32 if wl.dtype == "f32" else np.float64
    g = grid_from_domain(O, wl.dom)
    parts = [oracle_particles(O, sp, rt) for sp in wl.species]
    fields = {k: np.asarray(v, rt).astype(np.float64) for k, v in wl.fields.items()}
    return O, wl, g, parts, fields


def _oracle_step(O, wl, g, parts, fields):
    """one pass of the hot path in the oracle; returns particle updates done"""
    n = 0
    for p in parts:
        n += int(p.tag.sum())
        O.push(g, p, fields, wl.dt)
        O.deposit(g, p, wl.dt)
    return n


def _cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def cpu_baseline(name, shrink=16, steps=1):
    O, wl, g, parts, fields = _oracle_setup(name, shrink)
    t0 = time.perf_counter()
    n = 0
    for _ in range(steps):
        n += _oracle_step(O, wl, g, parts, fields)
    dt = time.perf_counter() - t0
    # one single-thread figure on a smaller sample
    nt = O.num_threads()
    O1, wl1, g1, parts1, fields1 = _oracle_setup(name, shrink * 2)
    O.set_num_threads(1)
    t1 = time.perf_counter()
    n1 = _oracle_step(O1, wl1, g1, parts1, fields1)
    dt1 = time.perf_counter() - t1
    O.set_num_threads(nt)
    return {"value": n / dt, "unit": UNIT, "cores": nt, "kind": "oracle", "cpu_model": _cpu_model(),
            "single_thread_value": n1 / dt1,
            "sample": f"{steps} step(s) of {_workload_desc(wl, shrink)}; oracle = oracle/grpic_oracle.c "
                      f"(FP64, OpenMP over particles), {dt:.1f} s"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    shrink = 4
    O, wl, g, parts, fields = _oracle_setup(args.workload, shrink)
    for _ in range(args.warmup):
        _oracle_step(O, wl, g, parts, fields)
    t0 = time.perf_counter()
    n = 0
    for _ in range(args.steps):
        n += _oracle_step(O, wl, g, parts, fields)
    dt = time.perf_counter() - t0
    val = n / dt
    sample = f"each step = one pass over {_workload_desc(wl, shrink)} (bounded sample of the N=1 workload)"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def reduce_over_ranks(ms, units, world, device="cuda"):
    """Contract of the N > 1 line: time = MAX over ranks (device-timed), units = SUM over ranks (replicas only,
    DESIGN.md section 9: no data-path collective; this all_reduce of two scalars is the only communication)."""
    if world <= 1:
        return float(ms), float(units)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    u = torch.tensor([units], device=device, dtype=torch.float64)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={gpu_index}", f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(", ") for r in open(self.f.name).read().strip().splitlines() if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        for r in rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                    if v.strip().lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2511_17701_b200 import grpic as G

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    wl = _workload(args.workload, seed_offset=rank, shrink=args.shrink)
    prec = wl.dtype if args.precision is None else args.precision
    dom = wl.dom
    names = ("D1", "D2", "D3", "B1", "B2", "B3")
    ctx = G.Context(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, nghost=dom.ng, precision=prec)
    if args.no_tile:
        ctx.set_int("tile_path", 0)
    for kv in args.set:                        # ablation knobs of include/grpic.h, e.g. --set lanes_path=0
        k, v = kv.split("=", 1)
        (ctx.set_real if k in ("sort_lookahead", "small_angle") else ctx.set_int)(k, float(v) if "." in v else int(v))
    fdev = G.grid_tensors(wl.fields, names, prec)
    # the fused step keeps the previous position in registers: no *_prev columns; two column sets per species,
    # swapped by the out-of-place sort (grpic_sort_into), so that a sort moves every byte once
    sets = [G.ParticleSet.from_host(sp, prec).drop_prev() for sp in wl.species]
    spare = [p.empty_like() for p in sets]
    J = {k: torch.zeros(ctx.shape, dtype=G.torch_real(prec), device="cuda") for k in ("J1", "J2", "J3")}
    stream = torch.cuda.current_stream()
    sort_every = wl.sort_every if wl.sort_every > 0 else 10
    # the sort orders by the cell predicted half a sort interval ahead (include/grpic.h "sort_lookahead"): the
    # particles of a warp are then closest together in the middle of the interval, not right after the sort
    ctx.set_real("sort_lookahead", 0.5 * sort_every)
    n_total = sum(p.n for p in sets)

    def one_step(it, evs=None):
        launches = 0
        if it % sort_every == 0:
            for i in range(len(sets)):
                ctx.sort_into(sets[i], spare[i], stream)
                sets[i], spare[i] = spare[i], sets[i]
                launches += 11
        for k in J.values():
            k.zero_()
        for p in sets:
            if evs is not None:
                a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                a.record(stream)
            ctx.step(p, fdev, J, wl.dt, stream)
            launches += 1
            if evs is not None:
                b.record(stream)
                evs.append((a, b))
        return launches

    it = 0
    sampler = ClockSampler(local) if rank == 0 else None      # nvidia-smi needs ~a second to start sampling
    for _ in range(args.warmup):
        one_step(it); it += 1
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    upd0 = ctx.updates_total()
    evs = []
    t_a = torch.cuda.Event(enable_timing=True); t_b = torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t_a.record(stream)
    launches = 0
    for _ in range(args.steps):
        launches += one_step(it, evs); it += 1
    t_b.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if sampler else None
    ms = t_a.elapsed_time(t_b)
    updates = ctx.updates_total() - upd0
    step_kernel_ms = sum(a.elapsed_time(b) for a, b in evs)
    counters = ctx.counters()

    ms_max, updates_all = reduce_over_ranks(ms, updates, world)

    # ---- end to end through the host-buffer ABI call (pinned host memory, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        hwl = wl
        hsets = [G.ParticleSet.from_host(sp, prec, device="cpu", pinned=True) for sp in hwl.species]
        hf = G.grid_tensors(hwl.fields, names, prec, device="cpu", pinned=True)
        hJ = {k: torch.zeros(ctx.shape, dtype=G.torch_real(prec)).pin_memory() for k in ("J1", "J2", "J3")}
        up = down = 0
        for p in hsets:                      # warm-up: allocates the library's device chunks
            ctx.step_host(p, hf, hJ, wl.dt, with_prev=False)
        u0 = ctx.updates_total()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            for p in hsets:
                a, b = ctx.step_host(p, hf, hJ, wl.dt, with_prev=False)
                up += a; down += b
        torch.cuda.synchronize()
        dt_e = time.perf_counter() - t0
        nup = ctx.updates_total() - u0
        dt_e, nup = reduce_over_ranks(dt_e, nup, world)
        e2e = {"value": nup / dt_e, "unit": UNIT, "h2d_bytes_per_step": up // e2e_steps,
               "d2h_bytes_per_step": down // e2e_steps, "steps": e2e_steps,
               "api": "grpic_step_host (C ABI, pinned host buffers, chunked H2D -> fused step -> D2H on three streams; *_prev columns not requested)"}
        del hsets, hf, hJ

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks, peak_src = _peaks()
    value = updates_all / (ms_max * 1e-3)
    n_step_launches = len(evs)
    upd_per_launch = updates / max(1, n_step_launches)
    sec_per_launch = step_kernel_ms * 1e-3 / max(1, n_step_launches)
    flops = FLOPS_PER_UPDATE_NITER10 * upd_per_launch
    ach_tflops = flops / sec_per_launch / 1e12
    alu_peak = ALU_PEAK_TFLOPS[prec]
    hbm_ach = BYTES_PER_UPDATE[prec] * upd_per_launch / sec_per_launch / 1e9
    kernel = "k_step_tiled" if not args.no_tile else "k_push_or_step<.,true>"
    tr = _ncu_traffic(prec, args.workload) if (not args.no_tile and args.shrink == 1) else None
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": prec, "data": "synthetic",
        "config": {"workload": _workload_desc(wl, args.shrink), "sort_every": sort_every,
                   "sort": "grpic_sort_into between two column sets per species; no *_prev columns (fused step); "
                           "sort_lookahead = sort_every/2",
                   "l2": "inputs (particle columns, several GB) larger than the 126 MB L2; no flush needed",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "paper_context": "paper: ~1.2-1.4e8 updates/s on 1x A100 (P:550), other hardware, not a target"},
        "roofline": {"bound": "alu", "kernel": kernel, "achieved": ach_tflops, "peak": alu_peak, "unit": "TFLOP/s",
                     "frac": ach_tflops / alu_peak, "traffic": (tr["bytes"] if tr else None),
                     "traffic_note": (f"dram read+write bytes of one {tr['kernel']} launch over {tr['particles']:.0f} particles, "
                                      f"{tr['source']}" if tr else None),
                     "peak_source": f"derived: 148 SMs x {128 if prec == 'f32' else 64} lanes x 2 (FMA) x 1.965 GHz",
                     "flops_per_update": FLOPS_PER_UPDATE_NITER10,
                     "updates_per_launch": upd_per_launch, "ms_per_launch": sec_per_launch * 1e3,
                     "kernel_share_of_step": step_kernel_ms / ms,
                     "hbm": {"achieved": hbm_ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                             "frac": hbm_ach / peaks["hbm_gbs"], "bytes_per_update": BYTES_PER_UPDATE[prec],
                             "peak_source": peak_src}},
        "without_sort": {"value": updates / (step_kernel_ms * 1e-3), "unit": UNIT,
                         "note": "fused step launches only (CUDA events around each launch); `value` includes grpic_sort_into every sort_every steps and the J zero-fills"},
        "clocks": clocks, "gpu_launches": launches,
        "counters_last_step": counters, "updates_timed": updates_all,
    }
    if e2e is not None:
        out["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, shrink=4, steps=16)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="large")
    ap.add_argument("--shrink", type=int, default=1, help="divide both grid edges (debugging only)")
    ap.add_argument("--precision", default=None, choices=[None, "f32", "f64"])
    ap.add_argument("--no-tile", action="store_true", help="force the direct kernel")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--set", action="append", default=[], metavar="KEY=VALUE",
                    help="grpic_set_int / grpic_set_real knob for ablation runs (repeatable)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
