#!/usr/bin/env python
"""bench.py — particle updates/s of the GRPIC per-particle hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload large|...] [--peaks]

A "step" = one pass of the whole hot path (interp + GR push + BCs + deposit, both species; the counting sort
every `sort_every` steps as config 4 says: grpic_sort_into between two column sets, key of the cell predicted
sort_every/2 steps ahead) over the resident particle set.  N = 1 workload:
BASELINE.json configs[3] "Large" (2048x1024, a = 0.9375, Wald field, ~134M e+- with density ~ r^-2,
FP32, sort every 10 steps) — the >= 100M-particle configuration north_star's target is quoted on.
N > 1: the path does not shard (replicas only) -> every rank runs an independent
replica of the same workload (seed + rank), weak scaling, no data-path collective.

The line carries, besides the contract's keys: `roofline` (ALU-bound: algorithmic and executed fractions of the FMA
peak MEASURED in this run by register-only FFMA/DFMA chains, and the HBM fraction), `other_workloads` (configs 3 and 5,
the latter in FP64), `cpu_baseline` (the oracle on one FULL step of the workload on the host cores) and `e2e`.

--impl reference times the oracle (oracle/, plain FP64 C, as it stands) on the host cores on a bounded
sample of the same workload; rank 0 only.   --peaks prints the measured throughput denominators and exits.
"""
from __future__ import annotations

import argparse
import csv
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

# Algorithmic figures per particle update: what the method, as the paper states it with
# n_iter = 10, must compute and move.  2051 = hand table with common sub-expressions shared and unused metric entries
# dropped; the oracle AS WRITTEN executes ~3160 (counted by code: oracle.count_ops, reported in cpu_baseline).
FLOPS_PER_UPDATE_NITER10 = 2051.0
BYTES_PER_UPDATE = {"f32": 70.0, "f64": 122.0}   # fused step: read i,dx,u,phi,w,tag; write i,dx,u,phi,tag
# FMA peak from unit counts and clocks (B200_PROFILING.md: 148 SMs, 1965 MHz; 128 FP32 / 64 FP64 lanes per SM, FMA = 2):
# kept beside the measured figure for comparison
ALU_PEAK_DERIVED = {"f32": 148 * 128 * 2 * 1.965e9 / 1e12, "f64": 148 * 64 * 2 * 1.965e9 / 1e12}
KERNELS_PER_STEP_CALL = 3       # k_step_tiled (sparse items) + k_step_lanes (dense items) + k_push_or_step_from (tail)
KERNELS_PER_SORT = 11           # hist, 3 x scan, items_count, 3 x scan, items_fill, rank, gather


def _profile_numbers(prec, workload):
    """Per-launch numbers of the dominant kernel from the committed `ncu --set full` extract of this workload
    (profiles/r2_top_kernel_<prec>_<workload>.csv, written from `ncu --page raw --csv` by the command named in the .md
    beside it): DRAM bytes and executed FP instructions."""
    path = os.path.join(ROOT, "profiles", f"r2_top_kernel_{prec}_{workload}.csv")
    try:
        rows = {r[0]: r[1] for r in csv.reader(open(path)) if len(r) >= 2 and not r[0].startswith("#")}
        f = lambda k: float(rows[k])
        return {"kernel": rows["kernel"], "particles": f("particles_per_launch"),
                "dram_bytes": f("dram__bytes_read.sum") + f("dram__bytes_write.sum"),
                "flop_executed": f("flop_executed_per_launch"), "inst_per_particle": f("warp_inst_per_32_particles"),
                "source": os.path.relpath(path, ROOT)}
    except Exception:
        return None


def _peaks_file():
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
    if name in ("geodesic", "geodesic_f64"):          # config 2: zero-field geodesic stress, q = 0 (no sort, no deposit)
        return W.config_geodesic(n=(1 << 24) // (shrink * shrink), dtype="f64" if name.endswith("f64") else "f32",
                                 seed=2 + seed_offset)
    raise SystemExit(f"unknown workload {name}")


def _workload_desc(wl, shrink):
    d = wl.dom
    return (f"config '{wl.name}'" + (f" /{shrink}" if shrink > 1 else "") +
            f": Kerr a={d.a}, grid {d.n1}x{d.n2} log-r {d.r_min:.3f}..{d.r_max:g} r_g, "
            f"{wl.n_particles} particles in {len(wl.species)} species, {wl.dtype}, dt={wl.dt:.4g}, n_iter=10")


# ------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle on the host cores (the only places bench.py touches oracle/)
# ------------------------------------------------------------------------------------------------
def _oracle_setup(wl):
    from oracle import oracle as O
    from oracle.parity import grid_from_domain, oracle_particles
    O.build()
    rt = np.float32 if wl.dtype == "f32" else np.float64
    g = grid_from_domain(O, wl.dom)
    parts = [oracle_particles(O, sp, rt) for sp in wl.species]
    fields = {k: np.asarray(v, rt).astype(np.float64) for k, v in wl.fields.items()}
    return O, g, parts, fields


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


def cpu_baseline(name, wl_full=None):
    """The oracle as it stands on ONE FULL step of the workload, all host cores; one single-thread figure on
    a /8 sample; and the operation count of the method by code (oracle.count_ops on a small sample)."""
    wl = wl_full if wl_full is not None else _workload(name)
    O, g, parts, fields = _oracle_setup(wl)
    t0 = time.perf_counter()
    n = _oracle_step(O, wl, g, parts, fields)
    dt = time.perf_counter() - t0
    del parts
    nt = O.num_threads()
    wl1 = _workload(name, shrink=8)
    O1, g1, parts1, fields1 = _oracle_setup(wl1)
    cnt = O.count_ops(g1, parts1[0], fields1, wl1.dt)
    O.set_num_threads(1)
    t1 = time.perf_counter()
    n1 = _oracle_step(O1, wl1, g1, parts1, fields1)
    dt1 = time.perf_counter() - t1
    O.set_num_threads(nt)
    return {"value": n / dt, "unit": UNIT, "cores": nt, "kind": "oracle", "cpu_model": _cpu_model(),
            "single_thread_value": n1 / dt1,
            "ops_per_update_counted": cnt["total_per_update"],
            "ops_per_update_by_stage": {k: round(v, 1) for k, v in cnt["per_stage"].items() if v > 0},
            "sample": f"1 full step of {_workload_desc(wl, 1)}; oracle = oracle/grpic_oracle.c "
                      f"(FP64, OpenMP over particles), {dt:.1f} s; single thread: 1 step of the /8 grid; operation count: "
                      f"the same source on a counting type, {cnt['particles']} particles"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    shrink = 4
    wl = _workload(args.workload, shrink=shrink)
    O, g, parts, fields = _oracle_setup(wl)
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


def measure_peaks(ctx, kinds=("ffma", "dfma", "mufu", "smem_rmw"), reps=5):
    """Throughput of the register-only probes of the library (include/grpic.h grpic_probe), CUDA events around each
    launch, best of `reps` after a warm-up: {"ffma": TFLOP/s, "dfma": TFLOP/s, "mufu": Tera thread-op/s, ...}."""
    import torch
    stream = torch.cuda.current_stream()
    out = {}
    for kind in kinds:
        iters = {"ffma": 4096, "dfma": 2048, "mufu": 1024, "smem_rmw": 512}[kind]
        best = None
        for r in range(reps + 1):
            a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ops = ctx.probe(kind, iters, stream)
            b.record(stream)
            torch.cuda.synchronize()
            ms = a.elapsed_time(b)
            if r > 0:
                best = ms if best is None else min(best, ms)
        out[kind] = ops / (best * 1e-3) / 1e12
    return out


def run_peaks(args):
    import torch
    from paper_2511_17701_b200 import grpic as G
    assert torch.cuda.is_available(), "bench.py needs a CUDA device"
    sampler = ClockSampler(0)
    ctx = G.Context(64, 64, 0.5, 1.5, 10.0, precision="f32")
    time.sleep(0.5)
    pk = measure_peaks(ctx, reps=8)
    clocks = sampler.stop()
    print(json.dumps({"peaks": {"fp32_fma_tflops": pk["ffma"], "fp64_fma_tflops": pk["dfma"],
                                "mufu_rsqrt_tera_ops": pk["mufu"], "shared_rmw_tera_ops": pk["smem_rmw"]},
                      "derived": {"fp32_fma_tflops": ALU_PEAK_DERIVED["f32"], "fp64_fma_tflops": ALU_PEAK_DERIVED["f64"],
                                  "how": "148 SMs x 128 (FP32) / 64 (FP64) lanes x 2 x 1.965 GHz"},
                      "how": "grpic_probe: 1184 x 256 threads, 8 independent chains per thread, CUDA events, best of 8",
                      "clocks": clocks}))


class DeviceRun:
    """The resident workload and its step loop: what `value` times."""

    def __init__(self, G, wl, prec, knobs=(), no_tile=False):
        import torch
        self.torch, self.G, self.wl, self.prec = torch, G, wl, prec
        dom = wl.dom
        names = ("D1", "D2", "D3", "B1", "B2", "B3")
        self.ctx = ctx = G.Context(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, nghost=dom.ng, precision=prec)
        if no_tile:
            ctx.set_int("tile_path", 0)
        for kv in knobs:                       # ablation knobs of include/grpic.h, e.g. --set lanes_path=0
            k, v = kv.split("=", 1)
            (ctx.set_real if k in ("sort_lookahead", "small_angle") else ctx.set_int)(k, float(v) if "." in v else int(v))
        self.fdev = G.grid_tensors(wl.fields, names, prec)
        # the fused step keeps the previous position in registers: no *_prev columns; two column sets per species,
        # swapped by the out-of-place sort (grpic_sort_into), so that a sort moves every byte once
        self.sets = [G.ParticleSet.from_host(sp, prec).drop_prev() for sp in wl.species]
        self.spare = [p.empty_like() for p in self.sets]
        self.J = {k: torch.zeros(ctx.shape, dtype=G.torch_real(prec), device="cuda") for k in ("J1", "J2", "J3")}
        self.stream = torch.cuda.current_stream()
        self.sort_every = wl.sort_every if wl.sort_every > 0 else 10
        self.sorted = any(sp.q_over_m != 0.0 for sp in wl.species)     # q = 0 (config 2): direct kernel, nothing to sort for
        # the sort orders by the cell predicted half a sort interval ahead (include/grpic.h "sort_lookahead")
        if not any(kv.startswith("sort_lookahead=") for kv in knobs):
            ctx.set_real("sort_lookahead", 0.5 * self.sort_every)
        self.it = 0

    def one_step(self, evs=None, sevs=None):
        torch = self.torch
        launches = 0
        if self.sorted and self.it % self.sort_every == 0:
            for i in range(len(self.sets)):
                if sevs is not None:
                    a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                    a.record(self.stream)
                self.ctx.sort_into(self.sets[i], self.spare[i], self.stream)
                self.sets[i], self.spare[i] = self.spare[i], self.sets[i]
                launches += KERNELS_PER_SORT
                if sevs is not None:
                    b.record(self.stream); sevs.append((a, b))
        for k in self.J.values():
            k.zero_()
        for p in self.sets:
            if evs is not None:
                a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
                a.record(self.stream)
            self.ctx.step(p, self.fdev, self.J, self.wl.dt, self.stream)
            launches += KERNELS_PER_STEP_CALL if self.sorted else 1
            if evs is not None:
                b.record(self.stream); evs.append((a, b))
        self.it += 1
        return launches

    def timed(self, steps, warmup, barrier=lambda: None):
        """W warm-up steps, then exactly K timed steps between synchronisations; device time by CUDA events."""
        torch = self.torch
        for _ in range(warmup):
            self.one_step()
        torch.cuda.synchronize()
        barrier()
        upd0 = self.ctx.updates_total()
        evs, sevs = [], []
        t_a = torch.cuda.Event(enable_timing=True); t_b = torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t_a.record(self.stream)
        launches = 0
        for _ in range(steps):
            launches += self.one_step(evs, sevs)
        t_b.record(self.stream)
        torch.cuda.synchronize()
        barrier()
        ms = t_a.elapsed_time(t_b)
        updates = self.ctx.updates_total() - upd0
        return dict(ms=ms, updates=updates, launches=launches,
                    step_ms=sum(a.elapsed_time(b) for a, b in evs), n_step_calls=len(evs),
                    sort_ms=sum(a.elapsed_time(b) for a, b in sevs), n_sorts=len(sevs))

    def close(self):
        self.ctx.close()
        del self.sets, self.spare, self.J, self.fdev
        self.torch.cuda.empty_cache()


def roofline_of(prec, workload, r, peak_measured, peaks_file, peak_src, full_size, kernel):
    """The `roofline` object of one timed run r (DeviceRun.timed)."""
    upd_per_launch = r["updates"] / max(1, r["n_step_calls"])
    sec_per_launch = r["step_ms"] * 1e-3 / max(1, r["n_step_calls"])
    ach = FLOPS_PER_UPDATE_NITER10 * upd_per_launch / sec_per_launch / 1e12
    hbm_ach = BYTES_PER_UPDATE[prec] * upd_per_launch / sec_per_launch / 1e9
    prof = _profile_numbers(prec, workload) if full_size else None
    out = {"bound": "alu", "kernel": kernel, "achieved": ach, "peak": peak_measured, "unit": "TFLOP/s",
           "frac": ach / peak_measured,
           "frac_is": "ALGORITHMIC operations of the method at n_iter = 10 (2051 per update, DESIGN.md section 7; the two "
                      "fixed-point loops leave early once an iterate repeats bit for bit, so fewer are executed) per second "
                      "over the FMA peak measured in this run",
           "peak_source": ("measured in this run: grpic_probe FFMA/DFMA chains (CUDA events, best of 5)"
                           if abs(peak_measured - ALU_PEAK_DERIVED[prec]) > 1e-9 else "derived (the probe failed)"),
           "peak_derived": ALU_PEAK_DERIVED[prec],
           "flops_per_update": FLOPS_PER_UPDATE_NITER10, "updates_per_launch": upd_per_launch,
           "ms_per_launch": sec_per_launch * 1e3, "kernel_share_of_step": r["step_ms"] / r["ms"],
           "traffic": (prof["dram_bytes"] if prof else None),
           "hbm": {"achieved": hbm_ach, "peak": peaks_file["hbm_gbs"], "unit": "GB/s", "frac": hbm_ach / peaks_file["hbm_gbs"],
                   "bytes_per_update": BYTES_PER_UPDATE[prec], "peak_source": peak_src}}
    if prof:
        ex = prof["flop_executed"] / prof["particles"]
        out["executed"] = {"flop_per_update": ex, "achieved": ex * upd_per_launch / sec_per_launch / 1e12,
                           "frac": ex * upd_per_launch / sec_per_launch / 1e12 / peak_measured,
                           "warp_inst_per_32_particles": prof["inst_per_particle"],
                           "note": "FP instructions the kernel EXECUTES (2 x FFMA + FMUL + FADD of the committed ncu opcode "
                                   "histogram) per second over the same measured peak"}
        out["traffic_note"] = (f"dram__bytes_read.sum + dram__bytes_write.sum of one {prof['kernel']} launch over "
                               f"{prof['particles']:.0f} particles, {prof['source']}")
    return out


def _other_workload(G, name, steps, pk, peaks_file, peak_src):
    """A short run of the same loop on another single-GPU configuration of BASELINE.json."""
    w2 = _workload(name)
    run2 = DeviceRun(G, w2, w2.dtype)
    try:
        r2 = run2.timed(steps, 3)
    finally:
        run2.close()
    base = {"workload": _workload_desc(w2, 1), "dtype": w2.dtype, "steps": steps, "value": r2["updates"] / (r2["ms"] * 1e-3),
            "unit": UNIT, "ms_per_step": r2["ms"] / steps}
    if name.startswith("geodesic"):                     # config 2: q = 0 -> push only, direct kernel, no sort
        base["workload"] += " (config 2: zero-field geodesics, q = 0: no deposit, no sort)"
        return base
    rf = roofline_of(w2.dtype, name, r2, pk["ffma"] if w2.dtype == "f32" else pk["dfma"], peaks_file, peak_src, True,
                     "k_step_lanes (dense items) + k_step_tiled (sparse items)")
    base.update({"ms_per_launch": rf["ms_per_launch"], "frac": rf["frac"], "peak": rf["peak"], "hbm_frac": rf["hbm"]["frac"],
                 "executed": rf.get("executed")})
    return base


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
    barrier = (lambda: dist.barrier()) if world > 1 else (lambda: None)

    wl = _workload(args.workload, seed_offset=rank, shrink=args.shrink)
    prec = wl.dtype if args.precision is None else args.precision
    run = DeviceRun(G, wl, prec, knobs=args.set, no_tile=args.no_tile)
    sampler = ClockSampler(local) if rank == 0 else None      # nvidia-smi needs ~a second to start sampling
    r = run.timed(args.steps, args.warmup, barrier)
    clocks = sampler.stop() if sampler else None
    counters = run.ctx.counters()
    ms_max, updates_all = reduce_over_ranks(r["ms"], r["updates"], world)
    # the ALU denominators, measured on this GPU right after the timed region
    pk = None
    if rank == 0:
        try:
            pk = measure_peaks(run.ctx, kinds=("ffma", "dfma"))
        except Exception:                                # noqa: BLE001  (fall back to the derived peaks, and say so)
            pk = None

    # ---- end to end through the host-buffer ABI call (pinned host memory, copies inside the timed region)
    e2e = None
    if not args.no_e2e:
        ctx = run.ctx
        names = ("D1", "D2", "D3", "B1", "B2", "B3")
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        hsets = [G.ParticleSet.from_host(sp, prec, device="cpu", pinned=True) for sp in wl.species]
        hf = G.grid_tensors(wl.fields, names, prec, device="cpu", pinned=True)
        hJ = {k: torch.zeros(ctx.shape, dtype=G.torch_real(prec)).pin_memory() for k in ("J1", "J2", "J3")}
        up = down = 0
        for p in hsets:                      # warm-up: allocates the library's device chunks
            ctx.step_host(p, hf, hJ, wl.dt, with_prev=False)
        u0 = ctx.updates_total()
        torch.cuda.synchronize()
        barrier()
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
    sort_every = run.sort_every
    run.close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks_file, peak_src = _peaks_file()
    full = args.shrink == 1 and not args.no_tile and not args.set
    kernel = "k_step_lanes (dense items) + k_step_tiled (sparse items)" if not args.no_tile else "k_push_or_step<.,true>"
    peak_measured = pk is not None
    if pk is None:
        pk = {"ffma": ALU_PEAK_DERIVED["f32"], "dfma": ALU_PEAK_DERIVED["f64"]}
    peak = pk["ffma"] if prec == "f32" else pk["dfma"]
    out = {
        "metric": METRIC, "value": updates_all / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": prec, "data": "synthetic",
        "config": {"workload": _workload_desc(wl, args.shrink), "sort_every": sort_every,
                   "sort": "grpic_sort_into between two column sets per species; no *_prev columns (fused step); "
                           "sort_lookahead = sort_every/2",
                   "l2": "inputs (particle columns, several GB) larger than the 126 MB L2; no flush needed",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "paper_context": "paper: ~1.2-1.4e8 updates/s on 1x A100 (P:550), other hardware, not a target"},
        "roofline": roofline_of(prec, args.workload, r, peak, peaks_file, peak_src, full, kernel),
        "peaks_measured": {"fp32_fma_tflops": pk["ffma"], "fp64_fma_tflops": pk["dfma"], "measured": peak_measured},
        "without_sort": {"value": r["updates"] / (r["step_ms"] * 1e-3), "unit": UNIT,
                         "note": "fused step calls only (CUDA events around each grpic_step); `value` includes grpic_sort_into every sort_every steps and the J zero-fills"},
        "sort": {"ms_per_call": r["sort_ms"] / max(1, r["n_sorts"]), "calls": r["n_sorts"],
                 "note": "grpic_sort_into of one species (CUDA events around the call; no host synchronisation inside)"},
        "clocks": clocks, "gpu_launches": r["launches"],
        "counters_last_step": counters, "updates_timed": updates_all,
    }
    if e2e is not None:
        out["e2e"] = e2e
    # the other single-GPU configurations of BASELINE.json, each as a short run of the same loop (config 5 in FP64)
    if world == 1 and not args.no_others and args.workload == "large" and full:
        others = []
        for name in ("magnetosphere", "two_species", "geodesic", "geodesic_f64"):
            try:                                         # a side result must never cost the main line
                others.append(_other_workload(G, name, min(args.steps, 20), pk, peaks_file, peak_src))
            except Exception as e:                       # noqa: BLE001
                others.append({"workload": name, "error": f"{type(e).__name__}: {e}"})
        out["other_workloads"] = others
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline(args.workload, wl_full=wl if args.shrink == 1 else None)
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
    ap.add_argument("--no-others", action="store_true", help="skip the short runs of configs 3 and 5")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--peaks", action="store_true", help="print the measured FFMA / DFMA / MUFU / shared-RMW peaks and exit")
    ap.add_argument("--set", action="append", default=[], metavar="KEY=VALUE",
                    help="grpic_set_int / grpic_set_real knob for ablation runs (repeatable)")
    args = ap.parse_args()
    if args.peaks:
        run_peaks(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
