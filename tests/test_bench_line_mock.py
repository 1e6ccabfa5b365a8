"""bench.py's own arm end to end on CPU with the device layer replaced by a stand-in: every line of `run_ours`
(step loop, sort cadence, CUDA-event bookkeeping, measured peaks, e2e, the other workloads, cpu_baseline, the JSON
contract) executes here, so that a mistake in the host logic cannot first show on the GPU box.  Nothing of the method
is computed: the stand-in context only counts calls and alive particles."""
import io
import json
import sys
import types
from contextlib import redirect_stdout

import numpy as np
import pytest
import torch

import bench


class _Event:
    clock = 0.0

    def __init__(self, enable_timing=True):
        self.t = None

    def record(self, stream=None):
        _Event.clock += 1.0
        self.t = _Event.clock

    def elapsed_time(self, other):
        return other.t - self.t


class _Set:
    def __init__(self, n):
        self.n = n
        self.cols = {}

    def drop_prev(self):
        return self

    def empty_like(self):
        return _Set(self.n)


class _Ctx:
    def __init__(self, n1, n2, a, r_min, r_max, nghost=2, precision="f32", **kw):
        self.shape = (n1 + 2 * nghost, n2 + 2 * nghost)
        self.updates = 0
        self.calls = {"step": 0, "sort_into": 0, "probe": 0, "step_host": 0}
        self.knobs = {}

    def set_int(self, k, v): self.knobs[k] = v
    def set_real(self, k, v): self.knobs[k] = v

    def step(self, p, f, J, dt, stream=None):
        self.calls["step"] += 1
        self.updates += p.n

    def sort_into(self, a, b, stream=None): self.calls["sort_into"] += 1

    def probe(self, what, iters, stream=None):
        self.calls["probe"] += 1
        return 10 ** 12

    def step_host(self, p, f, J, dt, with_prev=True):
        self.calls["step_host"] += 1
        self.updates += p.n
        return 1000, 900

    def counters(self, stream=None): return {"alive": 1, "absorbed_in": 0, "absorbed_out": 0, "overstep": 0}
    def updates_total(self, stream=None): return self.updates
    def close(self): pass


@pytest.fixture
def fake_device(monkeypatch):
    G = types.ModuleType("fake_grpic")
    G.Context = _Ctx
    G.ParticleSet = types.SimpleNamespace(from_host=lambda sp, prec, device="cuda", pinned=False, with_phi=None: _Set(int(sp.n)))
    G.grid_tensors = lambda arrays, names, prec, device="cuda", pinned=False: {k: None for k in names}
    G.torch_real = lambda prec: torch.float32 if prec == "f32" else torch.float64
    import paper_2511_17701_b200
    monkeypatch.setitem(sys.modules, "paper_2511_17701_b200.grpic", G)
    monkeypatch.setattr(paper_2511_17701_b200, "grpic", G, raising=False)
    monkeypatch.setattr(torch.cuda, "is_available", lambda: True)
    monkeypatch.setattr(torch.cuda, "set_device", lambda d: None)
    monkeypatch.setattr(torch.cuda, "synchronize", lambda *a: None)
    monkeypatch.setattr(torch.cuda, "current_stream", lambda *a: None)
    monkeypatch.setattr(torch.cuda, "empty_cache", lambda: None)
    monkeypatch.setattr(torch.cuda, "Event", _Event)
    real_zeros = torch.zeros
    monkeypatch.setattr(torch, "zeros", lambda *a, **k: real_zeros(*a, **{kk: vv for kk, vv in k.items() if kk != "device"}))
    monkeypatch.setattr(torch.Tensor, "pin_memory", lambda self: self)
    monkeypatch.setattr(bench, "ClockSampler", lambda idx: types.SimpleNamespace(stop=lambda: {"sm_mhz": 1965.0, "sm_max_mhz": 1965.0, "reasons": [], "samples": 1}))
    # the workloads at 1/32 of their edge so that the oracle legs take seconds
    real = bench._workload
    monkeypatch.setattr(bench, "_workload", lambda name, seed_offset=0, shrink=1: real(name, seed_offset, shrink=max(shrink, 32)))
    return G


def _args(**kw):
    d = dict(gpus=1, steps=12, warmup=3, impl="ours", workload="large", shrink=1, precision=None, no_tile=False, no_e2e=False,
             no_cpu_baseline=False, no_others=False, e2e_steps=2, peaks=False, set=[])
    d.update(kw)
    return types.SimpleNamespace(**d)


def test_our_arm_prints_the_contract_line(fake_device, monkeypatch):
    monkeypatch.setenv("RANK", "0"); monkeypatch.setenv("WORLD_SIZE", "1"); monkeypatch.setenv("LOCAL_RANK", "0")
    buf = io.StringIO()
    with redirect_stdout(buf):
        bench.run_ours(_args())
    d = json.loads(buf.getvalue().strip().splitlines()[-1])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks"):
        assert k in d, k
    assert d["unit"] == "updates/s" and d["value"] > 0 and d["vs_baseline"] is None and d["dtype"] == "f32"
    assert "workload" in d["config"] and "model" not in d["config"]
    r = d["roofline"]
    assert r["bound"] == "alu" and abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and r["flops_per_update"] == 2051.0
    assert r["hbm"]["unit"] == "GB/s" and r["traffic"] is not None and r["executed"]["frac"] > 0      # committed ncu extract read
    assert d["peaks_measured"]["measured"] is True
    # 12 timed steps from it = 3: one sort of both species at it = 10; 3 kernels per grpic_step call, 11 per sort
    assert d["gpu_launches"] == 12 * 2 * bench.KERNELS_PER_STEP_CALL + 2 * bench.KERNELS_PER_SORT and d["sort"]["calls"] == 2
    assert d["e2e"]["h2d_bytes_per_step"] == 2000 and d["e2e"]["d2h_bytes_per_step"] == 1800
    names = [o["workload"] for o in d["other_workloads"]]
    assert len(names) == 4 and not any("error" in o for o in d["other_workloads"]), d["other_workloads"]
    assert d["other_workloads"][1]["dtype"] == "f64" and "frac" in d["other_workloads"][1] and "frac" not in d["other_workloads"][2]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] > 0 and 2000 < cb["ops_per_update_counted"] < 5000


def test_a_failing_side_workload_does_not_cost_the_main_line(fake_device, monkeypatch):
    monkeypatch.setenv("RANK", "0"); monkeypatch.setenv("WORLD_SIZE", "1"); monkeypatch.setenv("LOCAL_RANK", "0")

    def boom(*a, **k):
        raise RuntimeError("device fault")
    monkeypatch.setattr(bench, "_other_workload", boom)
    monkeypatch.setattr(bench, "measure_peaks", boom)
    buf = io.StringIO()
    with redirect_stdout(buf):
        bench.run_ours(_args(no_cpu_baseline=True, no_e2e=True))
    d = json.loads(buf.getvalue().strip().splitlines()[-1])
    assert d["value"] > 0 and all("error" in o for o in d["other_workloads"])
    assert d["peaks_measured"]["measured"] is False and d["roofline"]["peak_source"].startswith("derived")
    assert abs(d["roofline"]["peak"] - bench.ALU_PEAK_DERIVED["f32"]) < 1e-9


def test_geodesic_workload_is_not_sorted(fake_device):
    run = bench.DeviceRun(fake_device, bench._workload("geodesic"), "f32")
    r = run.timed(12, 3)
    assert run.ctx.calls["sort_into"] == 0 and r["launches"] == 12 and r["n_sorts"] == 0
