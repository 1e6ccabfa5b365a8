"""A complete GRPIC run through the C ABI: config 1 ("Tiny": Kerr a = 0.9, 128x64, Wald field, e+- pairs) for a few
hundred timesteps of the closed loop of Sec. 3.4 — fields_prepare -> fused particle step -> fields_advance -> field
boundary conditions (axis reflection, constant layer inside the horizon, absorbing layer over the outer 15 % of the
radial range matched to the initial Wald field), with a cell sort every 10 steps.

    python -m paper_2511_17701_b200.example [--steps 200] [--precision f32|f64] [--k_J 1e-5]

Needs a CUDA device (there is no CPU path).  k_J scales the coupling of the deposited current back into Ampere's law:
the macro-particles of the synthetic workload carry unit weight, so the physical 4 pi would make an absurdly dense
plasma; the default keeps the run in the weakly loaded regime.
"""
from __future__ import annotations

import argparse

import numpy as np


def main():
    import torch
    from . import grpic as G, workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--precision", default="f32", choices=["f32", "f64"])
    ap.add_argument("--k_J", type=float, default=1e-5)
    args = ap.parse_args()
    assert torch.cuda.is_available(), "this example needs a CUDA device"
    wl = W.config_tiny()
    dom, prec = wl.dom, args.precision
    ctx = G.Context(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, nghost=dom.ng, precision=prec)
    ctx.set_real("k_J", args.k_J)
    rt = G.torch_real(prec)
    kb, kd, kj = ("B1", "B2", "B3"), ("D1", "D2", "D3"), ("J1", "J2", "J3")
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(rt).cuda()
    state = dict(B_prev={k: t(wl.fields[k]) for k in kb}, B={k: t(wl.fields[k]) for k in kb},
                 D_prev={k: t(wl.fields[k]) for k in kd}, D={k: t(wl.fields[k]) for k in kd})
    zeros = lambda ks: {k: torch.zeros(ctx.shape, dtype=rt, device="cuda") for k in ks}
    B_n, J_prev = zeros(kb), zeros(kj)
    species = [G.ParticleSet.from_host(sp, prec) for sp in wl.species]
    D0 = {k: v.clone() for k, v in state["D"].items()}
    target = {**D0, **{k: v.clone() for k, v in state["B"].items()}}   # the absorbing layer matches to the initial field
    r_abs = dom.r_max - 0.15 * (dom.r_max - dom.r_min)
    for step in range(args.steps):
        if step % 10 == 0:
            for ps in species:
                ctx.sort(ps)
        ctx.fields_prepare(state, B_n, wl.dt)                       # (n)B aligned with (n)D
        J = zeros(kj)
        for ps in species:
            ctx.step(ps, {**state["D"], **B_n}, J, wl.dt)           # interp + push + BCs + deposit
        ctx.filter_current(J, 1)
        ctx.fields_advance(state, B_n, J_prev, J, wl.dt)            # Faraday, two Ampere sub-steps
        ctx.field_bc({**state["D"], **state["B"]}, 1)               # axis reflection, constant layer inside the horizon
        ctx.field_match({**state["D"], **state["B"]}, target, r_abs)   # absorbing layer at the outer edge
        J_prev = J
        if (step + 1) % 50 == 0 or step + 1 == args.steps:
            alive = sum(int(ps.cols["tag"].sum()) for ps in species)
            lo = dom.ng + 4                                            # outside the constant layer at the inner edge
            dD = max(float((state["D"][k] - D0[k])[lo:].abs().max() / D0[k][lo:].abs().max()) for k in ("D1", "D2"))
            print(f"step {step + 1:5d}  t = {(step + 1) * wl.dt:7.3f} r_g  alive {alive:7d}  "
                  f"max|J| {max(float(v.abs().max()) for v in J.values()):.3e}  max rel. change of D^1,2 {dD:.3e}")
    ctx.close()


if __name__ == "__main__":
    main()
