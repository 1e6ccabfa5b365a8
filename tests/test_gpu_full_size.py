"""Full-size GPU checks (pytest -m gpu): BASELINE.json's configs at their real sizes, in the launch
configuration bench.py times (config 4: no *_prev columns, grpic_sort_into between two column sets, then the fused
tiled grpic_step, sort_lookahead = 5; configs 3 and 5: the in-place grpic_sort with all columns), checked on sampled particles
the oracle recomputes one by one and on properties that hold at any size (discrete continuity Eq. 32/34,
first moments, conserved u_3 and energy of geodesics)."""
import numpy as np
import pytest

from helpers import (TOL, compare_current, compare_particles, grid_from_domain, oracle_deposit_as_the_gpu_decided,
                     oracle_from_cols)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def G():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2511_17701_b200 import grpic
    grpic.load("f32"); grpic.load("f64")
    return grpic


def _gather(ps, idx):
    return {k: (None if v is None else v[idx].cpu().numpy().copy()) for k, v in ps.cols.items()}


def _cic_rho(torch, shape, ng, i1, i2, dx1, dx2, qw, mask):
    """rho~ on nodes with the linear shape (the definition Eq. 32/34 is written for), FP64 on the device."""
    ld = shape[1]
    rho = torch.zeros(shape[0] * shape[1], dtype=torch.float64, device=i1.device)
    base = (i1.long() + ng) * ld + (i2.long() + ng)
    x, y = dx1.double(), dx2.double()
    q = torch.where(mask, qw.double(), torch.zeros_like(x))
    for a, wx in ((0, 1 - x), (1, x)):
        for b, wy in ((0, 1 - y), (1, y)):
            rho.index_add_(0, base + a * ld + b, q * wx * wy)
    return rho.view(shape)


@pytest.mark.parametrize("name,prec,tol_cont,tol_mom", [("large", "f32", 5e-6, 1e-6),
                                                        ("magnetosphere", "f32", 5e-6, 1e-6),
                                                        ("two_species", "f64", 1e-13, 1e-13)])
def test_configs_3_4_5_full_size(G, O, W, name, prec, tol_cont, tol_mom):
    """Configs 3, 4, 5 at full size (config 4: 2048x1024, 134M particles, FP32, the bench workload): sort + tiled
    fused step as bench.py runs it.
    (a) 2^17 sampled particles per species (plus the ragged ends of the sorted order) against the oracle;
    (b) counters add up; (c) discrete continuity of the deposited J with the particles' own (prev -> new)
    positions at every node; (d) first moments of J."""
    import torch
    wl = dict(large=W.config_large, magnetosphere=W.config_magnetosphere, two_species=W.config_two_species)[name]()
    dom = wl.dom
    g = grid_from_domain(O, dom)
    ctx = G.Context(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, nghost=dom.ng, precision=prec)
    names = ("D1", "D2", "D3", "B1", "B2", "B3")
    fdev = G.grid_tensors(wl.fields, names, prec)
    fhost = {k: fdev[k].cpu().numpy().astype(np.float64) for k in names}
    Jtot = {k: torch.zeros(ctx.shape, dtype=torch.float64, device="cuda") for k in ("J1", "J2", "J3")}
    J = {k: torch.zeros(ctx.shape, dtype=G.torch_real(prec), device="cuda") for k in ("J1", "J2", "J3")}
    rng = np.random.default_rng(44)
    rho_diff = torch.zeros(ctx.shape, dtype=torch.float64, device="cuda")
    m1 = m2 = 0.0
    scale = 0.0
    bench_cfg = name == "large"                 # exactly what bench.py launches
    for sp in wl.species:
        ps = G.ParticleSet.from_host(sp, prec)
        n = ps.n
        if bench_cfg:
            src = ps.drop_prev()
            ps = src.empty_like()
            ctx.sort_into(src, ps)
            ctx.set_real("sort_lookahead", 5.0)       # as bench.py: key of the cell predicted half an interval ahead
            for _ in range(2):
                ctx.step(ps, fdev, J, wl.dt)
            ctx.sort_into(ps, src)
            ps = src
            del src
        else:
            ctx.sort(ps)
        ctx.step(ps, fdev, J, wl.dt)            # one step to leave the freshly sorted state (drifted particles)
        for v in J.values():
            v.zero_()
        idx_np = np.unique(np.concatenate([rng.integers(0, n, 1 << 17), np.arange(0, 4096), np.arange(n - 4096, n)]))
        idx = torch.from_numpy(idx_np).cuda()
        before = _gather(ps, idx)
        prev = {k: ps.cols[k].clone() for k in ("i1", "i2", "dx1", "dx2")}      # the position the step starts from
        ctx.step(ps, fdev, J, wl.dt)
        c = ctx.counters()
        for k in J:
            Jtot[k] += J[k].double()
        scale = max(scale, float(J["J1"].abs().max()), float(J["J2"].abs().max()))   # largest one-species |J| entry
        after = _gather(ps, idx)
        # (a) sampled particles, one by one in the oracle
        op = oracle_from_cols(O, before, ps.q_over_m, ps.charge, ps.massive)
        diag = {}
        O.push(g, op, fhost, wl.dt, diag=diag)
        res = compare_particles(op, after, prec, before["tag"], g.n1, g.n2, diag=diag, check_prev=not bench_cfg)
        if not bench_cfg:                       # the *_prev columns the kernel wrote are that position
            for k in prev:
                assert torch.equal(ps.cols[k + "_prev"][ps.cols["tag"] != 0], prev[k][ps.cols["tag"] != 0]), k
        print(name, "full", sp.name, res, c)
        # (b) counters
        alive_after = int(ps.cols["tag"].sum())
        assert c["alive"] == alive_after and c["overstep"] == 0
        assert c["alive"] + c["absorbed_in"] + c["absorbed_out"] <= n
        # (c), (d) accumulate continuity terms of this species: particles alive after the step deposited
        m = ps.cols["tag"] != 0
        qw = ps.cols["weight"] * ps.charge
        rho_new = _cic_rho(torch, ctx.shape, dom.ng, ps.cols["i1"], ps.cols["i2"], ps.cols["dx1"], ps.cols["dx2"], qw, m)
        rho_old = _cic_rho(torch, ctx.shape, dom.ng, prev["i1"], prev["i2"], prev["dx1"], prev["dx2"], qw, m)
        rho_diff += rho_new - rho_old
        d1 = (ps.cols["i1"] - prev["i1"]).double() + (ps.cols["dx1"].double() - prev["dx1"].double())
        d2 = (ps.cols["i2"] - prev["i2"]).double() + (ps.cols["dx2"].double() - prev["dx2"].double())
        q64 = torch.where(m, qw.double(), torch.zeros_like(d1))
        m1 += float((q64 * d1).sum()) / wl.dt
        m2 += float((q64 * d2).sum()) / wl.dt
        scale_sp = float(q64.abs().sum()) / wl.dt
        del ps, prev, rho_new, rho_old, d1, d2, q64
        torch.cuda.empty_cache()
    J1, J2 = Jtot["J1"], Jtot["J2"]
    div = torch.zeros_like(J1)
    div[1:, :] += J1[1:, :] - J1[:-1, :]
    div[:, 1:] += J2[:, 1:] - J2[:, :-1]
    resid = rho_diff / wl.dt + div
    # scale: the largest one-species |J| entry; FP32 sums of a few hundred contributions per entry -> ~1e-6 relative
    r = float(resid[1:, 1:].abs().max()) / scale
    print(name, "full: continuity residual / max|J| =", r)
    assert r < tol_cont
    # first moments: sum over the grid of J^i = sum_p q w dx^i/dt   (species of opposite charge cancel in the
    # total, so compare against the per-species magnitude scale)
    e1 = abs(float(J1.sum()) - m1) / scale_sp
    e2 = abs(float(J2.sum()) - m2) / scale_sp
    print(name, "full: first-moment errors", e1, e2)
    assert e1 < tol_mom and e2 < tol_mom


@pytest.mark.parametrize("name,prec", [("large", "f32"), ("two_species", "f64")])
def test_full_size_every_particle_and_every_J_entry(G, O, W, name, prec):
    """Element-wise parity at full size in the launch configuration bench.py times: one species of config 4
    (2048x1024, 67 M electrons, FP32) and of config 5 (1024x1024, 33.5 M electrons, FP64) - two column sets without
    *_prev, grpic_sort_into with sort_lookahead = 5, three steps of drift, then ONE fused grpic_step whose result is
    compared with the oracle run on ALL particles of the species: every particle (compare_particles) and every entry
    of J^1, J^2, J^3 (Eq. 34, 36) at 1e-5 max|J| (FP32) / 1e-10 max|J| (FP64)."""
    import torch
    wl = dict(large=W.config_large, two_species=W.config_two_species)[name]()
    dom = wl.dom
    g = grid_from_domain(O, dom)
    ctx = G.Context(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, nghost=dom.ng, precision=prec)
    names = ("D1", "D2", "D3", "B1", "B2", "B3")
    fdev = G.grid_tensors(wl.fields, names, prec)
    fhost = {k: fdev[k].cpu().numpy().astype(np.float64) for k in names}
    J = {k: torch.zeros(ctx.shape, dtype=G.torch_real(prec), device="cuda") for k in ("J1", "J2", "J3")}
    sp = wl.species[0]
    src = G.ParticleSet.from_host(sp, prec).drop_prev()
    ps = src.empty_like()
    ctx.sort_into(src, ps)                                # first sort: present-cell key (no dt yet)
    ctx.set_real("sort_lookahead", 5.0)
    for _ in range(2):
        ctx.step(ps, fdev, J, wl.dt)
    ctx.sort_into(ps, src)                                # look-ahead sort, as in bench.py's steady state
    ps = src
    for _ in range(3):                                    # drift away from the sorted order
        ctx.step(ps, fdev, J, wl.dt)
    for v in J.values():
        v.zero_()
    before = ps.to_numpy()
    ctx.step(ps, fdev, J, wl.dt)
    c = ctx.counters()
    after = ps.to_numpy()
    Jg = {k: v.cpu().numpy().astype(np.float64) for k, v in J.items()}
    del ps, src, J
    torch.cuda.empty_cache()
    op = oracle_from_cols(O, before, sp.q_over_m, sp.charge, sp.massive)
    diag = {}
    alive, a_in, a_out = O.push(g, op, fhost, wl.dt, diag=diag)
    res = compare_particles(op, after, prec, before["tag"], g.n1, g.n2, diag=diag, check_prev=False)
    Jo, over, n_sub = oracle_deposit_as_the_gpu_decided(O, g, op, after, before["tag"], wl.dt, prec)
    if n_sub == 0:
        assert (c["alive"], c["absorbed_in"], c["absorbed_out"], c["overstep"]) == (alive, a_in, a_out, over)
    res.update(compare_current(Jo, Jg, prec))
    print(name, "full, all particles:", res, c, "substituted", n_sub)
    assert c["alive"] > 0.9 * int((before["tag"] != 0).sum()) and c["absorbed_in"] > 0


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_config2_geodesic_full_size_100_steps(G, O, W, prec):
    """Config 2 at full size: 2^24 zero-charge particles, a = 0.95, 100 steps of dt = 0.01.
    Sampled particles against the oracle at the first and the last step; u_3 bit-identical after 100 steps
    (Eq. 27: u~_3 = u_3); the circular-orbit half keeps its radius (fixed points of Eq. 28-29) and the
    conserved energy -u_0 = alpha*gamma - beta^1 u_1 of every surviving geodesic stays within the
    integrator's second-order error."""
    import torch
    from helpers import energy_u0
    wl = W.config_geodesic(n=1 << 24, dtype=prec)
    dom = wl.dom
    g = grid_from_domain(O, dom)
    ctx = G.Context(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, nghost=dom.ng, precision=prec)
    ps = G.ParticleSet.from_host(wl.species[0], prec)
    n = ps.n
    u3_0 = ps.cols["u3"].clone()
    rng = np.random.default_rng(22)
    idx_np = np.unique(np.concatenate([rng.integers(0, n, 1 << 16), np.arange(0, 1024), np.arange(n - 1024, n)]))
    idx = torch.from_numpy(idx_np).cuda()
    s0 = _gather(ps, idx)
    E0 = energy_u0(O, g, s0["i1"] + s0["dx1"].astype(np.float64), s0["i2"] + s0["dx2"].astype(np.float64),
                   s0["u1"].astype(np.float64), s0["u2"].astype(np.float64), s0["u3"].astype(np.float64))
    for step in range(wl.steps):
        check = step in (0, wl.steps - 1)
        if check:
            before = _gather(ps, idx)
        ctx.step(ps, None, None, wl.dt)
        if check:
            after = _gather(ps, idx)
            op = oracle_from_cols(O, before, 0.0, 0.0, 1)
            diag = {}
            O.push(g, op, None, wl.dt, diag=diag)
            res = compare_particles(op, after, prec, before["tag"], g.n1, g.n2, diag=diag)
            print("config2 full", prec, "step", step, res)
    assert torch.equal(ps.cols["u3"], u3_0), "u_3 must be untouched by 100 geodesic steps"
    s1 = _gather(ps, idx)
    alive = s1["tag"] != 0
    assert alive.sum() > 0.4 * len(idx_np)            # the circular half survives
    E1 = energy_u0(O, g, s1["i1"] + s1["dx1"].astype(np.float64), s1["i2"] + s1["dx2"].astype(np.float64),
                   s1["u1"].astype(np.float64), s1["u2"].astype(np.float64), s1["u3"].astype(np.float64))
    dE = np.abs(E1 / E0 - 1.0)[alive]
    # plungers close to the horizon have large second-order errors at dt = 0.01; the bound is on the bulk
    tol_E = 1e-4
    print("config2 full", prec, "energy drift: median", np.median(dE), "99%", np.quantile(dE, 0.99), "max", dE.max())
    assert np.quantile(dE, 0.99) < tol_E and dE.max() < 5e-4
    # circular orbits (first half of the arrays) stay at their radius: |dr/r| small after t = 1
    circ = idx_np < n // 2
    x1_0 = s0["i1"] + s0["dx1"].astype(np.float64); x1_1 = s1["i1"] + s1["dx1"].astype(np.float64)
    drift = np.abs(x1_1 - x1_0)[circ & alive]
    print("config2 full", prec, "circular-orbit radial drift (cells): max", drift.max())
    assert drift.max() < 0.05
