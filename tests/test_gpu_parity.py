"""GPU-vs-oracle parity through the C ABI (pytest -m gpu).  Same seeded inputs on both sides; the
oracle (FP64, CPU) is the reference; tolerances are north_star's (helpers.TOL).

Every case runs the library through paper_2511_17701_b200.grpic (ctypes -> libgrpic_*.so)."""
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
    grpic.load("f32"); grpic.load("f64")       # fail loudly if the extension is missing
    return grpic


def _ctx(G, dom, prec, n_iter=10):
    return G.Context(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, nghost=dom.ng, precision=prec, n_iter=n_iter)


def _zeros_J(G, ctx, prec):
    import torch
    return {k: torch.zeros(ctx.shape, dtype=G.torch_real(prec), device="cuda") for k in ("J1", "J2", "J3")}


def _J_np(J):
    return {k: v.detach().cpu().numpy().astype(np.float64) for k, v in J.items()}


def _fields_both(G, wl, prec):
    """device tensors for the GPU and the same (precision-rounded) values as FP64 numpy for the oracle"""
    names = ("D1", "D2", "D3", "B1", "B2", "B3")
    dev = G.grid_tensors(wl.fields, names, prec)
    host = {k: dev[k].cpu().numpy().astype(np.float64) for k in names}
    return dev, host


def _one_step_parity(G, O, ctx, g, ps, fdev, fhost, dt, prec, mode, sort_first=False):
    """One step of species `ps` on the GPU (mode: 'split' = interp_push + deposit, 'fused' = step),
    the same step in the oracle from the GPU's own input state; returns the maxima."""
    if sort_first:
        ctx.sort(ps)
    before = ps.to_numpy()
    op = oracle_from_cols(O, before, ps.q_over_m, ps.charge, ps.massive)
    J = _zeros_J(G, ctx, prec)
    if mode == "split":
        ctx.interp_push(ps, fdev, dt)
        c_push = ctx.counters()
        ctx.deposit(ps, J)
        c = ctx.counters()
        c.update({k: c_push[k] for k in ("alive", "absorbed_in", "absorbed_out")})
    else:
        ctx.step(ps, fdev, J, dt)
        c = ctx.counters()
    diag = {}
    alive, a_in, a_out = O.push(g, op, fhost if ps.q_over_m != 0 and ps.massive else None, dt, diag=diag)
    after = ps.to_numpy()
    res = compare_particles(op, after, prec, before["tag"], g.n1, g.n2, diag=diag,
                            check_prev=before["i1_prev"] is not None)
    Jo, over, n_sub = oracle_deposit_as_the_gpu_decided(O, g, op, after, before["tag"], dt, prec)
    if n_sub:                                          # a face-straddler may have been absorbed on one side only
        alive, a_in, a_out = int(op.tag[before["tag"] != 0].sum()), None, None
        assert c["absorbed_in"] + c["absorbed_out"] == int((before["tag"] != 0).sum()) - alive
    exp = (alive, a_in, a_out, over)
    got = (c["alive"], c["absorbed_in"], c["absorbed_out"], c["overstep"])
    assert all(e is None or e == v for e, v in zip(exp, got)), (c, exp)
    res.update(compare_current(Jo, _J_np(J), prec))
    return res, c


@pytest.mark.parametrize("mode", ["split", "fused"])
def test_config1_tiny_f64_10_steps(G, O, W, mode):
    """BASELINE config 1 at full size: Kerr a=0.9, 128x64, Wald field, 16 pairs-particles/cell, FP64, 10 steps.
    Per-step parity (the oracle restarts every step from the GPU state), both species."""
    wl = W.config_tiny()
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, "f64")
    fdev, fhost = _fields_both(G, wl, "f64")
    sets = [G.ParticleSet.from_host(sp, "f64") for sp in wl.species]
    absorbed = 0
    worst = dict(x_err=0.0, u_err=0.0, J3=0.0)
    for step in range(wl.steps):
        for ps in sets:
            res, c = _one_step_parity(G, O, ctx, g, ps, fdev, fhost, wl.dt, "f64", mode)
            absorbed += c["absorbed_in"] + c["absorbed_out"]
            for k in worst:
                worst[k] = max(worst[k], res[k])
    assert absorbed > 0, "config 1 must exercise absorption inside the horizon"
    print("config1", mode, worst, "absorbed", absorbed)


def test_config1_tiled_path_f64(G, O, W):
    """Same workload through grpic_sort + the shared-memory tile kernel, several steps between sorts."""
    wl = W.config_tiny()
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, "f64")
    fdev, fhost = _fields_both(G, wl, "f64")
    sets = [G.ParticleSet.from_host(sp, "f64") for sp in wl.species]
    for step in range(6):
        for ps in sets:
            _one_step_parity(G, O, ctx, g, ps, fdev, fhost, wl.dt, "f64", "fused", sort_first=(step % 3 == 0))


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_config2_geodesic_sample(G, O, W, prec):
    """Config 2 (zero-field geodesics, a=0.95, q=0): a 2^17-particle sample against the oracle, 5 steps;
    u_3 must come back bit-identical (Eq. 27: u~_3 = u_3)."""
    wl = W.config_geodesic(n=1 << 17, dtype=prec)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, prec)
    ps = G.ParticleSet.from_host(wl.species[0], prec)
    u3_0 = ps.cols["u3"].clone()
    for step in range(5):
        res, c = _one_step_parity(G, O, ctx, g, ps, None, None, wl.dt, prec, "fused")
    import torch
    assert torch.equal(ps.cols["u3"], u3_0)
    print("config2", prec, res)


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_massless_particles(G, O, W, prec):
    """Photons (Eq. 20 with eps = 0; EM push skipped): the config-2 sample pushed as massless
    particles, 5 steps, against the oracle (whose massless branch is pinned by radial null rays dr/dt = -1);
    a massless species with a charge still deposits its current (split and fused paths)."""
    wl = W.config_geodesic(n=1 << 16, dtype=prec)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, prec)
    sp = wl.species[0]
    sp.massive = 0
    sp.charge = 1.0                      # q_over_m stays 0: no EM push, but the particle carries current
    for mode in ("fused", "split"):
        ps = G.ParticleSet.from_host(sp, prec)
        for step in range(5):
            res, c = _one_step_parity(G, O, ctx, g, ps, None, None, wl.dt, prec, mode)
        print("massless", prec, mode, res, c)


def _shrunk(W, name, shrink):
    return dict(magnetosphere=W.config_magnetosphere, large=W.config_large, two_species=W.config_two_species)[name](shrink=shrink)


@pytest.mark.parametrize("name,shrink,prec", [("magnetosphere", 8, "f32"), ("large", 16, "f32"),
                                              ("two_species", 8, "f64"), ("two_species", 8, "f32")])
@pytest.mark.parametrize("mode", ["split", "fused", "tiled", "tiled_split"])
def test_configs_3_4_5_shrunk(G, O, W, name, shrink, prec, mode):
    """Configs 3-5 with both grid edges divided by `shrink` (per-cell counts, fields, dt recipe kept):
    several tiles and a ragged tail; 3 steps per species."""
    wl = _shrunk(W, name, shrink)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, prec)
    fdev, fhost = _fields_both(G, wl, prec)
    sets = [G.ParticleSet.from_host(sp, prec) for sp in wl.species]
    worst = {}
    for step in range(3):
        for ps in sets:
            # "tiled": sort, then the fused tile kernel; "tiled_split": sort, then grpic_interp_push + the tiled grpic_deposit
            res, c = _one_step_parity(G, O, ctx, g, ps, fdev, fhost, wl.dt, prec,
                                      {"tiled": "fused", "tiled_split": "split"}.get(mode, mode),
                                      sort_first=(mode.startswith("tiled") and step == 0))
            for k, v in res.items():
                worst[k] = max(worst.get(k, 0), v)
    print(name, prec, mode, worst)


@pytest.mark.parametrize("n1,n2,ng,n_iter,tma,prec", [(90, 43, 1, 10, 1, "f32"),    # ragged tiles, ld*4 = 180 B: TMA refused -> plain staging
                                                      (90, 44, 2, 10, 1, "f32"),    # ragged tiles, TMA path
                                                      (90, 44, 2, 3, 0, "f64"),     # TMA switched off, few iterations
                                                      (50, 30, 3, 1, 1, "f64"),     # n_iter = 1 (explicit Euler), wide ghosts
                                                      (16, 16, 2, 10, 1, "f32")])   # one tile
def test_ragged_grids_ghost_widths_iteration_counts(G, O, W, n1, n2, ng, n_iter, tma, prec):
    """Grids that are not multiples of the 16-cell tile, 1-3 ghost layers, n_iter = 1, 3, 10, TMA on / off /
    refused (row pitch not a multiple of 16 bytes): split, fused and tiled paths against the oracle, 3 steps."""
    a = 0.8
    dom = W.Domain(n1, n2, a, 0.9 * W.horizon_radius(a), 25.0, ng)
    rng = np.random.Generator(np.random.Philox(n1 * 1000 + n2))
    fields = W.add_random_dB(dom, W.wald_fields(dom, 1.0), 0.1, rng)
    species = W._pairs(dom, W.counts_uniform(dom, 6), 0.5, rng)
    dt = W.cfl_dt(dom)
    g = grid_from_domain(O, dom, n_iter=n_iter)
    ctx = _ctx(G, dom, prec, n_iter=n_iter)
    ctx.set_int("tma", tma)
    names = ("D1", "D2", "D3", "B1", "B2", "B3")
    fdev = G.grid_tensors(fields, names, prec)
    fhost = {k: fdev[k].cpu().numpy().astype(np.float64) for k in names}
    for mode in ("split", "fused", "tiled"):
        sets = [G.ParticleSet.from_host(sp, prec) for sp in species]
        for step in range(3):
            for ps in sets:
                res, c = _one_step_parity(G, O, ctx, g, ps, fdev, fhost, dt, prec, "fused" if mode == "tiled" else mode,
                                          sort_first=(mode == "tiled" and step == 0))
    print("ragged", n1, n2, ng, n_iter, tma, prec, res, c)


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("r0,h0,lin,mass", [(0.6, 0.0, 0, 1.0), (0.0, 0.35, 0, 1.0), (0.5, -0.3, 0, 1.0), (0.0, 0.0, 1, 1.0),
                                            (0.0, 0.4, 1, 1.0), (0.0, 0.0, 1, 0.0)])
def test_general_a3_map(G, O, W, prec, r0, h0, lin, mass):
    """Full map of App. A.3: radial offset r0 and polar stretch h0.  The oracle's map is
    pinned by finite differences and brute-force traces (test_oracle_*); here the general-map kernels against it:
    split and fused paths, charged particles in smooth random fields, 4 steps."""
    a, n1, n2, ng = (0.9 if mass else 0.0), 96, 48, 2      # mass = 0, a = 0: flat kerr_schild_0 of App. A.1
    # lin = 1: the uniform-r map of App. A.2 (r_map = 0), here also combined with the polar stretch
    g = O.Grid(n1, n2, a, 0.9 * W.horizon_radius(a), 12.0 if lin else 30.0, ng=ng, r0=r0, h0=h0, linear_r=lin, mass=mass)
    rng = np.random.Generator(np.random.Philox(int(1000 * r0 + 100 * (h0 + 1)) + lin))
    shape = (n1 + 2 * ng, n2 + 2 * ng)
    ii, jj = np.meshgrid(np.arange(shape[0]), np.arange(shape[1]), indexing="ij")
    fields = {k: 0.3 * np.sin(0.21 * ii + p) * np.cos(0.17 * jj - p) + 0.05 * rng.uniform(-1, 1, shape)
              for p, k in enumerate(("D1", "D2", "D3", "B1", "B2", "B3"))}
    n = 40000
    # particles in every cell, the two rows next to the axes included: they reflect through the general map.
    # FP64: anywhere in the cell.  FP32: a lone particle a few 1e-4 cells from the axis owns max|J3| of this small case
    # (v^3 ~ 1/sin^2 theta) and the FP32 conditioning of 1/sin^2 at that angle, not the kernel, would set the J3 error,
    # so FP32 starts at least 0.1 cell from an axis (reflections still happen: paths of up to 0.4 cell per step).
    i1 = rng.integers(0, n1, n).astype(np.int32); i2 = rng.integers(0, n2, n).astype(np.int32)
    dx1, dx2 = rng.random(n), rng.random(n)
    if prec == "f32":
        dx2 = np.where(i2 == 0, np.maximum(dx2, 0.1), np.where(i2 == n2 - 1, np.minimum(dx2, 0.9), dx2))
    m = O.metric(g, i1 + dx1, i2 + dx2, derivs=False)
    uh = rng.uniform(-0.7, 0.7, (3, n))                       # roughly orthonormal-frame sized momenta
    cells = O.metric(g, *[v.ravel() for v in np.meshgrid(np.arange(n1) + 0.5, np.arange(n2) + 0.5, indexing="ij")], derivs=False)
    dt = 0.4 * float(np.min(1.0 / np.sqrt(cells["hu11"] + cells["hu22"])))

    class S:
        pass
    for q in (-1.0, 1.0):
        sp = S()
        sp.i1, sp.i2, sp.dx1, sp.dx2 = i1, i2, dx1, dx2
        sp.u1, sp.u2, sp.u3 = uh[0] * m["s1"], uh[1] * m["s2"] * m["r"], uh[2] * m["r"] * m["sth"]
        sp.weight = rng.random(n) + 0.5; sp.tag = np.ones(n, np.uint8); sp.phi = np.zeros(n)
        sp.q_over_m, sp.charge, sp.massive = q, q, 1
        ctx = G.Context(n1, n2, a, g.r_min, g.r_max, nghost=ng, precision=prec, r0=r0, h0=h0, r_map=0 if lin else 1, mass=mass)
        names = ("D1", "D2", "D3", "B1", "B2", "B3")
        fdev = G.grid_tensors(fields, names, prec)
        fhost = {k: fdev[k].cpu().numpy().astype(np.float64) for k in names}
        for mode in ("split", "fused"):
            ps = G.ParticleSet.from_host(sp, prec)
            ctx.sort(ps)                                  # a sorted species must still take the general-map kernels
            for step in range(4):
                res, c = _one_step_parity(G, O, ctx, g, ps, fdev, fhost, dt, prec, mode)
        print("map", "A.2" if lin else "A.3", r0, h0, prec, q, res, c)


def test_sort_is_a_permutation_into_key_order(G, O, W):
    import torch
    wl = W.config_large(shrink=16)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, "f32")
    sp = wl.species[0]
    rng = np.random.default_rng(7)
    perm = rng.permutation(sp.n)
    for k in ("i1", "i2", "dx1", "dx2", "u1", "u2", "u3", "weight", "tag", "phi"):
        setattr(sp, k, getattr(sp, k)[perm])
    sp.tag = sp.tag.copy(); sp.tag[rng.random(sp.n) < 0.1] = 0
    sp.weight = rng.random(sp.n) + 0.5
    ps = G.ParticleSet.from_host(sp, "f32")
    ps.cols["i1_prev"].copy_(torch.arange(sp.n, dtype=torch.int32))          # unique id to track the permutation
    before = ps.to_numpy()
    ctx.sort(ps)
    after = ps.to_numpy()
    ids = after["i1_prev"]
    assert np.array_equal(np.sort(ids), np.arange(sp.n))                      # a permutation
    for k, v in after.items():
        if v is not None:
            assert np.array_equal(v, before[k][ids]), k                       # every column moved alike
    T = ctx.tile_size()
    key, dead_key = O.sort_key(g, after["i1"], after["i2"], after["tag"], T)
    assert np.all(np.diff(key) >= 0)                                          # non-decreasing key
    assert np.all(after["tag"][: int((before["tag"] != 0).sum())] == 1)       # dead at the tail
    ref, _, key_ref = O.sort_reference(g, oracle_from_cols(O, before, -1.0, -1.0, 1), T)
    assert np.array_equal(key, key_ref)


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_sort_into_and_species_without_prev_columns(G, O, W, prec):
    """grpic_sort_into (two column sets, no snapshot) and the optional *_prev columns: the destination is the
    source permuted into key order, the source is untouched, and the fused tile-path step on the destination
    agrees with the oracle; several sort/step rounds swapping the two sets."""
    wl = W.config_magnetosphere(shrink=8)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, prec)
    fdev, fhost = _fields_both(G, wl, prec)
    sp = wl.species[0]
    rng = np.random.default_rng(11)
    perm = rng.permutation(sp.n)
    for k in ("i1", "i2", "dx1", "dx2", "u1", "u2", "u3", "weight", "tag", "phi"):
        setattr(sp, k, getattr(sp, k)[perm])
    sp.tag = sp.tag.copy(); sp.tag[rng.random(sp.n) < 0.05] = 0
    assert sp.n < (1 << 24)
    sp.phi = np.arange(sp.n, dtype=np.float64)                                # unique id (exact in FP32)
    a = G.ParticleSet.from_host(sp, prec).drop_prev()
    b = a.empty_like()
    T = ctx.tile_size()
    before = a.to_numpy()
    ctx.sort_into(a, b)
    src_after, dst = a.to_numpy(), b.to_numpy()
    ids = dst["phi"].astype(np.int64)
    assert np.array_equal(np.sort(ids), np.arange(sp.n))
    for k, v in dst.items():
        if v is not None:
            assert np.array_equal(src_after[k], before[k]), k                 # source untouched
            assert np.array_equal(v, before[k][ids]), k                       # every column moved alike
        else:
            assert k.endswith("_prev")
    key, _ = O.sort_key(g, dst["i1"], dst["i2"], dst["tag"], T)
    _, _, key_ref = O.sort_reference(g, oracle_from_cols(O, before, -1.0, -1.0, 1), T)
    assert np.array_equal(key, key_ref)
    assert ctx.sorted_alive(b) == int((before["tag"] != 0).sum())
    # sort / step rounds, swapping the two sets; every step against the oracle
    cur, other = b, a
    for rnd in range(3):
        for _ in range(2):
            res, c = _one_step_parity(G, O, ctx, g, cur, fdev, fhost, wl.dt, prec, "fused")
        ctx.sort_into(cur, other)
        cur, other = other, cur
        cols = cur.to_numpy()
        key, _ = O.sort_key(g, cols["i1"], cols["i2"], cols["tag"], T)
        assert np.all(np.diff(key) >= 0)
    # the in-place sort takes a species without *_prev columns too
    ctx.sort(cur)
    res, c = _one_step_parity(G, O, ctx, g, cur, fdev, fhost, wl.dt, prec, "fused")
    # refused: a shared column, a partial set of *_prev columns, different optional columns
    bad = cur.empty_like(); bad.cols["u1"] = cur.cols["u1"]
    with pytest.raises(G.GrpicError):
        ctx.sort_into(cur, bad)
    import torch
    part = cur.empty_like(); part.cols["i1_prev"] = torch.zeros_like(part.cols["i1"])
    with pytest.raises(G.GrpicError):
        ctx.sort(part)
    with pytest.raises(G.GrpicError):
        ctx.step(part, fdev, _zeros_J(G, ctx, prec), wl.dt)
    full = G.ParticleSet.from_host(sp, prec)
    with pytest.raises(G.GrpicError):
        ctx.sort_into(cur, full)
    with pytest.raises(G.GrpicError):                                         # the split calls still need them
        ctx.interp_push(cur, fdev, wl.dt)


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_sort_lookahead_gives_a_valid_order(G, O, W, prec):
    """"sort_lookahead" orders by the cell predicted L steps ahead (a heuristic; include/grpic.h): whatever it
    predicts, the result must be a permutation that moves every column alike, alive particles first, and the tile
    path on that order must still agree with the oracle step by step (particles outside their tile's window take
    the global path).  Before any step there is no dt and the order is the plain key order."""
    wl = W.config_magnetosphere(shrink=8)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, prec)
    fdev, fhost = _fields_both(G, wl, prec)
    sp = wl.species[1]
    rng = np.random.default_rng(13)
    sp.tag = sp.tag.copy(); sp.tag[rng.random(sp.n) < 0.05] = 0
    sp.weight = np.arange(1, sp.n + 1, dtype=np.float64)                     # unique id the step never changes
    a = G.ParticleSet.from_host(sp, prec).drop_prev()
    b = a.empty_like()
    T = ctx.tile_size()
    ctx.set_real("sort_lookahead", 5.0)
    ctx.sort_into(a, b)                                                      # no dt yet: present-cell keys
    cols = b.to_numpy()
    key, _ = O.sort_key(g, cols["i1"], cols["i2"], cols["tag"], T)
    assert np.all(np.diff(key) >= 0)
    cur, other = b, a
    for rnd in range(3):
        for _ in range(3):
            _one_step_parity(G, O, ctx, g, cur, fdev, fhost, wl.dt, prec, "fused")
        before = cur.to_numpy()
        ctx.sort_into(cur, other)
        cur, other = other, cur
        after = cur.to_numpy()
        ids = after["weight"].astype(np.int64) - 1
        ids0 = before["weight"].astype(np.int64) - 1
        assert np.array_equal(np.sort(ids), np.arange(sp.n))
        src_of = np.argsort(ids0)[ids]
        for k, v in after.items():
            if v is not None:
                assert np.array_equal(v, before[k][src_of]), k
        n_alive = int((before["tag"] != 0).sum())
        assert ctx.sorted_alive(cur) == n_alive and np.all(after["tag"][:n_alive] != 0) and not after["tag"][n_alive:].any()
        key, _ = O.sort_key(g, after["i1"], after["i2"], after["tag"], T)
        moved = float(np.mean(np.diff(key[:n_alive].astype(np.int64)) < 0))
        assert 0.0 < moved < 0.5                                            # predicted order: near, not equal to, the present one
    with pytest.raises(G.GrpicError):
        ctx.set_real("sort_lookahead", -1.0)


def test_step_host_matches_device_step(G, O, W):
    import torch
    wl = W.config_magnetosphere(shrink=8)
    ctx = _ctx(G, wl.dom, "f32")
    names = ("D1", "D2", "D3", "B1", "B2", "B3")
    fdev = G.grid_tensors(wl.fields, names, "f32")
    fhost = G.grid_tensors(wl.fields, names, "f32", device="cpu", pinned=True)
    sp = wl.species[0]
    pd = G.ParticleSet.from_host(sp, "f32")
    ph = G.ParticleSet.from_host(sp, "f32", device="cpu", pinned=True)
    Jd = _zeros_J(G, ctx, "f32")
    Jh = {k: torch.zeros(ctx.shape, dtype=torch.float32).pin_memory() for k in ("J1", "J2", "J3")}
    ctx.step(pd, fdev, Jd, wl.dt)
    cd = ctx.counters()
    up, down = ctx.step_host(ph, fhost, Jh, wl.dt)
    ch = ctx.counters()
    assert cd == ch
    a, b = pd.to_numpy(), ph.to_numpy()
    for k in a:
        if a[k] is not None:
            assert np.array_equal(a[k], b[k]), k
    for k in Jd:
        assert torch.allclose(Jd[k].cpu(), Jh[k], rtol=0, atol=1e-5 * float(Jd[k].abs().max()))
    assert up > 0 and down > 0
    # the four *_prev columns are optional on the host path: NULL -> nothing comes back for them
    ph2 = G.ParticleSet.from_host(sp, "f32", device="cpu", pinned=True)
    for k in ("i1_prev", "i2_prev"):
        ph2.cols[k].fill_(-7)
    Jh2 = {k: torch.zeros(ctx.shape, dtype=torch.float32).pin_memory() for k in ("J1", "J2", "J3")}
    up2, down2 = ctx.step_host(ph2, fhost, Jh2, wl.dt, with_prev=False)
    c2 = ph2.to_numpy()
    assert down2 < down and up2 == up
    assert np.all(c2["i1_prev"] == -7) and np.all(c2["i2_prev"] == -7)
    for k in ("i1", "i2", "dx1", "dx2", "u1", "u2", "u3", "phi", "tag"):
        assert np.array_equal(a[k], c2[k]), k
    # many chunks with the ramped sizes at both ends of the call, and J_host += on top of what is there
    assert sp.n >= 4 * 8192
    ctx.set_int("host_chunk", 8192)
    ph3 = G.ParticleSet.from_host(sp, "f32", device="cpu", pinned=True)
    up3, down3 = ctx.step_host(ph3, fhost, Jh2, wl.dt)
    c3 = ph3.to_numpy()
    for k in a:
        if a[k] is not None:
            assert np.array_equal(a[k], c3[k]), k
    for k in Jd:
        assert torch.allclose(2 * Jd[k].cpu(), Jh2[k], rtol=0, atol=2e-5 * float(Jd[k].abs().max()))
    assert ctx.counters() == cd
    with pytest.raises(G.GrpicError):
        ctx.set_int("host_chunk", 7)


def test_edge_cases(G, O, W):
    """n = 0; all dead; a particle crossing each axis (reflection); absorption at both radial edges; overstep."""
    import torch
    dom = W.Domain(32, 16, 0.9, 0.9 * W.horizon_radius(0.9), 20.0)
    g = grid_from_domain(O, dom)
    ctx = _ctx(G, dom, "f64")
    fields = W.wald_fields(dom)
    fdev = G.grid_tensors(fields, ("D1", "D2", "D3", "B1", "B2", "B3"), "f64")
    fhost = {k: np.asarray(v, np.float64) for k, v in fields.items()}

    class S:
        pass

    def mk(i1, i2, dx1, dx2, u1, u2, u3, tag=None, q=1.0):
        s = S()
        n = len(i1)
        s.i1, s.i2 = np.array(i1, np.int32), np.array(i2, np.int32)
        s.dx1, s.dx2 = np.array(dx1, float), np.array(dx2, float)
        s.u1, s.u2, s.u3 = np.array(u1, float), np.array(u2, float), np.array(u3, float)
        s.weight = np.ones(n); s.tag = np.ones(n, np.uint8) if tag is None else np.array(tag, np.uint8)
        s.phi = np.zeros(n); s.q_over_m = q; s.charge = q; s.massive = 1
        return s

    # empty
    ps = G.ParticleSet.from_host(mk([], [], [], [], [], [], []), "f64")
    J = _zeros_J(G, ctx, "f64")
    ctx.step(ps, fdev, J, 0.1); ctx.interp_push(ps, fdev, 0.1); ctx.deposit(ps, J); ctx.sort(ps)
    assert ctx.counters() == dict(alive=0, absorbed_in=0, absorbed_out=0, overstep=0)
    assert all(float(v.abs().max()) == 0 for v in J.values())
    # all dead: nothing changes
    s = mk([3, 4], [5, 6], [.1, .2], [.3, .4], [1, 2], [3, 4], [5, 6], tag=[0, 0])
    ps = G.ParticleSet.from_host(s, "f64")
    b = ps.to_numpy()
    ctx.step(ps, fdev, J, 0.1)
    a = ps.to_numpy()
    assert all(np.array_equal(a[k], b[k]) for k in ("i1", "i2", "dx1", "dx2", "u1", "u2", "u3", "phi", "tag"))
    assert all(float(v.abs().max()) == 0 for v in J.values())
    # axis crossings, radial exits
    s = mk(i1=[10, 10, 0, 31, 12], i2=[0, 15, 8, 8, 7], dx1=[.5, .5, .01, .99, .5],
           dx2=[.02, .98, .5, .5, .5],
           u1=[0, 0, -3.0, 40.0, 0.1], u2=[-1.5, 1.5, 0, 0, 0.2], u3=[.05, .05, 1, 1, 0.3])
    for mode in ("split", "fused"):
        ps = G.ParticleSet.from_host(s, "f64")
        res, c = _one_step_parity(G, O, ctx, g, ps, fdev, fhost, 0.2, "f64", mode)
        a = ps.to_numpy()
        assert a["i2"][0] == 0 and a["u2"][0] > 0, "reflected at theta = 0"
        assert a["i2"][1] == 15 and a["u2"][1] < 0, "reflected at theta = pi"
        assert a["tag"][2] == 0 and a["i1"][2] < 0 and c["absorbed_in"] == 1
        assert a["tag"][3] == 0 and a["i1"][3] >= 32 and c["absorbed_out"] == 1
        assert c["overstep"] == 0 and c["alive"] == 3
    # overstep: a fast particle and a time step large enough to cross more than one cell in theta
    s = mk(i1=[6, 12], i2=[8, 7], dx1=[.5, .5], dx2=[.5, .5], u1=[0.0, 0.1], u2=[60.0, 0.02], u3=[0.2, 0.3])
    for mode in ("split", "fused"):
        ps = G.ParticleSet.from_host(s, "f64")
        Jt = _zeros_J(G, ctx, "f64")
        res, c = _one_step_parity(G, O, ctx, g, ps, fdev, fhost, 1.5, "f64", mode)
        assert c["overstep"] == 1 and abs(int(ps.cols["i2"][0]) - 8) > 1


def test_abi_errors(G):
    import ctypes as C
    ctx = G.Context(16, 16, 0.5, 1.5, 10.0, precision="f32")
    with pytest.raises(G.GrpicError):
        ctx.set_int("n_iter", 0)
    with pytest.raises(G.GrpicError):
        ctx.set_int("nope", 1)
    with pytest.raises(G.GrpicError):
        ctx.set_real("small_angle", -1.0)
    # deposit before any push -> ESTATE; charged species without fields -> EINVAL
    import torch
    z = lambda dt: torch.zeros(4, dtype=dt, device="cuda")
    cols = {k: z(torch.int32) for k in ("i1", "i2", "i1_prev", "i2_prev")}
    cols.update({k: z(torch.float32) for k in ("dx1", "dx2", "u1", "u2", "u3", "phi", "dx1_prev", "dx2_prev", "weight")})
    cols["tag"] = torch.ones(4, dtype=torch.uint8, device="cuda")
    ps = G.ParticleSet(cols, 1.0, 1.0, 1)
    J = {k: torch.zeros(ctx.shape, device="cuda") for k in ("J1", "J2", "J3")}
    with pytest.raises(G.GrpicError) as e:
        ctx.deposit(ps, J)
    assert e.value.code == G.GRPIC_ESTATE
    with pytest.raises(G.GrpicError) as e:
        ctx.interp_push(ps, None, 0.1)
    assert e.value.code == G.GRPIC_EINVAL
    with pytest.raises(G.GrpicError) as e:
        ctx.step(ps, None, J, -1.0)
    assert e.value.code == G.GRPIC_EINVAL


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_early_exit_is_bit_identical_to_all_iterations(G, W, prec):
    """A fixed-point loop that stops when an iterate repeats bit for bit returns exactly what n_iter
    iterations return (the map is deterministic).  Proven by running both on the same inputs."""
    import torch
    wl = W.config_large(shrink=16)
    names = ("D1", "D2", "D3", "B1", "B2", "B3")
    fdev = G.grid_tensors(wl.fields, names, prec)
    outs = []
    for ee in (1, 0):
        ctx = _ctx(G, wl.dom, prec)
        ctx.set_int("early_exit", ee)
        ps = G.ParticleSet.from_host(wl.species[1], prec)
        J = _zeros_J(G, ctx, prec)
        for _ in range(3):
            ctx.step(ps, fdev, J, wl.dt)
        outs.append((ps.to_numpy(), _J_np(J)))
    a, b = outs
    for k in a[0]:
        if a[0][k] is not None:
            assert np.array_equal(a[0][k], b[0][k]), k
    for k in a[1]:
        assert np.allclose(a[1][k], b[1][k], rtol=0, atol=TOL[prec]["J"] * np.abs(b[1][k]).max())


# ------------------------------------------------------------------------------------------------
# field-solver half: auxiliary fields, Faraday, Ampere against the oracle
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("kw", [dict(), dict(r0=0.5, h0=0.3), dict(linear_r=1), dict(linear_r=1, mass=0.0)])
def test_field_solver_kernels(G, O, W, prec, kw):
    """grpic_aux_fields / grpic_faraday / grpic_ampere element by element against the oracle on random fields and
    currents (several thread blocks per row and a ragged tail in theta), on four maps; then div B and the Wald
    stationarity are re-checked on the GPU output of the default map."""
    import torch
    mass = kw.get("mass", 1.0)
    a = 0.9 if mass else 0.0
    n1, n2, ng = 70, 150, 2
    g = O.Grid(n1, n2, a, 1.3, 18.0, ng=ng, **kw)
    ctx = G.Context(n1, n2, a, g.r_min, g.r_max, nghost=ng, precision=prec, r0=kw.get("r0"), h0=kw.get("h0"),
                    r_map=0 if kw.get("linear_r") else 1, mass=kw.get("mass"))
    rng = np.random.default_rng(11)
    rt = np.float32 if prec == "f32" else np.float64
    names = ("D1", "D2", "D3", "B1", "B2", "B3")
    f = {k: rng.normal(size=g.shape).astype(rt).astype(np.float64) for k in names}
    J = {k: rng.normal(size=g.shape).astype(rt).astype(np.float64) for k in ("J1", "J2", "J3")}
    dev = lambda d: {k: torch.from_numpy(v.astype(rt)).cuda() for k, v in d.items()}
    tol = 2e-6 if prec == "f32" else 1e-12

    def close(got, ref, what):
        for k in ref:
            r = ref[k]; x = got[k].cpu().numpy().astype(np.float64)
            assert np.abs(x - r).max() <= tol * max(1.0, np.abs(r).max()), (what, k, np.abs(x - r).max(), np.abs(r).max())

    fd = dev(f)
    Ed = {k: torch.zeros(g.shape, dtype=G.torch_real(prec), device="cuda") for k in ("E1", "E2", "E3")}
    Hd = {k: torch.zeros(g.shape, dtype=G.torch_real(prec), device="cuda") for k in ("H1", "H2", "H3")}
    ctx.aux_fields(fd, Ed, Hd)
    aux = O.aux_fields(g, f)
    close({**Ed, **Hd}, aux, "aux")
    # Faraday / Ampere from the oracle's aux fields rounded to the build's precision (same inputs on both sides)
    auxr = {k: v.astype(rt).astype(np.float64) for k, v in aux.items()}
    dt = 0.013
    Bo = {k: f[k].copy() for k in ("B1", "B2", "B3")}; Do = {k: f[k].copy() for k in ("D1", "D2", "D3")}
    O.faraday(g, Bo, auxr, dt); O.ampere(g, Do, auxr, J, dt)
    Bd = {k: fd[k].clone() for k in ("B1", "B2", "B3")}; Dd = {k: fd[k].clone() for k in ("D1", "D2", "D3")}
    ad = dev(auxr)
    ctx.faraday(Bd, ad, dt); ctx.ampere(Dd, ad, dev(J), dt)
    close(Bd, Bo, "faraday"); close(Dd, Do, "ampere")
    # untouched entries: ghost columns beyond the axes and the outer two ghost rows
    assert torch.equal(Bd["B1"][:2], fd["B1"][:2]) and torch.equal(Dd["D2"][:, :ng], fd["D2"][:, :ng])
    assert torch.equal(Bd["B2"][:, ng], fd["B2"][:, ng])                  # B^2 on the axis is not evolved
    Dd2 = {k: fd[k].clone() for k in ("D1", "D2", "D3")}
    ctx.ampere(Dd2, ad, None, dt)                                         # J = NULL: vacuum
    Do2 = {k: f[k].copy() for k in ("D1", "D2", "D3")}
    O.ampere(g, Do2, auxr, None, dt)
    close(Dd2, Do2, "ampere vacuum")


def test_field_solver_wald_stationary_on_gpu(G, O, W):
    """The stationary Wald solution through the GPU kernels (FP64, 256x128, r >= 2.6): residual of one Faraday + Ampere
    update below 1e-4 of the field everywhere, axis rows included (same bound as the oracle pin)."""
    import torch
    a = 0.9
    dom = W.Domain(256, 128, a, 2.6, 20.0)
    ctx = G.Context(dom.n1, dom.n2, a, dom.r_min, dom.r_max, nghost=dom.ng, precision="f64")
    f = W.wald_fields(dom, 1.0)
    fd = {k: torch.from_numpy(np.ascontiguousarray(v)).cuda() for k, v in f.items()}
    E = {k: torch.zeros(dom.shape, dtype=torch.float64, device="cuda") for k in ("E1", "E2", "E3")}
    H = {k: torch.zeros(dom.shape, dtype=torch.float64, device="cuda") for k in ("H1", "H2", "H3")}
    ctx.aux_fields(fd, E, H)
    B = {k: fd[k].clone() for k in ("B1", "B2", "B3")}; D = {k: fd[k].clone() for k in ("D1", "D2", "D3")}
    ctx.faraday(B, E, 1.0); ctx.ampere(D, H, None, 1.0)
    G_ = dom.ng
    sl = (slice(G_ + 2, G_ + dom.n1 - 2), slice(G_, G_ + dom.n2 + 1))
    for k, new in list(B.items()) + list(D.items()):
        r = float((new - fd[k])[sl].abs().max() / fd[k][sl].abs().max())
        assert r < 1e-4, (k, r)


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_full_pic_cycle_against_the_oracle(G, O, W, prec):
    """Four complete timesteps of Sec. 3.4 on the GPU and in the oracle, each side with its own state:
    fields_prepare (Eq. 46-48) -> push with (n)B, (n)D -> deposit (n+1/2)J -> fields_advance (Eq. 51-56).
    Tiny magnetosphere (config 1 shape, Wald field, e+- pairs); tolerances as for the per-step parity but accumulated
    over the four steps (x2 per step for f32)."""
    import torch
    wl = W.config_tiny(shrink=2)
    dom = wl.dom
    g = grid_from_domain(O, dom)
    ctx = _ctx(G, dom, prec)
    rt = np.float32 if prec == "f32" else np.float64
    kb, kd, kj = ("B1", "B2", "B3"), ("D1", "D2", "D3"), ("J1", "J2", "J3")
    f = {k: np.asarray(v, rt).astype(np.float64) for k, v in wl.fields.items()}
    cp = lambda ks: {k: f[k].copy() for k in ks}
    so = dict(B_prev=cp(kb), B=cp(kb), D_prev=cp(kd), D=cp(kd))
    td = lambda d: {k: torch.from_numpy(v.astype(rt)).cuda() for k, v in d.items()}
    sg = {k: td(v) for k, v in so.items()}
    zeros = lambda ks: {k: torch.zeros(ctx.shape, dtype=G.torch_real(prec), device="cuda") for k in ks}
    Bn_g = zeros(kb)
    sets = [G.ParticleSet.from_host(sp, prec) for sp in wl.species]
    ops = [oracle_from_cols(O, ps.to_numpy(), ps.q_over_m, ps.charge, ps.massive) for ps in sets]
    Jprev_g, Jprev_o = zeros(kj), {k: np.zeros(g.shape) for k in kj}
    dt = wl.dt
    for step in range(4):
        ctx.fields_prepare(sg, Bn_g, dt)
        Bn_o = O.fields_prepare(g, so, dt)
        for k in kb:                                   # (n)B itself, ghost columns beyond the axes included
            d = np.abs(Bn_g[k].cpu().numpy().astype(np.float64) - Bn_o[k]).max() / np.abs(Bn_o[k]).max()
            assert d < (1e-5 if prec == "f32" else 1e-12), (step, k, d)
        Jg, Jo = zeros(kj), {k: np.zeros(g.shape) for k in kj}
        for ps, op in zip(sets, ops):
            ctx.step(ps, {**sg["D"], **Bn_g}, Jg, dt)
            O.push(g, op, {**so["D"], **Bn_o}, dt)
            O.deposit(g, op, dt, Jo)
        ctx.fields_advance(sg, Bn_g, Jprev_g, Jg, dt)
        so = O.fields_advance(g, so, Bn_o, Jprev_o, Jo, dt)
        Jprev_g, Jprev_o = Jg, Jo
    tol = (1e-4 if prec == "f32" else 1e-10)
    for name in ("B_prev", "B", "D_prev", "D"):
        for k, ref in so[name].items():
            got = sg[name][k].cpu().numpy().astype(np.float64)
            err = np.abs(got - ref).max() / max(1e-300, np.abs(ref).max())
            assert err < tol, (name, k, err)
    for ps, op in zip(sets, ops):
        c = ps.to_numpy()
        same = (c["i1"] == op.i1) & (c["i2"] == op.i2) & (c["tag"] == op.tag)
        assert same.mean() > (0.999 if prec == "f32" else 1.0 - 1e-9)
        ex = np.abs((c["i1"] + c["dx1"].astype(np.float64)) - (op.i1 + op.dx1))[c["tag"] != 0].max()
        assert ex < (1e-4 if prec == "f32" else 1e-10), ex


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("ng", [1, 2, 3])
def test_field_bc(G, O, W, prec, ng):
    """grpic_field_bc against the oracle on random arrays: bit-exact (copies and sign flips only)."""
    import torch
    g = O.Grid(20, 150, 0.9, 1.3, 15.0, ng=ng)
    ctx = G.Context(g.n1, g.n2, 0.9, g.r_min, g.r_max, nghost=ng, precision=prec)
    rng = np.random.default_rng(ng)
    rt = np.float32 if prec == "f32" else np.float64
    f = {k: rng.normal(size=g.shape).astype(rt).astype(np.float64) for k in ("D1", "D2", "D3", "B1", "B2", "B3")}
    for n_const in (-1, 0, 3):
        fd = {k: torch.from_numpy(v.astype(rt)).cuda() for k, v in f.items()}
        ctx.field_bc(fd, n_const)
        ref = O.field_bc(g, {k: v.copy() for k, v in f.items()}, n_const)
        for k in f:
            assert np.array_equal(fd[k].cpu().numpy().astype(np.float64), ref[k]), (k, n_const)


@pytest.mark.parametrize("prec", ["f32", "f64"])
@pytest.mark.parametrize("kw", [dict(), dict(r_map=0), dict(r0=0.4)], ids=["log", "linear", "offset"])
def test_field_match_absorbing_layer(G, O, W, prec, kw):
    """grpic_field_match against the oracle (reading R-F6): rows at r <= r_abs bit-unchanged, the layer rows to
    rounding of the weight (tanh in double on both sides), rows beyond r_max = target bit for bit; three maps,
    r_abs inside a cell, at the inner edge (whole grid is layer) and refused outside [r_min, r_max)."""
    import torch
    okw = dict(linear_r=1) if kw.get("r_map") == 0 else dict(kw)
    g = O.Grid(37, 21, 0.9, 1.3, 15.0, ng=3, **okw)
    ctx = G.Context(g.n1, g.n2, 0.9, g.r_min, g.r_max, nghost=3, precision=prec, **kw)
    rng = np.random.default_rng(5)
    rt = np.float32 if prec == "f32" else np.float64
    keys = ("D1", "D2", "D3", "B1", "B2", "B3")
    f = {k: rng.normal(size=g.shape).astype(rt).astype(np.float64) for k in keys}
    tg = {k: rng.normal(size=g.shape).astype(rt).astype(np.float64) for k in keys}
    tol = 2e-7 if prec == "f32" else 1e-14
    for r_abs in (11.3, g.r_min + 1e-9, 14.99):
        fd = {k: torch.from_numpy(v.astype(rt)).cuda() for k, v in f.items()}
        td = {k: torch.from_numpy(v.astype(rt)).cuda() for k, v in tg.items()}
        ctx.field_match(fd, td, r_abs)
        ref = O.field_match(g, {k: v.copy() for k, v in f.items()}, tg, r_abs)
        for k in keys:
            got = fd[k].cpu().numpy().astype(np.float64)
            off = 0.5 if k in ("D1", "B2", "B3") else 0.0
            r = O.radius(g, np.arange(-g.ng, g.n1 + g.ng) + off)
            assert np.array_equal(got[r <= r_abs], f[k][r <= r_abs]), (k, r_abs)
            assert np.array_equal(got[r >= g.r_max * (1 + 1e-12)], tg[k][r >= g.r_max * (1 + 1e-12)]), (k, r_abs)
            # r(x1) of the two sides agrees to a few ulp of r_max (two exponentials); the weight turns that into
            # 4 / (r_max - r_abs) per unit of r, so a thin layer is conditioned by r_max / (r_max - r_abs)
            bound = tol * 4.0 * max(1.0, g.r_max / (g.r_max - r_abs))
            assert np.abs(got - ref[k]).max() <= bound, (k, r_abs, np.abs(got - ref[k]).max())
            assert np.array_equal(td[k].cpu().numpy().astype(np.float64), tg[k])
    for bad in (g.r_max, 0.5 * g.r_min, float("nan")):
        with pytest.raises(G.GrpicError):
            ctx.field_match(fd, td, bad)


def test_vacuum_loop_with_absorbing_layer_follows_the_oracle(G, O, W):
    """Field side of the loop with every boundary condition on the GPU (prepare, advance, axis reflection, absorbing
    layer) against the same sequence in the oracle: flat space (App. A.1), a toroidal pulse that runs into the layer
    and is absorbed; FP64, every 50th step compared, and the pulse is gone at the end on both sides."""
    import torch
    g = O.Grid(96, 8, 0.0, 2.0, 8.0, linear_r=1, mass=0.0)
    ctx = G.Context(g.n1, g.n2, 0.0, g.r_min, g.r_max, nghost=g.ng, precision="f64", r_map=0, mass=0.0)
    keys, kb, kd = ("D1", "D2", "D3", "B1", "B2", "B3"), ("B1", "B2", "B3"), ("D1", "D2", "D3")
    f = {k: np.zeros(g.shape) for k in keys}
    r = O.radius(g, np.arange(-g.ng, g.n1 + g.ng) + 0.5)
    f["B3"][:] = (np.exp(-((r - 5.5) / 0.4) ** 2) / r)[:, None]
    amp0 = np.abs(f["B3"]).max()
    cp = lambda ks: {k: f[k].copy() for k in ks}
    so = dict(B_prev=cp(kb), B=cp(kb), D_prev=cp(kd), D=cp(kd))
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    sg = {n: {k: t(v) for k, v in d.items()} for n, d in so.items()}
    zero = {k: torch.zeros(ctx.shape, dtype=torch.float64, device="cuda") for k in keys}
    zero_o = {k: np.zeros(g.shape) for k in keys}
    Bn = {k: torch.zeros(ctx.shape, dtype=torch.float64, device="cuda") for k in kb}
    dt, r_abs = 0.5 * (g.r_max - g.r_min) / g.n1, 6.5
    worst = 0.0
    n_steps = int(14.0 / dt)
    for step in range(1, n_steps + 1):
        ctx.fields_prepare(sg, Bn, dt)
        ctx.fields_advance(sg, Bn, None, None, dt)
        cur = {**sg["D"], **sg["B"]}
        ctx.field_bc(cur)
        ctx.field_match(cur, zero, r_abs)
        Bo = O.fields_prepare(g, so, dt)
        so = O.fields_advance(g, so, Bo, None, None, dt)
        cur_o = {**so["D"], **so["B"]}
        O.field_bc(g, cur_o)
        O.field_match(g, cur_o, zero_o, r_abs)
        if step % 50 == 0 or step == n_steps:
            for k in keys:
                worst = max(worst, float(np.abs(cur[k].cpu().numpy() - cur_o[k]).max()) / amp0)
    assert worst < 1e-11, worst
    left = float(sg["B"]["B3"].abs().max()) / amp0
    assert left < 0.03 and np.abs(so["B"]["B3"]).max() / amp0 < 0.03, left


def _closed_loop_gauss(G, O, W, wl, prec, steps, bench_cfg, tol):
    """`steps` complete timesteps (prepare, fused step, advance [, field BCs, re-sort every 10 steps]); returns the
    largest drift of G = d_i(sqrt(h) D^i) - k_J rho~ at the interior nodes in units of k_J x mean charge per node."""
    import torch
    dom = wl.dom
    g = grid_from_domain(O, dom)
    ctx = _ctx(G, dom, prec)
    rt = G.torch_real(prec)
    kb, kd, kj = ("B1", "B2", "B3"), ("D1", "D2", "D3"), ("J1", "J2", "J3")
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).to(rt).cuda()
    st = dict(B_prev={k: t(wl.fields[k]) for k in kb}, B={k: t(wl.fields[k]) for k in kb},
              D_prev={k: t(wl.fields[k]) for k in kd}, D={k: t(wl.fields[k]) for k in kd})
    zeros = lambda ks: {k: torch.zeros(ctx.shape, dtype=rt, device="cuda") for k in ks}
    Bn, Jprev = zeros(kb), zeros(kj)
    sets = [G.ParticleSet.from_host(sp, prec) for sp in wl.species]
    spare = None
    if bench_cfg:                                       # as bench.py: no *_prev columns, two column sets, look-ahead sort
        sets = [ps.drop_prev() for ps in sets]
        spare = [ps.empty_like() for ps in sets]
        ctx.set_real("sort_lookahead", 5.0)
    Gn, ld = dom.ng, ctx.shape[1]
    t64 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64)).cuda()
    ii = np.arange(-Gn, dom.n1 + Gn, dtype=np.float64); jj = np.clip(np.arange(-Gn, dom.n2 + Gn, dtype=np.float64), 0, dom.n2)
    s1 = t64(O.sqrt_h(g, *[v.ravel() for v in np.meshgrid(ii + 0.5, jj, indexing="ij")]).reshape(ctx.shape))
    s2 = t64(O.sqrt_h(g, *[v.ravel() for v in np.meshgrid(ii, np.clip(jj + 0.5, 0, dom.n2), indexing="ij")]).reshape(ctx.shape))
    kJ = 4 * np.pi

    def gauss():
        f1, f2 = s1 * st["D"]["D1"].double(), s2 * st["D"]["D2"].double()
        div = (f1[1:, 1:] - f1[:-1, 1:]) + (f2[1:, 1:] - f2[1:, :-1])
        rho = torch.zeros(ctx.shape[0] * ld, dtype=torch.float64, device="cuda")
        for ps in sets:
            c = ps.cols
            q = torch.where(c["tag"] != 0, c["weight"].double() * ps.charge, torch.zeros_like(c["weight"], dtype=torch.float64))
            base = (c["i1"].long() + Gn) * ld + (c["i2"].long() + Gn)
            x, y = c["dx1"].double(), c["dx2"].double()
            for da, wa in ((0, 1 - x), (1, x)):
                for db, wb in ((0, 1 - y), (1, y)):
                    rho.index_add_(0, base + da * ld + db, q * wa * wb)
        return (div - kJ * rho.view(ctx.shape)[1:, 1:])[Gn + 2:Gn + dom.n1 - 3, Gn:Gn + dom.n2 - 2]
    n0 = sum(int(ps.cols["tag"].sum()) for ps in sets)
    scale = float(kJ * n0 / (dom.n1 * dom.n2))          # k_J * mean charge magnitude per node
    g0 = None
    absorbed, worst = 0, 0.0
    for step in range(steps):
        if step % 10 == 0:
            for i, ps in enumerate(sets):
                if bench_cfg:
                    ctx.sort_into(ps, spare[i]); sets[i], spare[i] = spare[i], ps
                else:
                    ctx.sort(ps)
        if g0 is None:
            g0 = gauss()
        ctx.fields_prepare(st, Bn, wl.dt)
        J = zeros(kj)
        for ps in sets:
            ctx.step(ps, {**st["D"], **Bn}, J, wl.dt)
            c = ctx.counters()
            absorbed += c["absorbed_in"] + c["absorbed_out"]
            assert c["overstep"] == 0
        ctx.fields_advance(st, Bn, Jprev, J, wl.dt)
        if bench_cfg:
            ctx.field_bc({**st["D"], **st["B"]})
        Jprev = J
        if step % 10 == 9 or step == steps - 1 or steps <= 30:
            drift = float((gauss() - g0).abs().max()) / scale
            worst = max(worst, drift)
            assert drift < tol * (step + 1), (step, drift)
    ctx.close()
    return worst, absorbed / n0


def test_gauss_law_is_kept_by_the_closed_loop_on_the_gpu(G, O, W):
    """"Perfect charge conservation" through the whole GPU loop in FP64: G = d_i(sqrt(h) D^i) - k_J rho~ at
    the nodes is the same after every timestep, because the deposit satisfies the discrete continuity equation
    (Eq. 32-34) and Ampere's curl terms cancel in the divergence.  30 complete timesteps of a tiny magnetosphere
    (prepare, fused tiled step after a sort, advance); rho~ by its definition (linear shape on nodes) in torch.
    Nodes of the first three rows are left out: particles absorbed at i1 < 0 vanish there without a current."""
    drift, gone = _closed_loop_gauss(G, O, W, W.config_tiny(shrink=2), "f64", 30, False, 1e-11)
    assert gone > 0          # the run did exercise absorption (outside the checked nodes)
    print("Gauss-law drift after 30 steps:", drift, "absorbed fraction", gone)


@pytest.mark.parametrize("prec,tol", [("f64", 1e-13), ("f32", 3e-7)])
def test_closed_loop_soak_in_the_bench_configuration(G, O, W, prec, tol):
    """400 complete timesteps of config 1 at full size (128 x 64, 131 k particles) in the configuration bench.py runs:
    species without *_prev columns, grpic_sort_into between two column sets every 10 steps with the look-ahead key,
    the fused step (k_step_lanes for the dense tiles), grpic_field_bc after every step.  The Gauss-law residual must
    not drift: per step at most `tol` of k_J x the mean charge per node (rounding of the deposit and of Ampere only),
    while a large part of the plasma falls through the horizon."""
    drift, gone = _closed_loop_gauss(G, O, W, W.config_tiny(), prec, 400, True, tol)
    print(f"soak {prec}: 400 steps, largest Gauss-law drift {drift:.2e} of k_J x charge per node, {100 * gone:.0f} % absorbed")
    assert gone > 0.05 and drift < (1e-13 if prec == "f64" else 5e-6)


@pytest.mark.parametrize("prec,dense_min,look", [("f32", 2048, 0.0), ("f32", 4, 3.0), ("f64", 4, 3.0), ("f64", 1024, 0.0)])
def test_lanes_kernel_dense_and_degenerate_items(G, O, W, prec, dense_min, look):
    """k_step_lanes (one particle run per lane, lane-private J windows, 128-bit column blocks) against the oracle, in
    both precisions (FP64 switched on explicitly): dense_min = 4 sends EVERY work item through it - items of a handful
    of particles, runs of one partial block, items that begin and end inside a 16-byte block - and six steps without a
    re-sort let the particles drift out of the windows (the strays take the L2 path).  Species without *_prev columns,
    two column sets, look-ahead sort as in bench.py; then a species truncated to its alive count after the sort."""
    wl = W.config_large(shrink=16)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, prec)
    ctx.set_int("lanes_path", 1)
    ctx.set_int("dense_min", dense_min)
    fdev, fhost = _fields_both(G, wl, prec)
    for sp in wl.species:
        rng = np.random.default_rng(3)
        sp.tag = sp.tag.copy(); sp.tag[rng.random(sp.n) < 0.03] = 0          # dead slots: ragged item boundaries
        src = G.ParticleSet.from_host(sp, prec).drop_prev()
        ps = src.empty_like()
        ctx.sort_into(src, ps)
        ctx.set_real("sort_lookahead", look)
        for step in range(6):
            if step == 2:
                ctx.sort_into(ps, src)                # now with a dt: the look-ahead key
                ps, src = src, ps
            res, c = _one_step_parity(G, O, ctx, g, ps, fdev, fhost, wl.dt, prec, "fused")
        print("lanes", prec, dense_min, look, res, c)
        # compaction: drop the dead tail (p->n < n at the sort): the table still covers [0, n_alive)
        ctx.sort_into(ps, src)
        n_alive = ctx.sorted_alive(src)
        cut = G.ParticleSet({k: (None if v is None else v[:n_alive]) for k, v in src.cols.items()},
                            src.q_over_m, src.charge, src.massive)
        res, c = _one_step_parity(G, O, ctx, g, cut, fdev, fhost, wl.dt, prec, "fused")
        assert c["alive"] + c["absorbed_in"] + c["absorbed_out"] == n_alive


def test_forget_drops_the_tile_table(G, O, W):
    """grpic_forget: the table of a sorted species is gone (grpic_sorted_alive says so), and the species then steps
    through the direct kernel with the same results."""
    wl = W.config_magnetosphere(shrink=16)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, "f32")
    fdev, fhost = _fields_both(G, wl, "f32")
    ps = G.ParticleSet.from_host(wl.species[0], "f32")
    ctx.sort(ps)
    assert ctx.sorted_alive(ps) == int((wl.species[0].tag != 0).sum())
    _one_step_parity(G, O, ctx, g, ps, fdev, fhost, wl.dt, "f32", "fused")
    ctx.forget(ps)
    with pytest.raises(G.GrpicError):
        ctx.sorted_alive(ps)
    _one_step_parity(G, O, ctx, g, ps, fdev, fhost, wl.dt, "f32", "fused")
    ctx.forget(ps)                                     # nothing to forget: not an error


def test_lanes_kernel_declines_unaligned_columns(G, O, W):
    """Columns that are only 4-byte aligned (views one element into a buffer): grpic_step must not take the 128-bit
    block path (include/grpic.h asks for 16-byte alignment; the library checks instead of trusting) and still be right."""
    import torch
    wl = W.config_magnetosphere(shrink=16)
    g = grid_from_domain(O, wl.dom)
    ctx = _ctx(G, wl.dom, "f32")
    fdev, fhost = _fields_both(G, wl, "f32")
    base = G.ParticleSet.from_host(wl.species[0], "f32").drop_prev()
    cols = {}
    for k, v in base.cols.items():
        if v is None:
            cols[k] = None
            continue
        buf = torch.empty(v.numel() + 8, dtype=v.dtype, device="cuda")
        buf[1:1 + v.numel()] = v
        cols[k] = buf[1:1 + v.numel()]
    ps = G.ParticleSet(cols, base.q_over_m, base.charge, base.massive)
    assert ps.cols["dx1"].data_ptr() % 16 != 0
    ctx.sort(ps)
    for step in range(2):
        _one_step_parity(G, O, ctx, g, ps, fdev, fhost, wl.dt, "f32", "fused")


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_injection_and_compaction_after_a_sort(G, O, W, prec):
    """after grpic_sort the alive particles sit in [0, n_alive) (grpic_sorted_alive).  Particles written
    into dead slots (tag 0 -> 1) and particles appended beyond the sorted range must be pushed and deposited by the
    next grpic_step although the tile table does not know them; truncating the set to n_alive drops only dead ones."""
    import torch
    wl = W.config_large(shrink=32)
    dom = wl.dom
    g = grid_from_domain(O, dom)
    ctx = _ctx(G, dom, prec)
    fdev, fhost = _fields_both(G, wl, prec)
    sp = wl.species[0]
    rng = np.random.default_rng(8)
    sp.tag = sp.tag.copy(); sp.tag[rng.random(sp.n) < 0.2] = 0
    ps = G.ParticleSet.from_host(sp, prec)
    ctx.sort(ps)
    n_alive = ctx.sorted_alive(ps)
    assert n_alive == int(sp.tag.sum()) and bool((ps.cols["tag"][:n_alive] == 1).all()) and bool((ps.cols["tag"][n_alive:] == 0).all())
    # revive every second dead slot with a fresh particle, and append 1000 more beyond the old length
    n_old = ps.n
    idx = torch.arange(n_alive, n_old, 2, device="cuda")
    extra = 1000
    cols = {}
    for k, v in ps.cols.items():
        cols[k] = torch.cat([v, v[:extra].clone()])
    rt = G.torch_real(prec)
    gen = torch.Generator(device="cuda"); gen.manual_seed(5)
    newi = torch.cat([idx, torch.arange(n_old, n_old + extra, device="cuda")])
    m = newi.numel()
    cols["i1"][newi] = torch.randint(4, dom.n1 - 4, (m,), device="cuda", generator=gen, dtype=torch.int32)
    cols["i2"][newi] = torch.randint(1, dom.n2 - 1, (m,), device="cuda", generator=gen, dtype=torch.int32)
    for k in ("dx1", "dx2"):
        cols[k][newi] = torch.rand(m, device="cuda", generator=gen, dtype=torch.float64).to(rt) * 0.999
    for k in ("u1", "u2", "u3"):
        cols[k][newi] = (torch.rand(m, device="cuda", generator=gen, dtype=torch.float64).to(rt) - 0.5) * 0.02
    cols["weight"][newi] = 1.0
    cols["tag"][newi] = 1
    # the sort table is keyed by the address of the i1 column: keep the original storage for the sorted part
    ps2 = G.ParticleSet(cols, ps.q_over_m, ps.charge, ps.massive)
    ctx.sort(ps2)                                   # a table for the new storage ...
    n2_alive = ctx.sorted_alive(ps2)
    assert n2_alive == n_alive + m
    # ... then make it stale again: kill some, revive others, so that the direct path must serve slots >= n_alive
    cols["tag"][n2_alive - 500:n2_alive] = 0
    dead = torch.arange(n2_alive, ps2.n, device="cuda")[:300]
    cols["tag"][dead] = 1
    cols["i1"][dead] = 10; cols["i2"][dead] = 5
    res, c = _one_step_parity(G, O, ctx, g, ps2, fdev, fhost, wl.dt, prec, "fused")
    assert c["alive"] + c["absorbed_in"] + c["absorbed_out"] == n2_alive - 500 + 300


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_filter_current(G, O, W, prec):
    """grpic_filter_current against the oracle (1 and 3 passes) on random currents; ghost columns untouched."""
    import torch
    g = O.Grid(37, 150, 0.9, 1.3, 15.0, ng=2)
    ctx = G.Context(g.n1, g.n2, 0.9, g.r_min, g.r_max, nghost=2, precision=prec)
    rng = np.random.default_rng(4)
    rt = np.float32 if prec == "f32" else np.float64
    J = {k: rng.normal(size=g.shape).astype(rt).astype(np.float64) for k in ("J1", "J2", "J3")}
    for n in (1, 3):
        Jd = {k: torch.from_numpy(v.astype(rt)).cuda() for k, v in J.items()}
        ctx.filter_current(Jd, n)
        ref = O.filter_current(g, {k: v.copy() for k, v in J.items()}, n)
        for k in J:
            got = Jd[k].cpu().numpy().astype(np.float64)
            assert np.abs(got - ref[k]).max() <= (2e-6 if prec == "f32" else 1e-14), (k, n)
            assert np.array_equal(got[:, :2], J[k][:, :2])
