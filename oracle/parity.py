"""Parity harness shared by tests/, __graft_entry__.smoke() and bench.py's oracle legs - TEST INFRASTRUCTURE, part of
oracle/ (the product path never imports it).  Host-side bookkeeping only: conversion of seeded workload columns into
oracle particles and the comparison rules of DESIGN.md section 3.  No step of the method is computed here."""
import numpy as np

def grid_from_domain(O, dom, n_iter=10):
    return O.Grid(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, ng=dom.ng, n_iter=n_iter)


def oracle_particles(O, sp, dtype=np.float64):
    """workloads.Species -> oracle Particles, values rounded through `dtype` first."""
    r = lambda x: np.asarray(x, dtype).astype(np.float64)
    return O.Particles(i1=sp.i1, i2=sp.i2, dx1=r(sp.dx1), dx2=r(sp.dx2), u1=r(sp.u1), u2=r(sp.u2), u3=r(sp.u3),
                       weight=r(sp.weight), tag=sp.tag, phi=None if sp.phi is None else r(sp.phi),
                       q_over_m=sp.q_over_m, charge=sp.charge, massive=sp.massive)


# --------------------------------------------------------------------------------------------
# GPU-vs-oracle parity helpers (north_star tolerances made operational)
# --------------------------------------------------------------------------------------------
TOL = {"f64": dict(x=1e-12, u=1e-12, J=1e-10), "f32": dict(x=1e-5, u=1e-5, J=1e-5)}
AXIS_STATS = []      # one row per compare_particles call: (precision, particles, n with kappa > 1, their max raw error, max kappa)


def oracle_from_cols(O, cols, q_over_m, charge, massive):
    """numpy column dict (ParticleSet.to_numpy()) -> oracle Particles (FP64 copies of the same values)."""
    f = lambda k: np.asarray(cols[k], np.float64)
    if cols.get("i1_prev") is None:          # species kept without *_prev columns (fused step only)
        n = len(cols["i1"])
        cols = dict(cols, i1_prev=np.zeros(n, np.int32), i2_prev=np.zeros(n, np.int32),
                    dx1_prev=np.zeros(n), dx2_prev=np.zeros(n))
    return O.Particles(i1=cols["i1"], i2=cols["i2"], dx1=f("dx1"), dx2=f("dx2"), u1=f("u1"), u2=f("u2"), u3=f("u3"),
                       weight=f("weight"), tag=cols["tag"], phi=None if cols.get("phi") is None else f("phi"),
                       i1_prev=cols["i1_prev"], i2_prev=cols["i2_prev"], dx1_prev=f("dx1_prev"),
                       dx2_prev=f("dx2_prev"), q_over_m=q_over_m, charge=charge, massive=massive)


def compare_particles(op, gc, prec, was_alive, n1, n2, check_prev=True, diag=None):
    """op: oracle Particles after the step; gc: GPU columns (numpy) after the same step from the same
    inputs; was_alive: tag before the step.  Returns a dict of maxima; raises AssertionError on a miss.

    Rules: tag exact; for particles alive before the step the position
    x = (i1 + dx1, i2 + dx2, phi) obeys ||dx||_inf <= tol*kappa*max(1, ||x||_inf) (kappa = 1 except for
    particles whose midpoint grazes the polar axis, see below) and the momentum
    ||du||_inf <= tol*max(1, ||u||_inf); cell indices and tags exact except where the oracle position
    is within the position tolerance of a cell face (counted; must be empty for f64); prev columns
    exact (copies of the inputs).  Also returned, not asserted: the largest in-cell displacement error
    `dx_abs` in cell units."""
    tol = TOL[prec]
    m = was_alive.astype(bool)
    out = {}
    f = lambda k: np.asarray(gc[k], np.float64)
    ox1 = op.i1.astype(np.float64) + op.dx1; ox2 = op.i2.astype(np.float64) + op.dx2
    gx1 = gc["i1"].astype(np.float64) + f("dx1"); gx2 = gc["i2"].astype(np.float64) + f("dx2")
    has_phi = op.phi is not None and gc.get("phi") is not None
    ophi = op.phi if has_phi else np.zeros_like(ox1)
    gphi = f("phi") if has_phi else np.zeros_like(ox1)
    xn = np.maximum(1.0, np.max(np.abs(np.stack([ox1, ox2, ophi])), axis=0))
    ex = np.max(np.abs(np.stack([gx1 - ox1, gx2 - ox2, gphi - ophi])), axis=0)
    out["dx_abs"] = float(np.max(np.abs(np.stack([gx1 - ox1, gx2 - ox2]))[:, m], initial=0.0))
    out["phi_abs"] = float(np.max(np.abs(gphi - ophi)[m], initial=0.0))
    # axis conditioning: the midpoint angle of Eq. 29/30 is theta_n + dtheta/2, so a relative rounding error
    # in the computed displacement is amplified by kappa = (|dx2|/2) / (distance of the midpoint to the axis)
    # in every quantity that depends on 1/sin^2(theta_mid)
    # `diag` = the oracle's raw displacement (before renormalisation / reflection)
    p2 = op.i2_prev.astype(np.float64) + op.dx2_prev
    del2 = diag["del2"] if diag is not None else ox2 - p2
    mid2 = p2 + 0.5 * del2
    d_axis = np.maximum(np.minimum(mid2, n2 - mid2), 1e-5 / (np.pi / n2))
    kappa = np.maximum(1.0, 0.5 * np.abs(del2) / d_axis)
    if prec == "f64":
        kappa = np.ones_like(kappa)                   # FP64 meets the flat north_star bound everywhere: no allowance
    ax = (kappa > 1.0) & m
    out["n_axis"] = int(ax.sum())
    out["axis_raw"] = float((ex / xn)[ax].max(initial=0.0))      # their largest error WITHOUT the allowance
    out["k_max"] = float(kappa[m].max(initial=1.0))
    AXIS_STATS.append((prec, int(m.sum()), out["n_axis"], out["axis_raw"], out["k_max"]))
    ex = (ex / (xn * kappa))[m]
    out["x_err"] = float(ex.max(initial=0.0))
    du = np.max(np.abs(np.stack([f("u1") - op.u1, f("u2") - op.u2, f("u3") - op.u3])), axis=0)[m]
    un = np.max(np.abs(np.stack([op.u1, op.u2, op.u3])), axis=0)[m]
    eu = du / np.maximum(1.0, un)
    out["u_err"] = float(eu.max(initial=0.0))
    # indices / tags
    tx = tol["x"]
    near1 = np.minimum(op.dx1, 1 - op.dx1) <= tx * xn
    near2 = np.minimum(op.dx2, 1 - op.dx2) <= tx * xn
    near = (near1 | near2) & m
    bad_idx = ((gc["i1"] != op.i1) | (gc["i2"] != op.i2) | (gc["tag"] != op.tag)) & m
    out["n_face"] = int(near.sum())
    out["n_idx_mismatch"] = int(bad_idx.sum())
    assert not np.any(bad_idx & ~near), f"cell index / tag mismatch away from faces: {np.flatnonzero(bad_idx & ~near)[:10]}"
    if prec == "f64":
        assert out["n_idx_mismatch"] == 0, "FP64 build must reproduce every cell index"
    # a particle whose index differs sits on a face; if that face is an axis it was reflected on one side
    # only (u_2 flips), so momenta are compared only where indices agree; positions always
    ok = ~(bad_idx[m])
    assert np.all(ex[ok] <= tx), f"position error {out['x_err']:.3e} > {tx}"
    assert np.all(eu[ok] <= tol["u"]), f"momentum error {out['u_err']:.3e} > {tol['u']}"
    # absolute bounds in cell units / radians (the norm-wise rule above is loose at i1 ~ 2000): measured 2e-7 (f32)
    abs_tol = 2e-6 if prec == "f32" else 1e-11
    plain = m & ~((kappa > 1.0))
    dxa = np.max(np.abs(np.stack([gx1 - ox1, gx2 - ox2])), axis=0)
    assert np.all(dxa[plain] <= abs_tol), f"in-cell position error {dxa[plain].max():.3e} cells > {abs_tol}"
    dph = np.abs(gphi - ophi)
    assert np.all(dph[plain] <= abs_tol * np.maximum(1.0, np.abs(ophi[plain]))), f"phi error {dph[plain].max():.3e}"
    # the axis allowance: a handful of FP32 particles, their raw error bounded absolutely as well
    assert out["n_axis"] <= max(4, 2e-4 * m.sum()), f"{out['n_axis']} particles lean on the axis-conditioning allowance"
    assert out["axis_raw"] <= 5e-5, f"raw error of an axis-grazing particle {out['axis_raw']:.3e}"
    # dead-before particles are untouched
    d = ~m
    for k in ("i1", "i2", "dx1", "dx2", "u1", "u2", "u3", "tag"):
        assert np.array_equal(np.asarray(gc[k])[d], np.asarray(getattr(op, k))[d].astype(gc[k].dtype)), k
    if check_prev:
        for k in ("i1_prev", "i2_prev", "dx1_prev", "dx2_prev"):
            assert np.array_equal(np.asarray(gc[k])[m], np.asarray(getattr(op, k))[m].astype(gc[k].dtype)), k
    return out


STRADDLE_STEPS = []      # (precision, particles) of every step whose J comparison went through the substitution below


def oracle_deposit_as_the_gpu_decided(O, g, op, after, was_alive, dt, prec):
    """Oracle deposit of the pushed oracle particles `op`, entry-by-entry comparable with the GPU's J even when a few
    FP32 particles within rounding of a cell face ended in the neighbouring cell (or, at a radial edge, on the other
    side of the absorption test): those particles - compare_particles has checked that their continuous position
    agrees within tolerance, and asserts that FP64 has none - are deposited from the GPU's (cell, displacement, tag).
    Returns (J, n_overstep, n_substituted)."""
    bad = np.flatnonzero(((after["i1"] != op.i1) | (after["i2"] != op.i2) | (after["tag"] != op.tag)) & (was_alive != 0))
    if len(bad):
        for k in ("i1", "i2", "dx1", "dx2", "tag"):
            getattr(op, k)[bad] = after[k][bad]
        STRADDLE_STEPS.append((prec, len(bad)))
    Jo, over = O.deposit(g, op, dt)
    return Jo, over, len(bad)


def compare_current(Jo, Jg, prec):
    tol = TOL[prec]["J"]
    out = {}
    for k in ("J1", "J2", "J3"):
        ref = np.asarray(Jo[k], np.float64); got = np.asarray(Jg[k], np.float64)
        scale = np.abs(ref).max()
        err = np.abs(got - ref).max() / (scale if scale > 0 else 1.0)
        out[k] = float(err)
        assert err <= tol, f"{k}: {err:.3e} > {tol}"
    return out
