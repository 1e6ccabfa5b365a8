"""Seeded synthetic inputs shaped like the paper's black-hole magnetosphere runs.

This module is the ONE thing the CUDA path's callers (tests, bench.py, smoke) and the
oracle's callers share.  It holds none of the per-particle method (no interpolation, no
pusher, no deposit): only the recipe that makes initial conditions — Kerr–Schild closed
forms used to (a) evaluate the analytic Wald / monopole potentials on the Yee mesh
(Eq. 12, 17, 60, 62) and (b) turn thermal samples drawn
in a local orthonormal frame into covariant code-basis momenta.  Neither oracle/ nor csrc/
imports it, and no parity result depends on it being physically right: any arrays it
returns are valid inputs to both sides.  Everything is numpy on the host, FP64,
counter-based RNG (Philox) with the seed the config names.

Array layout of every grid array: [n1 + 2*ng][n2 + 2*ng], i2 fastest, Yee locations
D1(i+1/2,j) D2(i,j+1/2) D3(i,j) B1(i,j+1/2) B2(i+1/2,j) B3(i+1/2,j+1/2).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass(frozen=True)
class Domain:
    n1: int
    n2: int
    a: float
    r_min: float
    r_max: float
    ng: int = 2

    @property
    def dxi(self):
        return np.log(self.r_max / self.r_min) / self.n1

    @property
    def deta(self):
        return np.pi / self.n2

    @property
    def shape(self):
        return (self.n1 + 2 * self.ng, self.n2 + 2 * self.ng)

    @property
    def r_h(self):
        return 1.0 + np.sqrt(1.0 - self.a * self.a)


def horizon_radius(a: float) -> float:
    return 1.0 + np.sqrt(1.0 - a * a)


# --------------------------------------------------------------------------------------
# Kerr-Schild closed forms used by the recipe (signed sin(theta): analytic continuation
# across the axis gives ghost values with the parity of P:395 Fig. 1).
# --------------------------------------------------------------------------------------
def ks(dom: Domain, x1, x2):
    x1 = np.asarray(x1, np.float64); x2 = np.asarray(x2, np.float64)
    a = dom.a
    r = dom.r_min * np.exp(x1 * dom.dxi)
    th = x2 * dom.deta
    s, c = np.sin(th), np.cos(th)
    Sig = r * r + a * a * c * c
    Del = r * r - 2 * r + a * a
    A = (r * r + a * a) ** 2 - a * a * Del * s * s
    z = 2 * r / Sig
    s1 = dom.dxi * r
    s2 = dom.deta
    return dict(r=r, th=th, s=s, c=c, Sig=Sig, Del=Del, A=A, z=z, s1=s1, s2=s2,
                alpha=1 / np.sqrt(1 + z), beta1=z / (1 + z) / s1,
                hu11=A / (Sig * (Sig + 2 * r)) / s1 ** 2, hu22=1 / (Sig * s2 ** 2),
                hu13=a / (Sig * s1),
                hd11=s1 ** 2 * (1 + z), hd22=s2 ** 2 * Sig, hd33=A * s * s / Sig,
                hd13=-s1 * a * (1 + z) * s * s)


def wald_potential(dom: Domain, x1, x2, B0=1.0, vertical=False):
    """Code-basis A_0, A_1, A_3 of Eq. 60; vertical=True drops the 2a*xi term."""
    m = ks(dom, x1, x2)
    a, z, s2 = dom.a, m["z"], m["s"] ** 2
    g00, g01, g03 = -(1 - z), z, -a * z * s2
    g13, g33 = -a * (1 + z) * s2, m["A"] * s2 / m["Sig"]
    k = 0.0 if vertical else 2.0 * a
    A0 = 0.5 * B0 * (g03 + k * g00)
    A1 = 0.5 * B0 * (g13 + k * g01) * m["s1"]
    A3 = 0.5 * B0 * (g33 + k * g03)
    return A0, A1, A3


def _yee_coords(dom: Domain, off1: float, off2: float):
    i = np.arange(-dom.ng, dom.n1 + dom.ng, dtype=np.float64) + off1
    j = np.arange(-dom.ng, dom.n2 + dom.ng, dtype=np.float64) + off2
    return np.meshgrid(i, j, indexing="ij")


def em_at(dom: Domain, pot, X1, X2, h: float = 1e-4):
    """All six contravariant code-basis components at the points (X1, X2):
    B^i = eps^{ijk} d_j A_k / sqrt(h) (Eq. 12) and D^i from E_i = d_i A_0 with
    E = alpha D + beta x B (Eq. 17, 38), written in the axis-regular form (sqrt(h) B^k is never
    divided out and multiplied back).  Derivatives of the analytic potential by central
    differences of step h (error ~1e-10 relative)."""
    X1 = np.asarray(X1, np.float64); X2 = np.asarray(X2, np.float64)
    P1p, P1m = pot(dom, X1 + h, X2), pot(dom, X1 - h, X2)
    P2p, P2m = pot(dom, X1, X2 + h), pot(dom, X1, X2 - h)
    d1 = [(P1p[k] - P1m[k]) / (2 * h) for k in range(3)]       # d_1 of (A0, A1, A3)
    d2 = [(P2p[k] - P2m[k]) / (2 * h) for k in range(3)]
    m = ks(dom, X1, X2)
    sqrt_h = m["s1"] * m["s2"] * m["Sig"] * m["s"] / m["alpha"]
    with np.errstate(divide="ignore", invalid="ignore"):
        B1 = d2[2] / sqrt_h
        B2 = -d1[2] / sqrt_h
        B3 = -d2[1] / sqrt_h
        D1 = (m["hu11"] * d1[0] + m["hu13"] * m["beta1"] * d1[2]) / m["alpha"]
        D2 = m["hu22"] * (d2[0] - m["beta1"] * d2[1]) / m["alpha"]
        D3 = (m["hu13"] * d1[0] + m["beta1"] * d1[2] / (m["Sig"] * m["s"] ** 2)) / m["alpha"]
    return dict(D1=D1, D2=D2, D3=D3, B1=B1, B2=B2, B3=B3)


_YEE_OFFSETS = {"D1": (0.5, 0.0), "D2": (0.0, 0.5), "D3": (0.0, 0.0),
                "B1": (0.0, 0.5), "B2": (0.5, 0.0), "B3": (0.5, 0.5)}


def fields_from_potential(dom: Domain, pot, h: float = 1e-4):
    """em_at evaluated pointwise at every Yee location incl. ghosts (signed sin(theta): the
    analytic continuation across the axis gives the ghost parities of P:395)."""
    out = {}
    for k, (o1, o2) in _YEE_OFFSETS.items():
        X1, X2 = _yee_coords(dom, o1, o2)
        out[k] = np.ascontiguousarray(em_at(dom, pot, X1, X2, h)[k])
    # exactly on the axes: theta/phi components vanish by symmetry
    for j_axis in (dom.ng, dom.ng + dom.n2):
        out["B2"][:, j_axis] = 0.0
        out["D3"][:, j_axis] = 0.0
    return out


def wald_fields(dom: Domain, B0=1.0, vertical=False):
    return fields_from_potential(dom, lambda d, a, b: wald_potential(d, a, b, B0, vertical))


def split_monopole_fields(dom: Domain, B0=1.0):
    """Eq. 62: B^1 = B0 sin(theta) sgn(cos theta)/sqrt(h), all else zero.
    In the code basis sin(theta) cancels: B^1 = B0 alpha / (s1 Sigma) * dtheta/dx2 / s2."""
    out = zero_fields(dom)
    X1, X2 = _yee_coords(dom, 0.0, 0.5); m = ks(dom, X1, X2)
    out["B1"] = np.ascontiguousarray(B0 * np.sign(m["c"]) * m["alpha"] / (m["s1"] * m["Sig"]))
    return out


def zero_fields(dom: Domain):
    return {k: np.zeros(dom.shape) for k in ("D1", "D2", "D3", "B1", "B2", "B3")}


def add_random_dB(dom: Domain, fields, amp: float, rng: np.random.Generator):
    """Config 5: each orthonormal component of B gets amp*U(-1,1) per Yee sample, scaled to the
    code basis with the diagonal frame factors at that sample (theta kept 1e-3 cell off the axis)."""
    locs = {"B1": (0.0, 0.5), "B2": (0.5, 0.0), "B3": (0.5, 0.5)}
    for k, (o1, o2) in locs.items():
        X1, X2 = _yee_coords(dom, o1, o2)
        X2 = np.where(np.abs(np.sin(X2 * dom.deta)) < 1e-3 * dom.deta, X2 + 1e-3, X2)
        m = ks(dom, X1, X2)
        scale = {"B1": np.sqrt(m["hu11"]), "B2": 1 / np.sqrt(m["hd22"]), "B3": 1 / np.sqrt(np.abs(m["hd33"]))}[k]
        fields[k] = np.ascontiguousarray(fields[k] + amp * rng.uniform(-1.0, 1.0, size=dom.shape) * scale)
    return fields


# --------------------------------------------------------------------------------------
# Particles
# --------------------------------------------------------------------------------------
@dataclass
class Species:
    """One species = one grpic_particles struct. Host FP64 columns."""
    name: str
    q_over_m: float
    charge: float
    massive: int
    i1: np.ndarray
    i2: np.ndarray
    dx1: np.ndarray
    dx2: np.ndarray
    u1: np.ndarray
    u2: np.ndarray
    u3: np.ndarray
    weight: np.ndarray
    tag: np.ndarray
    phi: np.ndarray | None = None

    @property
    def n(self):
        return int(self.i1.size)


def _mj_speed(rng: np.random.Generator, n: int, T: float):
    """|u| = gamma*beta drawn from Maxwell-Juttner f(u) ~ u^2 exp(-(sqrt(1+u^2)-1)/T) by a
    tabulated inverse CDF (20001 points)."""
    umax = 12.0 * T + 8.0 * np.sqrt(T)
    u = np.linspace(0.0, umax, 20001)
    pdf = u * u * np.exp(-(np.sqrt(1 + u * u) - 1) / T)
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (pdf[1:] + pdf[:-1]))])
    cdf /= cdf[-1]
    return np.interp(rng.random(n), cdf, u)


def _isotropic(rng, n):
    mu = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2 * np.pi, n)
    st = np.sqrt(1 - mu * mu)
    return st * np.cos(ph), st * np.sin(ph), mu


def _frame_to_cov(dom: Domain, i1, i2, uh1, uh2, uh3):
    """Orthonormal-frame momenta -> covariant code basis, frame evaluated at the CELL CENTRE of
    each particle's cell (recipe choice: keeps 1e8-particle generation cheap)."""
    ci, cj = np.meshgrid(np.arange(dom.n1) + 0.5, np.arange(dom.n2) + 0.5, indexing="ij")
    m = ks(dom, ci, cj)
    e11 = 1 / np.sqrt(m["hu11"]); e13 = m["hd13"] / np.sqrt(m["hd33"])
    e22 = np.sqrt(m["hd22"]); e33 = np.sqrt(m["hd33"])
    c = i1.astype(np.int64) * dom.n2 + i2
    u1 = e11.ravel()[c] * uh1 + e13.ravel()[c] * uh3
    u2 = e22.ravel()[c] * uh2
    u3 = e33.ravel()[c] * uh3
    return u1, u2, u3


def thermal_species(dom: Domain, name, counts, T, q_over_m, charge, rng, with_phi=True, chunk=1 << 23):
    """counts: int array [n1][n2] of macro-particles per cell. Uniform in-cell positions,
    Maxwell-Juttner(T) isotropic in the local frame, weight 1."""
    counts = np.asarray(counts, np.int64)
    n = int(counts.sum())
    cell = np.repeat(np.arange(dom.n1 * dom.n2, dtype=np.int64), counts.ravel())
    i1 = (cell // dom.n2).astype(np.int32); i2 = (cell % dom.n2).astype(np.int32)
    del cell
    dx1 = np.empty(n); dx2 = np.empty(n); u1 = np.empty(n); u2 = np.empty(n); u3 = np.empty(n)
    for lo in range(0, n, chunk):
        hi = min(n, lo + chunk); k = hi - lo
        dx1[lo:hi] = rng.random(k); dx2[lo:hi] = rng.random(k)
        sp = _mj_speed(rng, k, T)
        n1_, n2_, n3_ = _isotropic(rng, k)
        a, b, c = _frame_to_cov(dom, i1[lo:hi], i2[lo:hi], sp * n1_, sp * n2_, sp * n3_)
        u1[lo:hi] = a; u2[lo:hi] = b; u3[lo:hi] = c
    return Species(name, q_over_m, charge, 1, i1, i2, dx1, dx2, u1, u2, u3,
                   np.ones(n), np.ones(n, np.uint8), np.zeros(n) if with_phi else None)


def counts_uniform(dom: Domain, per_cell: int):
    return np.full((dom.n1, dom.n2), per_cell, np.int64)


def counts_r2(dom: Domain, total: int):
    """Per-cell count proportional to r_i^-2, largest-remainder rounding to `total`."""
    r = dom.r_min * np.exp((np.arange(dom.n1) + 0.5) * dom.dxi)
    w = np.repeat((r ** -2.0)[:, None], dom.n2, axis=1)
    w = w / w.sum() * total
    base = np.floor(w).astype(np.int64)
    rem = total - int(base.sum())
    if rem > 0:
        idx = np.argsort(-(w - base).ravel(), kind="stable")[:rem]
        base.ravel()[idx] += 1
    return base


def cfl_dt(dom: Domain, cfl: float = 0.5):
    """Reading of "CFL dt 0.5": dt = cfl * min over cell centres of (h^11 + h^22)^-1/2."""
    ci, cj = np.meshgrid(np.arange(dom.n1) + 0.5, np.arange(dom.n2) + 0.5, indexing="ij")
    m = ks(dom, ci, cj)
    return float(cfl * np.min(1 / np.sqrt(m["hu11"] + m["hu22"])))


# Kerr equatorial circular orbits, M = 1, prograde (Bardeen, Press & Teukolsky 1972 closed forms).
def kerr_isco(a: float) -> float:
    z1 = 1 + (1 - a * a) ** (1 / 3) * ((1 + a) ** (1 / 3) + (1 - a) ** (1 / 3))
    z2 = np.sqrt(3 * a * a + z1 * z1)
    return float(3 + z2 - np.sqrt((3 - z1) * (3 + z1 + 2 * z2)))


def kerr_circular_EL(a: float, r):
    r = np.asarray(r, np.float64)
    den = r ** 0.75 * np.sqrt(r ** 1.5 - 3 * np.sqrt(r) + 2 * a)
    return (r ** 1.5 - 2 * np.sqrt(r) + a) / den, (r * r - 2 * a * np.sqrt(r) + a * a) / den


def bl_to_ks_u1(a, r, u0, u3, u1_bl=0.0):
    """Eq. 57: physical-basis u_r in Kerr-Schild from Boyer-Lindquist components."""
    return -(2 * r * u0 + a * u3) / (r * r - 2 * r + a * a) + u1_bl


def geodesic_species(dom: Domain, n: int, rng: np.random.Generator, with_phi=True):
    """Config 2: half near-circular equatorial orbits r in [ISCO, 15], half plunging from r=10."""
    n_c = n // 2; n_p = n - n_c
    a = dom.a
    # near-circular
    r = rng.uniform(kerr_isco(a), 15.0, n_c)
    th = np.pi / 2 + rng.uniform(-0.05, 0.05, n_c)
    E, L = kerr_circular_EL(a, r)
    u1c = bl_to_ks_u1(a, r, -E, L) * (dom.dxi * r)
    u2c = np.zeros(n_c); u3c = L
    # plunging
    rp = np.full(n_p, 10.0)
    thp = np.arccos(rng.uniform(-0.95, 0.95, n_p))
    uh1 = np.full(n_p, -0.5); uh2 = rng.uniform(-1, 1, n_p); uh3 = rng.uniform(-1, 1, n_p)
    x1 = np.log(np.concatenate([r, rp]) / dom.r_min) / dom.dxi
    x2 = np.concatenate([th, thp]) / dom.deta
    i1 = np.floor(x1).astype(np.int32); i2 = np.floor(x2).astype(np.int32)
    dx1 = x1 - i1; dx2 = x2 - i2
    m = ks(dom, x1[n_c:], x2[n_c:])
    u1p = uh1 / np.sqrt(m["hu11"]) + m["hd13"] / np.sqrt(m["hd33"]) * uh3
    u2p = np.sqrt(m["hd22"]) * uh2
    u3p = np.sqrt(m["hd33"]) * uh3
    return Species("test", 0.0, 0.0, 1, i1, i2, dx1, dx2,
                   np.concatenate([u1c, u1p]), np.concatenate([u2c, u2p]), np.concatenate([u3c, u3p]),
                   np.ones(n), np.ones(n, np.uint8), np.zeros(n) if with_phi else None)


# --------------------------------------------------------------------------------------
# The five BASELINE.json configs. `shrink` divides both grid edges (and keeps per-cell
# counts) so the oracle finishes in seconds; shrink=1 is the full size.
# --------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    dom: Domain
    fields: dict
    species: list
    dt: float
    dtype: str
    steps: int
    sort_every: int = 0
    notes: str = ""

    @property
    def n_particles(self):
        return sum(s.n for s in self.species)


def _pairs(dom, counts_each, T, rng, with_phi=True):
    return [thermal_species(dom, "e-", counts_each, T, -1.0, -1.0, rng, with_phi),
            thermal_species(dom, "e+", counts_each, T, +1.0, +1.0, rng, with_phi)]


def config_tiny(shrink: int = 1, seed: int = 0) -> Workload:
    a = 0.9
    dom = Domain(128 // shrink, 64 // shrink, a, 0.9 * horizon_radius(a), 20.0)
    rng = np.random.Generator(np.random.Philox(seed))
    return Workload("tiny", dom, wald_fields(dom, 1.0), _pairs(dom, counts_uniform(dom, 8), 0.1, rng),
                    cfl_dt(dom), "f64", 10)


def config_geodesic(n: int = 1 << 24, dtype: str = "f64", seed: int = 2) -> Workload:
    a = 0.95
    dom = Domain(1024, 512, a, 0.9 * horizon_radius(a), 20.0)
    rng = np.random.Generator(np.random.Philox(seed))
    return Workload("geodesic", dom, zero_fields(dom), [geodesic_species(dom, n, rng)], 0.01, dtype, 100)


def config_magnetosphere(shrink: int = 1, seed: int = 3, ppc_each: int = 32) -> Workload:
    a = 0.99
    dom = Domain(1024 // shrink, 512 // shrink, a, 0.9 * horizon_radius(a), 50.0)
    rng = np.random.Generator(np.random.Philox(seed))
    return Workload("magnetosphere", dom, split_monopole_fields(dom, 1.0),
                    _pairs(dom, counts_uniform(dom, ppc_each), 1.0, rng), cfl_dt(dom), "f32", 10)


def config_large(shrink: int = 1, seed: int = 4, total: int | None = None, with_phi: bool = True) -> Workload:
    a = 0.9375
    dom = Domain(2048 // shrink, 1024 // shrink, a, 0.9 * horizon_radius(a), 100.0)
    rng = np.random.Generator(np.random.Philox(seed))
    if total is None:
        total = 64 * dom.n1 * dom.n2
    cnt = counts_r2(dom, total // 2)
    return Workload("large", dom, wald_fields(dom, 1.0), _pairs(dom, cnt, 0.3, rng, with_phi), cfl_dt(dom),
                    "f32", 10, sort_every=10)


def config_two_species(shrink: int = 1, seed: int = 5, ppc_each: int = 32) -> Workload:
    a = 0.9
    dom = Domain(1024 // shrink, 1024 // shrink, a, 0.9 * horizon_radius(a), 50.0)
    rng = np.random.Generator(np.random.Philox(seed))
    f = add_random_dB(dom, wald_fields(dom, 1.0, vertical=True), 0.1, rng)
    sp = [thermal_species(dom, "e-", counts_uniform(dom, ppc_each), 1.0, -1.0, -1.0, rng),
          thermal_species(dom, "ion", counts_uniform(dom, ppc_each), 0.01, 1.0 / 100.0, +1.0, rng)]
    return Workload("two_species", dom, f, sp, cfl_dt(dom), "f64", 10)
