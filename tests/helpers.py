"""Shared test helpers (host side only; no method arithmetic of the CUDA path)."""
import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def table1():
    rows = {}
    with open(os.path.join(GOLDEN, "table1_orbits.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            t = line.split()
            rows[t[0]] = dict(field=t[1], a=float(t[2]), rmax=float(t[3]), N=int(t[4]), dt=float(t[5]),
                              E=float(t[6]), L=float(t[7]), r=float(t[8]), theta=float(t[9]),
                              u1=float(t[10]), u3=float(t[11]), Bn=float(t[12]))
    return rows


def code_position(O, g, r, theta):
    """(x1, x2) of physical (r, theta) under the A.3 map of grid g (r0, h0 may be non-zero): the radial map is
    inverted in closed form, the polar one by bisection on the oracle's own theta(x2)."""
    r0, h0 = getattr(g, "r0", 0.0), getattr(g, "h0", 0.0)
    if getattr(g, "linear_r", 0):
        x1 = (r - g.r_min) / ((g.r_max - g.r_min) / g.n1)
    else:
        dxi = np.log((g.r_max - r0) / (g.r_min - r0)) / g.n1
        x1 = np.log((r - r0) / (g.r_min - r0)) / dxi
    if h0 == 0.0:
        return x1, theta / (np.pi / g.n2)
    lo, hi = 0.0, float(g.n2)
    for _ in range(80):
        mid = 0.5 * (lo + hi)
        if O.metric(g, x1, mid, derivs=False)["th"][0] < theta:
            lo = mid
        else:
            hi = mid
    return x1, 0.5 * (lo + hi)


def one_particle(O, g, r, theta, u1_phys, u2_phys, u3, q_over_m=0.0, massive=1, phi=0.0):
    """Particle at physical (r, theta) with covariant components in the physical basis:
    u_1 = u_r dr/dx1, u_2 = u_theta dtheta/dx2 (scale factors s1, s2 of the map at that point)."""
    x1, x2 = code_position(O, g, r, theta)
    m = O.metric(g, x1, x2, derivs=False)
    i1, i2 = int(np.floor(x1)), int(np.floor(x2))
    return O.Particles(i1=[i1], i2=[i2], dx1=[x1 - i1], dx2=[x2 - i2],
                       u1=[u1_phys * m["s1"][0]], u2=[u2_phys * m["s2"][0]], u3=[u3],
                       weight=[1.0], tag=[1], phi=[phi], q_over_m=q_over_m, charge=q_over_m, massive=massive)


def pos(p):
    return p.i1.astype(np.float64) + p.dx1, p.i2.astype(np.float64) + p.dx2


def energy_u0(O, g, x1, x2, u1, u2, u3, eps=1.0):
    """-u_0 = alpha*gamma - beta^1 u_1  (P:215 footnote 8 with Eq. 20)."""
    m = O.metric(g, x1, x2, derivs=False)
    gam = np.sqrt(eps + m["hu11"] * u1 ** 2 + m["hu22"] * u2 ** 2 + m["hu33"] * u3 ** 2 + 2 * m["hu13"] * u1 * u3)
    return m["alpha"] * gam - m["beta1"] * u1


def eq59_energy(a, r, th, u1, u2, u3):
    """Eq. 59 retyped with the contravariant 4-metric of A1, physical basis."""
    Sig = r * r + a * a * np.cos(th) ** 2
    Del = r * r - 2 * r + a * a
    z = 2 * r / Sig
    g00, g01, g11, g22 = -(1 + z), z, Del / Sig, 1 / Sig
    g33, g13 = 1 / (Sig * np.sin(th) ** 2), a / Sig
    A = g00
    B = -2 * g01 * u1
    Cc = g11 * u1 ** 2 + g22 * u2 ** 2 + g33 * u3 ** 2 + 2 * g13 * u1 * u3 + 1
    return (-B - np.sqrt(B * B - 4 * A * Cc)) / (2 * A)


# the parity rules and the workload -> oracle conversions live in oracle/parity.py (bench.py and smoke() use them too)
from oracle.parity import (AXIS_STATS, STRADDLE_STEPS, TOL, compare_current, compare_particles, grid_from_domain,  # noqa: E402,F401
                           oracle_deposit_as_the_gpu_decided, oracle_from_cols, oracle_particles)
