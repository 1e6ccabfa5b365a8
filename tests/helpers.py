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


def one_particle(O, g, r, theta, u1_phys, u2_phys, u3, q_over_m=0.0, massive=1, phi=0.0):
    """Particle at physical (r, theta) with covariant components in the physical basis."""
    dxi = np.log(g.r_max / g.r_min) / g.n1
    deta = np.pi / g.n2
    x1 = np.log(r / g.r_min) / dxi
    x2 = theta / deta
    i1, i2 = int(np.floor(x1)), int(np.floor(x2))
    return O.Particles(i1=[i1], i2=[i2], dx1=[x1 - i1], dx2=[x2 - i2],
                       u1=[u1_phys * dxi * r], u2=[u2_phys * deta], u3=[u3],
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


def grid_from_domain(O, dom, n_iter=10):
    return O.Grid(dom.n1, dom.n2, dom.a, dom.r_min, dom.r_max, ng=dom.ng, n_iter=n_iter)


def oracle_particles(O, sp, dtype=np.float64):
    """workloads.Species -> oracle Particles, values rounded through `dtype` first."""
    r = lambda x: np.asarray(x, dtype).astype(np.float64)
    return O.Particles(i1=sp.i1, i2=sp.i2, dx1=r(sp.dx1), dx2=r(sp.dx2), u1=r(sp.u1), u2=r(sp.u2), u3=r(sp.u3),
                       weight=r(sp.weight), tag=sp.tag, phi=None if sp.phi is None else r(sp.phi),
                       q_over_m=sp.q_over_m, charge=sp.charge, massive=sp.massive)
