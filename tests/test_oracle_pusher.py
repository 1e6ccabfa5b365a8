"""Pins for oracle S5-S9 (Boris, geodesic u/x pushes, phi, BCs): Table 1 of the paper,
Kerr closed forms, conservation laws and textbook limits."""
import numpy as np
import pytest

from helpers import code_position, energy_u0, eq59_energy, one_particle, pos, table1


def _grid(O, row, n_iter=10):
    a = row["a"]
    return O.Grid(row["N"], row["N"], a, 0.9 * (1 + np.sqrt(1 - a * a)), row["rmax"], n_iter=n_iter)


def _phys(O, g, p):
    x1, x2 = pos(p)
    m = O.metric(g, x1, x2, derivs=False)
    return m["r"][0], m["th"][0]


# ------------------------------------------------------------------ Table 1 initial values
def test_table1_gr_row_eq57_eq59(O):
    row = table1()["GR"]
    a, r = row["a"], row["r"]
    # Eq. 57 with u_{1,BL}=0, u_0 = -E, u_3 = L reproduces the printed u_1
    u1 = -(2 * r * (-row["E"]) + a * row["L"]) / (r * r - 2 * r + a * a)
    assert abs(u1 - row["u1"]) < 1e-5
    # Eq. 59 reproduces the printed E; the oracle's -u_0 agrees with Eq. 59 to rounding
    E59 = eq59_energy(a, r, row["theta"], row["u1"], 0.0, row["u3"])
    assert abs(E59 - row["E"]) < 1e-5
    g = _grid(O, row)
    p = one_particle(O, g, r, row["theta"], row["u1"], 0.0, row["u3"])
    x1, x2 = pos(p)
    assert abs(energy_u0(O, g, x1, x2, p.u1, p.u2, p.u3)[0] - E59) < 1e-13


def _wald_A(W, g, x1, x2, B0):
    dom = W.Domain(g.n1, g.n2, g.a, g.r_min, g.r_max, g.ng)
    return W.wald_potential(dom, x1, x2, B0)


def test_table1_em_rows_E_L(O, W):
    t = table1()
    # GR-EM-2D: Eq. 61 gives u_phi from L; E = -u_0 (A_0 = 0 for a = 0)
    row = t["GR-EM-2D"]
    B0 = 2 * row["Bn"]                                      # q/m = 1, qB0/2m = Bn
    assert abs((row["L"] - row["r"] ** 2 * row["Bn"]) - row["u3"]) < 1e-12       # Eq. 61
    g = _grid(O, row)
    p = one_particle(O, g, row["r"], row["theta"], row["u1"], 0.0, row["u3"], q_over_m=1.0)
    x1, x2 = pos(p)
    A0, A1, A3 = _wald_A(W, g, x1, x2, B0)
    E = energy_u0(O, g, x1, x2, p.u1, p.u2, p.u3)[0] - A0[0]
    L = p.u3[0] + A3[0]
    assert abs(E - row["E"]) < 5e-4 and abs(E - 0.87339) < 1e-5      # 0.87339: Eq. 59 by hand, see DESIGN.md
    assert abs(L - row["L"]) < 1e-12
    # GR-EM-3D: Eq. 22-23 with Eq. 60, qB0/2m = 1
    row = t["GR-EM-3D"]
    B0 = 2 * row["Bn"]
    g = _grid(O, row)
    p = one_particle(O, g, row["r"], row["theta"], row["u1"], 0.0, row["u3"], q_over_m=1.0)
    x1, x2 = pos(p)
    A0, A1, A3 = _wald_A(W, g, x1, x2, B0)
    E = energy_u0(O, g, x1, x2, p.u1, p.u2, p.u3)[0] - A0[0]
    L = p.u3[0] + A3[0]
    assert abs(E / row["E"] - 1) < 2e-4        # inputs are printed to 4 digits
    assert abs(L / row["L"] - 1) < 2e-4


# ------------------------------------------------------------------ geodesics
def _trace_geodesic(O, g, p, dt, nsteps, eps=1.0):
    E = np.empty(nsteps); R = np.empty(nsteps)
    for k in range(nsteps):
        x1a, x2a = pos(p)
        O.push(g, p, None, dt)
        x1b, x2b = pos(p)
        xm1, xm2 = 0.5 * (x1a + x1b), 0.5 * (x2a + x2b)                 # position at the velocity time level
        E[k] = energy_u0(O, g, xm1, xm2, p.u1, p.u2, p.u3, eps)[0]
        R[k] = O.metric(g, x1b, x2b, derivs=False)["r"][0]
    return E, R


def test_three_leaf_orbit_energy_second_order_and_turning_points(O):
    row = table1()["GR"]
    a = row["a"]
    errs = []
    for dt in (0.04, 0.02, 0.01):
        g = _grid(O, row)
        p = one_particle(O, g, row["r"], row["theta"], row["u1"], 0.0, row["u3"])
        u3_0 = p.u3.copy()
        E0 = energy_u0(O, g, *pos(p), p.u1, p.u2, p.u3)[0]
        E, R = _trace_geodesic(O, g, p, dt, int(round(300 / dt)))
        assert np.array_equal(p.u3, u3_0)                               # u_3 untouched, bit for bit (Eq. 27)
        errs.append(np.max(np.abs(E / E0 - 1)))
        if dt == 0.01:
            # turning points = roots of the Kerr equatorial radial potential (textbook):
            # R(r) = [E(r^2+a^2) - aL]^2 - Delta [r^2 + (L - aE)^2]
            Ee, L = E0, row["L"]
            P = np.poly1d([Ee, 0, Ee * a * a - a * L]) ** 2 - np.poly1d([1, -2, a * a]) * np.poly1d([1, 0, (L - a * Ee) ** 2])
            roots = np.sort(P.roots[np.abs(P.roots.imag) < 1e-9].real)
            r_apo, r_peri = roots[-1], roots[-2]
            assert abs(r_apo - row["r"]) < 2e-4                         # printed start radius is the apocentre
            assert abs(R.max() - r_apo) < 1e-3 and abs(R.min() - r_peri) < 1e-3
    assert errs[0] < 2e-6 and errs[2] < 1e-7                            # bounded
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5


def test_circular_orbits_are_fixed_points(O, W):
    a = 0.95
    g = O.Grid(1024, 512, a, 0.9 * (1 + np.sqrt(1 - a * a)), 20.0)
    risco = W.kerr_isco(a)
    assert abs(risco - 1.93724) < 1e-5
    for r0 in (1.0001 * risco, 6.0, 15.0):
        E, L = W.kerr_circular_EL(a, r0)
        u1 = W.bl_to_ks_u1(a, r0, -E, L)
        p = one_particle(O, g, r0, np.pi / 2, u1, 0.0, L)
        assert abs(energy_u0(O, g, *pos(p), p.u1, p.u2, p.u3)[0] - E) < 1e-12
        dt, n = 0.01, 1000
        for _ in range(n):
            O.push(g, p, None, dt)
        r, th = _phys(O, g, p)
        assert abs(r / r0 - 1) < 1e-9 and abs(th - np.pi / 2) < 1e-12
        assert abs(p.phi[0] / (n * dt) - 1 / (r0 ** 1.5 + a)) < 1e-8      # Kepler frequency in Kerr


def test_schwarzschild_radial_plunge_closed_form(O):
    """E = 1, L = 0 infall from rest at infinity, a = 0, in Kerr-Schild time:
    u_r = -s/(1+s),  dr/dt = -s(1+s)/(1+s+s^2),  s = sqrt(2/r)  (derivation in DESIGN.md)."""
    g = O.Grid(512, 64, 0.0, 1.5, 40.0)
    r0 = 30.0
    s = np.sqrt(2 / r0)
    p = one_particle(O, g, r0, np.pi / 2, -s / (1 + s), 0.0, 0.0)
    dt = 0.01
    for _ in range(2000):
        x1a, _ = pos(p)
        ra = O.metric(g, x1a, [32.0], derivs=False)["r"][0]
        O.push(g, p, None, dt)
        x1b, x2b = pos(p)
        mb = O.metric(g, x1b, x2b, derivs=False)
        rb = mb["r"][0]
        rm = 0.5 * (ra + rb); sm = np.sqrt(2 / rm)
        assert abs((rb - ra) / dt + sm * (1 + sm) / (1 + sm + sm * sm)) < 2e-4
    sb = np.sqrt(2 / rb)
    assert abs(p.u1[0] / mb["s1"][0] + sb / (1 + sb)) < 2e-4
    assert rb < r0 - 4.0


def test_radial_photons_schwarzschild(O):
    """Massless (Eq. 20): in Kerr-Schild coordinates ingoing radial null rays have dr/dt = -1
    and outgoing ones (1-z)/(1+z)."""
    g = O.Grid(512, 64, 0.0, 1.5, 40.0, n_iter=10)
    for sign in (-1.0, +1.0):
        p = one_particle(O, g, 10.0, np.pi / 2, sign * 3.0, 0.0, 0.0, massive=0)
        dt = 0.01
        E = []
        for _ in range(300):
            x1a, x2a = pos(p)
            ra = O.metric(g, x1a, [32.0], derivs=False)["r"][0]
            O.push(g, p, None, dt)
            x1b, x2b = pos(p)
            rb = O.metric(g, x1b, [32.0], derivs=False)["r"][0]
            rm = 0.5 * (ra + rb); z = 2 / rm
            want = -1.0 if sign < 0 else (1 - z) / (1 + z)
            assert abs((rb - ra) / dt - want) < 1e-6
            E.append(energy_u0(O, g, 0.5 * (x1a + x1b), 0.5 * (x2a + x2b), p.u1, p.u2, p.u3, eps=0.0)[0])
        # photon energy -u_0 conserved along the ray (time-aligned as in P:585)
        assert abs(max(E) / min(E) - 1) < 1e-6          # O(dt^2)


def test_n_iter_one_is_explicit_euler(O):
    """First guess = start value and exactly n_iter applications: with n_iter = 1 both
    updates are explicit Euler steps evaluated at the start state."""
    a = 0.9
    g = O.Grid(128, 64, a, 1.2, 20.0, n_iter=1)
    p = one_particle(O, g, 5.0, 1.0, 0.3, -0.2, 2.5)
    x1, x2 = pos(p)
    m = O.metric(g, x1, x2)
    u = np.array([p.u1[0], p.u2[0], p.u3[0]])
    dt = 0.05

    def gam(u):
        return np.sqrt(1 + m["hu11"][0] * u[0] ** 2 + m["hu22"][0] * u[1] ** 2 + m["hu33"][0] * u[2] ** 2
                       + 2 * m["hu13"][0] * u[0] * u[2])
    u0 = gam(u) / m["alpha"][0]
    unew = u.copy()
    for i, ax in enumerate(("d1_", "d2_")):
        unew[i] = u[i] + dt * (-m["alpha"][0] * u0 * m[ax + "alpha"][0] + u[0] * m[ax + "beta1"][0]
                               - (m[ax + "hu11"][0] * u[0] ** 2 + m[ax + "hu22"][0] * u[1] ** 2
                                  + m[ax + "hu33"][0] * u[2] ** 2 + 2 * m[ax + "hu13"][0] * u[0] * u[2]) / (2 * u0))
    u0n = gam(unew) / m["alpha"][0]
    d1 = dt * ((m["hu11"][0] * unew[0] + m["hu13"][0] * unew[2]) / u0n - m["beta1"][0])
    d2 = dt * (m["hu22"][0] * unew[1] / u0n)
    O.push(g, p, None, dt)
    assert np.allclose([p.u1[0], p.u2[0], p.u3[0]], unew, rtol=1e-13)
    y1, y2 = pos(p)
    assert abs((y1 - x1)[0] - d1) < 1e-12 and abs((y2 - x2)[0] - d2) < 1e-12


def test_fixed_point_iteration_converges_to_implicit_midpoint(O):
    """n_iter = 10 vs 30 agree to rounding for a typical step ("convergence ... within ten iterations")."""
    a = 0.9
    out = []
    for n_iter in (10, 30):
        g = O.Grid(128, 64, a, 1.2, 20.0, n_iter=n_iter)
        p = one_particle(O, g, 3.0, 0.7, 0.4, -0.3, 2.0)
        O.push(g, p, None, 0.02)
        out.append(np.array([*pos(p), p.u1, p.u2]).ravel())
    assert np.allclose(out[0], out[1], rtol=1e-13, atol=1e-13)


# ------------------------------------------------------------------ EM push
def test_boris_rotation_closed_form(O):
    """Uniform tetrad-frame B, no D: |u| conserved and a half push turns u by 2*atan(c|B|/gamma)."""
    a = 0.0
    g = O.Grid(64, 32, a, 1.5, 30.0, n_iter=0)                 # n_iter = 0: no geodesic update at all
    x1, x2 = 30.2, 13.4
    m = O.metric(g, [x1], [x2], derivs=False)
    Bh = np.array([0.0, 0.0, 0.7]); uh = np.array([1.3, 0.4, 0.0])
    Bc = O.tetrad_to_cntrv(g, x1, x2, Bh)
    uc = O.tetrad_to_cov(g, x1, x2, uh)
    p = O.Particles(i1=[30], i2=[13], dx1=[x1 - 30], dx2=[x2 - 13], u1=[uc[0]], u2=[uc[1]], u3=[uc[2]],
                    weight=[1.0], tag=[1], phi=[0.0], q_over_m=-1.0, charge=-1.0)
    dt = 0.3
    O.push_given_fields(g, p, np.zeros(3), Bc, dt)
    un = O.cov_to_tetrad(g, x1, x2, [p.u1[0], p.u2[0], p.u3[0]])
    assert abs(np.linalg.norm(un) - np.linalg.norm(uh)) < 1e-13
    gam = np.sqrt(1 + uh @ uh)
    c = -1.0 * m["alpha"][0] * dt / 4
    want = 2 * (2 * np.arctan(c * 0.7 / gam))                 # two half pushes
    got = np.arctan2(un[1], un[0]) - np.arctan2(uh[1], uh[0])
    # u' = u + u x t: for B along +3 and q<0 ... sign fixed by dv/dt = (q/m) v x B
    assert abs(got - (-want)) < 1e-12
    # pure electric kick: u_hat changes by 4 c D_hat
    Dh = np.array([0.2, -0.1, 0.05])
    p2 = O.Particles(i1=[30], i2=[13], dx1=[x1 - 30], dx2=[x2 - 13], u1=[uc[0]], u2=[uc[1]], u3=[uc[2]],
                     weight=[1.0], tag=[1], phi=[0.0], q_over_m=-1.0, charge=-1.0)
    O.push_given_fields(g, p2, O.tetrad_to_cntrv(g, x1, x2, Dh), np.zeros(3), dt)
    un2 = O.cov_to_tetrad(g, x1, x2, [p2.u1[0], p2.u2[0], p2.u3[0]])
    assert np.allclose(un2 - uh, 4 * c * Dh, rtol=1e-12, atol=1e-14)


def _trace_wald(O, W, row, dt, T):
    g = _grid(O, row)
    dom = W.Domain(g.n1, g.n2, g.a, g.r_min, g.r_max, g.ng)
    B0 = 2 * row["Bn"]
    pot = lambda d, a, b: W.wald_potential(d, a, b, B0)
    p = one_particle(O, g, row["r"], row["theta"], row["u1"], 0.0, row["u3"], q_over_m=1.0)

    def EL(x1, x2):
        A0, A1, A3 = pot(dom, x1, x2)
        return energy_u0(O, g, x1, x2, p.u1, p.u2, p.u3)[0] - A0[0], p.u3[0] + A3[0]
    E0, L0 = EL(*pos(p))
    eE = eL = 0.0
    for _ in range(int(round(T / dt))):
        x1a, x2a = pos(p)
        f = W.em_at(dom, pot, x1a, x2a)
        O.push_given_fields(g, p, [f["D1"][0], f["D2"][0], f["D3"][0]], [f["B1"][0], f["B2"][0], f["B3"][0]], dt)
        x1b, x2b = pos(p)
        E, L = EL(0.5 * (x1a + x1b), 0.5 * (x2a + x2b))
        eE = max(eE, abs(E / E0 - 1)); eL = max(eL, abs(L / L0 - 1))
    return eE, eL


def test_wald_orbit_a0_conserves_E_and_L(O, W):
    """GR-EM-2D: with the analytic Wald field at the particle the canonical
    energy and angular momentum (Eq. 22-23) are conserved to O(dt^2).  Pins the lapse in the
    Boris coefficient (R-S5), the cross-product sign and the tetrad projections."""
    row = table1()["GR-EM-2D"]
    e1 = _trace_wald(O, W, row, 0.02, 60.0)
    e2 = _trace_wald(O, W, row, 0.01, 60.0)
    assert e2[0] < 2e-6 and e2[1] < 2e-6
    assert 2.5 < e1[0] / e2[0] < 5.0 and 2.5 < e1[1] / e2[1] < 5.0


def test_wald_orbit_a09_conserves_E_and_L(O, W):
    row = table1()["GR-EM-3D"]
    e1 = _trace_wald(O, W, row, 0.002, 4.0)
    e2 = _trace_wald(O, W, row, 0.001, 4.0)
    assert e2[0] < 1e-6 and e2[1] < 1e-6
    assert 2.5 < e1[0] / e2[0] < 5.0 and 2.5 < e1[1] / e2[1] < 5.0


# ------------------------------------------------------------------ boundary conditions
def _bc_particle(O, i1, i2, dx1, dx2, u1, u2, u3=0.0):
    return O.Particles(i1=[i1], i2=[i2], dx1=[dx1], dx2=[dx2], u1=[u1], u2=[u2], u3=[u3],
                       weight=[1.0], tag=[1], phi=[0.0])


def test_axis_reflection_and_radial_absorption(O):
    a = 0.9
    g = O.Grid(128, 64, a, 0.9 * (1 + np.sqrt(1 - a * a)), 20.0)
    # towards theta = 0: reflected, u_2 flips, stays in cell 0
    p = _bc_particle(O, 60, 0, 0.5, 0.02, 0.0, -0.05)
    c = O.push(g, p, None, 0.5)
    assert c == (1, 0, 0) and p.tag[0] == 1 and p.i2[0] == 0 and 0 <= p.dx2[0] < 1 and p.u2[0] > 0
    # towards theta = pi
    p = _bc_particle(O, 60, 63, 0.5, 0.98, 0.0, +0.05)
    O.push(g, p, None, 0.5)
    assert p.i2[0] == 63 and 0 <= p.dx2[0] < 1 and p.u2[0] < 0 and p.tag[0] == 1
    # inside the horizon everything falls inward: leaves through i1 < 0
    p = _bc_particle(O, 0, 30, 0.01, 0.5, -0.1, 0.0)
    c = O.push(g, p, None, 0.5)
    assert c == (0, 1, 0) and p.tag[0] == 0 and p.i1[0] < 0
    # outer edge
    p = _bc_particle(O, 127, 30, 0.99, 0.5, 3.0, 0.0)
    c = O.push(g, p, None, 0.5)
    assert c == (0, 0, 1) and p.tag[0] == 0 and p.i1[0] >= 128
    # dead particles are ignored by later calls
    before = (p.i1[0], p.dx1[0], p.u1[0])
    c = O.push(g, p, None, 0.5)
    assert c == (0, 0, 0) and (p.i1[0], p.dx1[0], p.u1[0]) == before


def test_previous_position_saved_and_renormalised(O):
    a = 0.9
    g = O.Grid(128, 64, a, 0.9 * (1 + np.sqrt(1 - a * a)), 20.0)
    rng = np.random.default_rng(3)
    n = 2000
    p = O.Particles(i1=rng.integers(5, 120, n), i2=rng.integers(1, 63, n), dx1=rng.random(n), dx2=rng.random(n),
                    u1=rng.normal(size=n) * 0.05, u2=rng.normal(size=n) * 0.05, u3=rng.normal(size=n) * 3,
                    weight=np.ones(n), tag=np.ones(n), phi=np.zeros(n))
    q = p.copy()
    O.push(g, p, None, 0.2)
    assert np.array_equal(p.i1_prev, q.i1) and np.array_equal(p.dx1_prev, q.dx1)
    assert np.array_equal(p.i2_prev, q.i2) and np.array_equal(p.dx2_prev, q.dx2)
    assert np.all((p.dx1 >= 0) & (p.dx1 < 1) & (p.dx2 >= 0) & (p.dx2 < 1))
    moved = np.abs((p.i1 + p.dx1) - (q.i1 + q.dx1))
    assert moved.max() > 0.05


# --------------------------------------------------------------------------------------------
# Brute-force single-particle traces (north_star): Hamilton's equations of the 3+1 split,
#   H = -u_0 = alpha*sqrt(eps + h^ij u_i u_j) - beta^i u_i  (P:215 footnote 8 with Eq. 20),
#   dx^i/dt = dH/du_i,  du_i/dt = -dH/dx^i,
# in PHYSICAL Kerr-Schild coordinates (r, theta), with the textbook contravariant 3-metric typed out
# here and the derivatives of H taken numerically (central differences): nothing of App. A's
# derivative list, of the code basis or of the midpoint scheme is shared with the oracle.
# Integrated by scipy's DOP853 to 1e-12; the oracle's trajectory must converge to it at second order.
# A wrong sign or a dropped term in Eq. 26-29 or in the A.2/A.3 derivatives fails this test.
# --------------------------------------------------------------------------------------------
def _H_phys(a, eps, r, th, ur, uth, uph):
    S = r * r + a * a * np.cos(th) ** 2
    D = r * r - 2 * r + a * a
    A = (r * r + a * a) ** 2 - a * a * D * np.sin(th) ** 2
    z = 2 * r / S
    alpha, beta_r = 1 / np.sqrt(1 + z), z / (1 + z)
    g2 = eps + A / (S * (S + 2 * r)) * ur * ur + uth * uth / S + uph * uph / (S * np.sin(th) ** 2) + 2 * a / S * ur * uph
    return alpha * np.sqrt(g2) - beta_r * ur


def _brute_force_trace(a, eps, y0, times):
    """state (r, theta, phi, u_r, u_theta, u_phi) at each of `times` (any sign), from y0 at t = 0"""
    from scipy.integrate import solve_ivp

    def rhs(t, y):
        r, th, ph, ur, uth, uph = y
        h = 1e-6
        d = lambda k: (_H_phys(a, eps, *(np.array([r, th, ur, uth, uph]) + h * np.eye(5)[k])) -
                       _H_phys(a, eps, *(np.array([r, th, ur, uth, uph]) - h * np.eye(5)[k]))) / (2 * h)
        return [d(2), d(3), d(4), -d(0), -d(1), 0.0]

    back = [t for t in times if t < 0]
    fwd = sorted(t for t in times if t > 0)
    out = {}
    for t in back:
        out[t] = solve_ivp(rhs, (0.0, t), y0, method="DOP853", rtol=1e-12, atol=1e-13).y[:, -1]
    if fwd:
        sol = solve_ivp(rhs, (0.0, fwd[-1]), y0, method="DOP853", rtol=1e-12, atol=1e-13, t_eval=fwd)
        for k, t in enumerate(fwd):
            out[t] = sol.y[:, k]
    return [out[t] for t in times]


@pytest.mark.parametrize("a,eps,r0,th0,ur,uth,uph", [(0.9, 1.0, 6.0, 1.2, -0.1, 0.8, 2.5),      # inclined bound-ish orbit
                                                     (0.995, 1.0, 3.0, np.pi / 2 - 0.3, 0.05, -0.5, 1.9),  # near the hole
                                                     (0.7, 0.0, 8.0, 0.9, -0.6, 1.5, -2.0)])   # photon, retrograde
@pytest.mark.parametrize("r_off,h0,lin", [(0.0, 0.0, 0), (0.6, 0.35, 0), (0.0, 0.0, 1)])
def test_brute_force_single_particle_trace(O, a, eps, r0, th0, ur, uth, uph, r_off, h0, lin):
    T = 1.0
    y0 = [r0, th0, 0.0, ur, uth, uph]
    errs = []
    for dt in (0.02, 0.01, 0.005):
        # leapfrog (Sec. 3.1): positions live at t_n, velocities at t_(n-1/2).  The oracle starts from
        # x(0) and u(-dt/2) of the brute-force trajectory and must end at x(T), u(T - dt/2) of the same trajectory.
        y_m, y_u, y_x = _brute_force_trace(a, eps, y0, [-0.5 * dt, T - 0.5 * dt, T])
        g = O.Grid(256, 128, a, 0.9 * (1 + np.sqrt(1 - a * a)), 30.0, n_iter=25, r0=r_off, h0=h0, linear_r=lin)
        # u_1 = u_r dr/dx1, u_2 = u_theta dtheta/dx2 are the momenta conjugate to x1, x2: their scale factors are
        # taken where u lives (t = -dt/2), the position where x lives (t = 0)
        s_m = O.metric(g, *code_position(O, g, y_m[0], y_m[1]), derivs=False)
        s_0 = O.metric(g, *code_position(O, g, r0, th0), derivs=False)
        p = one_particle(O, g, r0, th0, y_m[3] * s_m["s1"][0] / s_0["s1"][0], y_m[4] * s_m["s2"][0] / s_0["s2"][0],
                         y_m[5], massive=int(eps))
        for _ in range(int(round(T / dt))):
            O.push(g, p, None, dt)
        r, th = _phys(O, g, p)
        # covariant components at (T - dt/2) back in the physical basis, scale factors where u lives
        s_u = O.metric(g, *code_position(O, g, y_u[0], y_u[1]), derivs=False)
        got = np.array([r, th, p.phi[0], p.u1[0] / s_u["s1"][0], p.u2[0] / s_u["s2"][0], p.u3[0]])
        ref = np.array([y_x[0], y_x[1], y_x[2], y_u[3], y_u[4], y_u[5]])
        errs.append(np.max(np.abs(got - ref) / np.maximum(1.0, np.abs(ref))))
    assert errs[2] < 1e-5, errs                                           # converged to the brute-force trace
    assert 3.3 < errs[0] / errs[1] < 4.7 and 3.3 < errs[1] / errs[2] < 4.7, errs   # at second order


def _A_wald_phys(a, B0, r, th):
    """Eq. 60: A_mu = (B0/2)(g_{mu phi} + 2a g_{mu t}) with the covariant Kerr-Schild 4-metric (A1)."""
    S = r * r + a * a * np.cos(th) ** 2
    D = r * r - 2 * r + a * a
    A = (r * r + a * a) ** 2 - a * a * D * np.sin(th) ** 2
    z, s2 = 2 * r / S, np.sin(th) ** 2
    g00, g01, g03 = -(1 - z), z, -a * z * s2
    g13, g33 = -a * (1 + z) * s2, A * s2 / S
    return 0.5 * B0 * (g03 + 2 * a * g00), 0.5 * B0 * (g13 + 2 * a * g01), 0.5 * B0 * (g33 + 2 * a * g03)


def _brute_force_charged(a, B0, qm, y0, times):
    """Canonical Hamiltonian of a charge in the stationary Wald field, t as the parameter:
    H = alpha*gamma(u) - beta^r u_r - (q/m) A_0,  u_i = pi_i - (q/m) A_i;  y = (r, theta, pi_r, pi_theta, pi_phi)."""
    from scipy.integrate import solve_ivp

    def H(r, th, pr, pth, pph):
        A0, Ar, Aph = _A_wald_phys(a, B0, r, th)
        return _H_phys(a, 1.0, r, th, pr - qm * Ar, pth, pph - qm * Aph) - qm * A0

    def rhs(t, y):
        h = 1e-6
        d = lambda k: (H(*(y + h * np.eye(5)[k])) - H(*(y - h * np.eye(5)[k]))) / (2 * h)
        return [d(2), d(3), -d(0), -d(1), 0.0]

    out = []
    for t in times:
        out.append(solve_ivp(rhs, (0.0, t), y0, method="DOP853", rtol=1e-12, atol=1e-13).y[:, -1])
    return out


def test_brute_force_charged_trace_in_wald_field(O, W):
    """GR-EM-3D row of Table 1 (a = 0.9, Wald field): the oracle's EM + geodesic push with the
    analytic D, B at the particle against the brute-force canonical trajectory.  Pins the Boris coefficient
    (q/m) alpha dt/4 of R-S5, the tetrad projections and the order of the two half pushes: second-order convergence
    to an independent solution, not only conservation of two invariants."""
    row = table1()["GR-EM-3D"]
    a, B0, qm, T = row["a"], 2 * row["Bn"], 1.0, 0.5
    r0, th0 = row["r"], row["theta"]
    A0, Ar, Aph = _A_wald_phys(a, B0, r0, th0)
    y0 = np.array([r0, th0, row["u1"] + qm * Ar, 0.0, row["u3"] + qm * Aph])
    errs = []
    for dt in (0.004, 0.002, 0.001):
        y_m, y_u, y_x = _brute_force_charged(a, B0, qm, y0, [-0.5 * dt, T - 0.5 * dt, T])
        g = _grid(O, row)
        dom = W.Domain(g.n1, g.n2, g.a, g.r_min, g.r_max, g.ng)
        pot = lambda d, x, y: W.wald_potential(d, x, y, B0)
        # kinetic u at t = -dt/2 from the canonical momenta of the brute-force trajectory
        _, Ar_m, Aph_m = _A_wald_phys(a, B0, y_m[0], y_m[1])
        p = one_particle(O, g, r0, th0, (y_m[2] - qm * Ar_m) * y_m[0] / r0, y_m[3], y_m[4] - qm * Aph_m, q_over_m=qm)
        for _ in range(int(round(T / dt))):
            f = W.em_at(dom, pot, *pos(p))
            O.push_given_fields(g, p, [f["D1"][0], f["D2"][0], f["D3"][0]], [f["B1"][0], f["B2"][0], f["B3"][0]], dt)
        r, th = _phys(O, g, p)
        dxi, deta = np.log(g.r_max / g.r_min) / g.n1, np.pi / g.n2
        _, Ar_u, Aph_u = _A_wald_phys(a, B0, y_u[0], y_u[1])
        got = np.array([r, th, p.u1[0] / (dxi * y_u[0]), p.u2[0] / deta, p.u3[0]])
        ref = np.array([y_x[0], y_x[1], y_u[2] - qm * Ar_u, y_u[3], y_u[4] - qm * Aph_u])
        errs.append(np.max(np.abs(got - ref) / np.maximum(1.0, np.abs(ref))))
    assert errs[2] < 1e-5, errs
    assert 3.3 < errs[0] / errs[1] < 4.7 and 3.3 < errs[1] / errs[2] < 4.7, errs


# ------------------------------------------------------------------ flat spherical metric (App. A.1) and the SR-EM row
def _flat_grid(O, n=256, n_iter=10):
    return O.Grid(n, n, 0.0, 1.0, 20.0, linear_r=1, mass=0.0, n_iter=n_iter)


def test_flat_metric_is_appendix_a1(O):
    """kerr_schild_0: h_ij = diag(dr^2, dtheta^2 r^2, r^2 sin^2), alpha = 1, beta = 0,
    sqrt(h) = dr dtheta r^2 sin(theta); every derivative vanishes except the three the paper prints."""
    g = _flat_grid(O)
    x1 = np.array([3.3, 100.7, 200.2]); x2 = np.array([20.4, 128.0, 230.9])
    m = O.metric(g, x1, x2)
    dr, dth = (g.r_max - g.r_min) / g.n1, np.pi / g.n2
    r, th = g.r_min + x1 * dr, x2 * dth
    assert np.allclose(m["r"], r, rtol=1e-15) and np.allclose(m["th"], th, rtol=1e-15)
    assert np.all(m["alpha"] == 1.0) and np.all(m["beta1"] == 0.0) and np.all(m["hd13"] == 0.0) and np.all(m["hu13"] == 0.0)
    assert np.allclose(m["hd11"], dr ** 2, rtol=1e-14) and np.allclose(m["hd22"], (dth * r) ** 2, rtol=1e-14)
    assert np.allclose(m["hd33"], (r * np.sin(th)) ** 2, rtol=1e-14)
    assert np.allclose(m["sqrt_h"], dr * dth * r ** 2 * np.sin(th), rtol=1e-14)
    assert np.allclose(m["d1_hu33"], -dr * 2 / (r ** 3 * np.sin(th) ** 2), rtol=1e-13)
    assert np.allclose(m["d1_hu22"], -dr * 2 / (r ** 3 * dth ** 2), rtol=1e-13)
    assert np.allclose(m["d2_hu33"], -2 * dth * np.cos(th) / (r ** 2 * np.sin(th) ** 3), rtol=1e-13)
    for k in ("d1_hu11", "d2_hu11", "d2_hu22", "d1_hu13", "d2_hu13", "d1_alpha", "d2_alpha", "d1_beta1", "d2_beta1"):
        assert np.all(m[k] == 0.0), k


def test_table1_sr_em_gyration_closed_orbit(O):
    """SR-EM row of Table 1: flat metric, uniform vertical field, rho0 = 2 r_g.  Textbook
    gyration: E = sqrt(2) (printed 1.41421), and the orbit is the circle of Larmor radius
    rho = rho0 * u_phi-hat = 2 r_g that closes after T = 2 pi gamma/(qB/m); "the trajectory remains closed
    and the energy error stays bounded".  The curvilinear inertial terms of Eq. 26-29 and the tetrad
    projections must cancel to leave a circle in the plane."""
    row = table1()["SR-EM"]
    g = _flat_grid(O, 1024)
    qB = 2 * row["Bn"]                                                   # q B0/m with q/m = 1
    p = one_particle(O, g, row["r"], row["theta"], row["u1"], 0.0, row["u3"], q_over_m=1.0)
    gam0 = np.sqrt(1 + (row["u3"] / row["r"]) ** 2)
    assert abs(gam0 - row["E"]) < 1e-5                                    # printed energy
    dt = row["dt"]
    T = 2 * np.pi * gam0 / qB
    n = int(round(T / dt))
    xs, ys, gs = [], [], []
    for _ in range(n):
        m = O.metric(g, *pos(p), derivs=False)
        r, th = m["r"][0], m["th"][0]
        B = [qB * np.cos(th) / m["s1"][0], -qB * np.sin(th) / (r * m["s2"][0]), 0.0]   # uniform B0 z-hat, code basis
        xa = pos(p)
        O.push_given_fields(g, p, [0.0, 0.0, 0.0], B, dt)
        xb = pos(p)
        m = O.metric(g, *xb, derivs=False)
        r = m["r"][0]
        xs.append(r * np.cos(p.phi[0])); ys.append(r * np.sin(p.phi[0]))
        mm = O.metric(g, 0.5 * (xa[0] + xb[0]), 0.5 * (xa[1] + xb[1]), derivs=False)   # position at the velocity time level
        gs.append(np.sqrt(1 + mm["hu11"][0] * p.u1[0] ** 2 + mm["hu22"][0] * p.u2[0] ** 2 + mm["hu33"][0] * p.u3[0] ** 2))
        assert abs(m["th"][0] - np.pi / 2) < 1e-12                        # stays in the equatorial plane
    xs, ys, gs = np.array(xs), np.array(ys), np.array(gs)
    assert np.max(np.abs(gs / gam0 - 1)) < 1e-6                           # bounded energy error
    cx, cy = xs.mean(), ys.mean()
    rho = np.hypot(xs - cx, ys - cy)
    # gyro-centre 2 r_g from the start point; the printed u is used as u(-dt/2) (leapfrog), which shifts the circle by
    # v dt/2 = 0.0035 r_g along the initial velocity
    assert abs(abs(cx - row["r"]) - 2.0) < 2e-3 and abs(cy) < 6e-3
    assert np.max(np.abs(rho - 2.0)) < 2e-3                               # Larmor radius rho = 2 r_g
    assert np.hypot(xs[-1] - row["r"], ys[-1]) < 2e-2                     # closed after one period (n*dt ~ T)
