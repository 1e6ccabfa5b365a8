"""Pins for oracle S4 (interpolation) and S10 (deposit), plus the sort reference."""
import numpy as np
import pytest

COMPS = ("D1", "D2", "D3", "B1", "B2", "B3")
OFFS = {"D1": (0.5, 0.0), "D2": (0.0, 0.5), "D3": (0.0, 0.0), "B1": (0.0, 0.5), "B2": (0.5, 0.0), "B3": (0.5, 0.5)}


@pytest.fixture(scope="module")
def g(O):
    return O.Grid(24, 16, 0.9, 1.3, 20.0)


def _field_from(g, fn):
    """Sample fn(comp, x1, x2) at each component's own Yee location, ghosts included."""
    out = {}
    for k in COMPS:
        i = np.arange(-g.ng, g.n1 + g.ng) + OFFS[k][0]
        j = np.arange(-g.ng, g.n2 + g.ng) + OFFS[k][1]
        X1, X2 = np.meshgrid(i, j, indexing="ij")
        out[k] = np.ascontiguousarray(fn(k, X1, X2))
    return out


def test_interp_reproduces_constant_and_linear_fields(O, g):
    rng = np.random.default_rng(0)
    n = 500
    i1 = rng.integers(0, g.n1, n); i2 = rng.integers(0, g.n2, n)
    dx1 = rng.random(n); dx2 = rng.random(n)
    coef = {k: rng.normal(size=3) for k in COMPS}
    F = _field_from(g, lambda k, X1, X2: coef[k][0] + coef[k][1] * X1 + coef[k][2] * X2)
    D, B = O.interp(g, F, i1, i2, dx1, dx2)
    got = dict(D1=D[:, 0], D2=D[:, 1], D3=D[:, 2], B1=B[:, 0], B2=B[:, 1], B3=B[:, 2])
    x1, x2 = i1 + dx1, i2 + dx2
    for k in COMPS:
        want = coef[k][0] + coef[k][1] * x1 + coef[k][2] * x2
        assert np.allclose(got[k], want, rtol=0, atol=1e-12), k


def test_interp_continuous_across_faces_and_first_order_footprint(O, g):
    rng = np.random.default_rng(1)
    F = {k: rng.normal(size=g.shape) for k in COMPS}
    # continuity: (i, dx=1-eps) vs (i+1, dx=0)
    eps = 1e-12
    for (ia, da, ib, db, ja, ea, jb, eb) in [(5, 1 - eps, 6, 0.0, 7, 0.3, 7, 0.3), (5, 0.6, 5, 0.6, 7, 1 - eps, 8, 0.0)]:
        Da, Ba = O.interp(g, F, [ia], [ja], [da], [ea])
        Db, Bb = O.interp(g, F, [ib], [jb], [db], [eb])
        assert np.allclose(Da, Db, atol=1e-10) and np.allclose(Ba, Bb, atol=1e-10)
    # footprint: only samples in cells (i-1..i+1, j-1..j+1) matter
    D0, B0 = O.interp(g, F, [10], [8], [0.37], [0.81])
    F2 = {k: v.copy() for k, v in F.items()}
    mask = np.ones(g.shape, bool)
    mask[10 - 1 + g.ng:10 + 2 + g.ng, 8 - 1 + g.ng:8 + 2 + g.ng] = False
    for k in COMPS:
        F2[k][mask] = 1e6
    D1, B1 = O.interp(g, F2, [10], [8], [0.37], [0.81])
    assert np.array_equal(D0, D1) and np.array_equal(B0, B1)
    # at a node the value is the average of the nearest samples of that component
    Dn, Bn = O.interp(g, F, [10], [8], [0.0], [0.0])
    G = g.ng
    assert np.isclose(Dn[0, 0], 0.5 * (F["D1"][9 + G, 8 + G] + F["D1"][10 + G, 8 + G]))
    assert np.isclose(Dn[0, 1], 0.5 * (F["D2"][10 + G, 7 + G] + F["D2"][10 + G, 8 + G]))
    assert np.isclose(Dn[0, 2], F["D3"][10 + G, 8 + G])
    assert np.isclose(Bn[0, 2], 0.25 * F["B3"][9 + G:11 + G, 7 + G:9 + G].sum())


# ------------------------------------------------------------------------------ deposit
def _moved_particles(O, g, rng, n, max_move=0.9, charge=-1.0):
    i1 = rng.integers(2, g.n1 - 2, n); i2 = rng.integers(2, g.n2 - 2, n)
    dx1 = rng.random(n); dx2 = rng.random(n)
    m1 = rng.uniform(-max_move, max_move, n); m2 = rng.uniform(-max_move, max_move, n)
    y1 = i1 + dx1 + m1; y2 = i2 + dx2 + m2
    j1 = np.floor(y1).astype(np.int32); j2 = np.floor(y2).astype(np.int32)
    p = O.Particles(i1=j1, i2=j2, dx1=y1 - j1, dx2=y2 - j2, u1=rng.normal(size=n) * 0.1, u2=rng.normal(size=n) * 0.1,
                    u3=rng.normal(size=n) * 2, weight=rng.uniform(0.5, 2.0, n), tag=np.ones(n),
                    i1_prev=i1, i2_prev=i2, dx1_prev=dx1, dx2_prev=dx2, q_over_m=charge, charge=charge)
    return p


def _node_charge(g, i, dx, j, dy, qw):
    """rho~ = q w S on nodes with the linear (cloud-in-cell) shape."""
    rho = np.zeros(g.shape)
    G = g.ng
    for a, wa in ((0, 1 - dx), (1, dx)):
        for b, wb in ((0, 1 - dy), (1, dy)):
            np.add.at(rho, (i + a + G, j + b + G), qw * wa * wb)
    return rho


def test_deposit_satisfies_discrete_continuity(O, g):
    """Eq. 32/34: [rho~(n+1) - rho~(n)]/dt + d_1 J^1 + d_2 J^2 = 0 at every node, to rounding."""
    rng = np.random.default_rng(5)
    p = _moved_particles(O, g, rng, 3000)
    dt = 0.37
    J, over = O.deposit(g, p, dt)
    assert over == 0
    qw = p.charge * p.weight
    rho0 = _node_charge(g, p.i1_prev, p.dx1_prev, p.i2_prev, p.dx2_prev, qw)
    rho1 = _node_charge(g, p.i1, p.dx1, p.i2, p.dx2, qw)
    J1, J2 = J["J1"], J["J2"]
    div = np.zeros(g.shape)
    div[1:, :] += J1[1:, :] - J1[:-1, :]        # J1(i+1/2,j) - J1(i-1/2,j)
    div[:, 1:] += J2[:, 1:] - J2[:, :-1]
    res = (rho1 - rho0) / dt + div
    assert np.max(np.abs(res[1:, 1:])) < 1e-11 * np.max(np.abs(J1))


def test_deposit_first_moments(O, g):
    rng = np.random.default_rng(6)
    p = _moved_particles(O, g, rng, 2000)
    dt = 0.5
    J, _ = O.deposit(g, p, dt)
    qw = p.charge * p.weight
    d1 = (p.i1 + p.dx1) - (p.i1_prev + p.dx1_prev)
    d2 = (p.i2 + p.dx2) - (p.i2_prev + p.dx2_prev)
    assert np.isclose(J["J1"].sum(), np.sum(qw * d1) / dt, rtol=1e-12)
    assert np.isclose(J["J2"].sum(), np.sum(qw * d2) / dt, rtol=1e-12)
    # Eq. 36: sum J3 = sum q w (alpha/gamma)(h^13 u_1 + h^33 u_3) at the path midpoint
    xm1 = 0.5 * ((p.i1 + p.dx1) + (p.i1_prev + p.dx1_prev)); xm2 = 0.5 * ((p.i2 + p.dx2) + (p.i2_prev + p.dx2_prev))
    m = O.metric(g, xm1, xm2, derivs=False)
    gam = np.sqrt(1 + m["hu11"] * p.u1 ** 2 + m["hu22"] * p.u2 ** 2 + m["hu33"] * p.u3 ** 2 + 2 * m["hu13"] * p.u1 * p.u3)
    v3 = m["alpha"] / gam * (m["hu13"] * p.u1 + m["hu33"] * p.u3)
    assert np.isclose(J["J3"].sum(), np.sum(qw * v3), rtol=1e-12)


def test_deposit_single_cell_hand_formula(O, g):
    """One particle that stays inside cell (5,6): four-point formula, midpoint weights."""
    p = O.Particles(i1=[5], i2=[6], dx1=[0.7], dx2=[0.4], u1=[0.0], u2=[0.0], u3=[0.0], weight=[2.0], tag=[1],
                    i1_prev=[5], i2_prev=[6], dx1_prev=[0.2], dx2_prev=[0.9], q_over_m=1.0, charge=1.5)
    dt = 0.25
    J, _ = O.deposit(g, p, dt)
    G = g.ng
    F1 = 1.5 * 2.0 * (0.7 - 0.2) / dt; F2 = 1.5 * 2.0 * (0.4 - 0.9) / dt
    W1 = 0.45; W2 = 0.65
    assert np.isclose(J["J1"][5 + G, 6 + G], F1 * (1 - W2)) and np.isclose(J["J1"][5 + G, 7 + G], F1 * W2)
    assert np.isclose(J["J2"][5 + G, 6 + G], F2 * (1 - W1)) and np.isclose(J["J2"][6 + G, 6 + G], F2 * W1)
    assert np.count_nonzero(J["J1"]) == 2 and np.count_nonzero(J["J2"]) == 2 and np.count_nonzero(J["J3"]) == 0


def _v3_schwarzschild(g, x1, x2, u3):
    """Eq. 36 velocity (alpha/gamma) h^33 u_3 for a = 0, u_1 = u_2 = 0, from the textbook Schwarzschild
    Kerr-Schild closed forms alpha = (1 + 2/r)^-1/2, h^{phi phi} = 1/(r sin theta)^2 (not from the oracle's metric)."""
    r = g.r_min * (g.r_max / g.r_min) ** (x1 / g.n1)          # log-r map
    th = x2 * np.pi / g.n2
    h33 = 1.0 / (r * np.sin(th)) ** 2
    return (1.0 + 2.0 / r) ** -0.5 / np.sqrt(1.0 + h33 * u3 * u3) * h33 * u3


def test_deposit_j3_node_weights_one_cell_hand_formula(O):
    """Eq. 36 with J^3 located like D^3 on the nodes (i, j), reading R-S10: a particle that
    stays in cell (5, 6) with u_3 != 0; the relay point is the midpoint of the path, each of the two half paths carries
    q w v^3 / 2 (v^3 at the midpoint of the whole path) and puts (1-W1)(1-W2) of it on node (5, 6), W1 (1-W2) on
    (6, 6), (1-W1) W2 on (5, 7) and W1 W2 on (6, 7), W = offsets of the half path's own midpoint.  W1 != W2
    everywhere, so that a transposed node or swapped weights fail."""
    gs = O.Grid(24, 16, 0.0, 2.2, 20.0)                        # a = 0
    xa, ya, xb, yb, u3, q, w, dt = 0.2, 0.9, 0.7, 0.5, 1.7, 1.5, 2.0, 0.25
    p = O.Particles(i1=[5], i2=[6], dx1=[xb], dx2=[yb], u1=[0.0], u2=[0.0], u3=[u3], weight=[w], tag=[1],
                    i1_prev=[5], i2_prev=[6], dx1_prev=[xa], dx2_prev=[ya], q_over_m=1.0, charge=q)
    J, _ = O.deposit(gs, p, dt)
    G = gs.ng
    xm, ym = 0.45, 0.70                                         # midpoint of the path = relay point
    F3 = 0.5 * q * w * _v3_schwarzschild(gs, 5 + xm, 6 + ym, u3)
    halves = ((0.5 * (xa + xm), 0.5 * (ya + ym)), (0.5 * (xm + xb), 0.5 * (ym + yb)))   # (0.325, 0.8), (0.575, 0.6)
    want = {(5, 6): sum(F3 * (1 - W1) * (1 - W2) for W1, W2 in halves),
            (6, 6): sum(F3 * W1 * (1 - W2) for W1, W2 in halves),
            (5, 7): sum(F3 * (1 - W1) * W2 for W1, W2 in halves),
            (6, 7): sum(F3 * W1 * W2 for W1, W2 in halves)}
    assert len({round(v / F3, 12) for v in want.values()}) == 4      # four different weights
    for (i, j), v in want.items():
        assert np.isclose(J["J3"][i + G, j + G], v, rtol=1e-12, atol=0), (i, j)
    assert np.count_nonzero(J["J3"]) == 4
    assert np.isclose(J["J3"].sum(), 2 * F3, rtol=1e-13)


def test_deposit_j3_node_weights_across_a_face_hand_formula(O):
    """The same for a path from cell (5, 6) into cell (6, 6) (R-S10): relay point on the face x1 = 6; each of the two
    segments carries half of q w v^3 (v^3 at the midpoint of the whole path), spread bilinearly on the four nodes
    of ITS cell with the offsets of ITS midpoint."""
    gs = O.Grid(24, 16, 0.0, 2.2, 20.0)
    xa, ya, xb, yb, u3, q, w, dt = 0.8, 0.3, 0.1, 0.5, -0.9, -1.0, 3.0, 0.4     # xb is in cell 6: x = 6.1
    p = O.Particles(i1=[6], i2=[6], dx1=[xb], dx2=[yb], u1=[0.0], u2=[0.0], u3=[u3], weight=[w], tag=[1],
                    i1_prev=[5], i2_prev=[6], dx1_prev=[xa], dx2_prev=[ya], q_over_m=1.0, charge=q)
    J, _ = O.deposit(gs, p, dt)
    G = gs.ng
    # path (5.8, 6.3) -> (6.1, 6.5); relay: x1 = 6 (the face), x2 = midpoint 6.4 (no face crossed along x2)
    F3 = 0.5 * q * w * _v3_schwarzschild(gs, 0.5 * (5.8 + 6.1), 0.5 * (6.3 + 6.5), u3)
    want = np.zeros(gs.shape)
    for (c1, W1, W2) in ((5, 0.5 * (0.8 + 1.0), 0.5 * (0.3 + 0.4)),        # segment 1 in cell (5, 6)
                         (6, 0.5 * (0.0 + 0.1), 0.5 * (0.4 + 0.5))):       # segment 2 in cell (6, 6)
        want[c1 + G, 6 + G] += F3 * (1 - W1) * (1 - W2)
        want[c1 + 1 + G, 6 + G] += F3 * W1 * (1 - W2)
        want[c1 + G, 7 + G] += F3 * (1 - W1) * W2
        want[c1 + 1 + G, 7 + G] += F3 * W1 * W2
    assert np.allclose(J["J3"], want, rtol=1e-12, atol=1e-18)
    assert np.count_nonzero(J["J3"]) == 6
    # J^1 of the same path: all of it through the face-normal edge samples J1(5+1/2, .) and J1(6+1/2, .)
    F1a, F1b = q * w * (1.0 - 0.8) / dt, q * w * 0.1 / dt
    assert np.isclose(J["J1"][5 + G, 6 + G], F1a * (1 - 0.35)) and np.isclose(J["J1"][5 + G, 7 + G], F1a * 0.35)
    assert np.isclose(J["J1"][6 + G, 6 + G], F1b * (1 - 0.45)) and np.isclose(J["J1"][6 + G, 7 + G], F1b * 0.45)


def test_deposit_skips_dead_zero_charge_and_oversteps(O, g):
    rng = np.random.default_rng(7)
    p = _moved_particles(O, g, rng, 100)
    p.tag[:50] = 0
    q = p.copy(); q.tag[:] = 1
    for k in ("i1", "i2", "dx1", "dx2", "u1", "u2", "u3", "weight", "tag", "i1_prev", "i2_prev", "dx1_prev", "dx2_prev"):
        setattr(q, k, getattr(q, k)[50:].copy())
    Ja, _ = O.deposit(g, p, 0.3); Jb, _ = O.deposit(g, q, 0.3)
    for k in Ja:
        assert np.array_equal(Ja[k], Jb[k])
    p.i1[60] = p.i1_prev[60] + 2
    Jc, over = O.deposit(g, p, 0.3)
    assert over == 1
    p.charge = 0.0
    Jd, over = O.deposit(g, p, 0.3)
    assert over == 0 and all(np.count_nonzero(v) == 0 for v in Jd.values())


def test_push_then_deposit_conserves_charge_through_reflection_and_absorption(O, W):
    """Whole path on a tiny magnetosphere: continuity holds with rho~ taken over the particles
    that are alive after the step (dead ones deposit nothing: R-S10)."""
    wl = W.config_tiny(shrink=4)
    from helpers import grid_from_domain, oracle_particles
    g = grid_from_domain(O, wl.dom)
    sp = wl.species[0]
    p = oracle_particles(O, sp)
    O.push(g, p, wl.fields, wl.dt)
    assert (p.tag == 0).sum() > 0
    J, over = O.deposit(g, p, wl.dt)
    assert over == 0
    al = p.tag == 1
    qw = p.charge * p.weight[al]
    rho0 = _node_charge(g, p.i1_prev[al], p.dx1_prev[al], p.i2_prev[al], p.dx2_prev[al], qw)
    rho1 = _node_charge(g, p.i1[al], p.dx1[al], p.i2[al], p.dx2[al], qw)
    div = np.zeros(g.shape)
    div[1:, :] += J["J1"][1:, :] - J["J1"][:-1, :]
    div[:, 1:] += J["J2"][:, 1:] - J["J2"][:, :-1]
    res = (rho1 - rho0) / wl.dt + div
    assert np.max(np.abs(res[1:, 1:])) < 1e-11 * np.max(np.abs(J["J1"]))


def test_sort_reference_keys(O, g):
    rng = np.random.default_rng(9)
    n = 5000
    p = O.Particles(i1=rng.integers(0, g.n1, n), i2=rng.integers(0, g.n2, n), dx1=rng.random(n), dx2=rng.random(n),
                    u1=rng.normal(size=n), u2=rng.normal(size=n), u3=rng.normal(size=n), weight=np.ones(n),
                    tag=(rng.random(n) > 0.1))
    q, perm, keys = O.sort_reference(g, p, tile=8)
    assert np.all(np.diff(keys) >= 0)
    assert np.array_equal(np.sort(perm), np.arange(n))
    nd = int((p.tag == 0).sum())
    assert np.all(q.tag[n - nd:] == 0) and np.all(q.tag[:n - nd] == 1)
    # key is a bijection cell <-> key on alive particles, tile-major
    key, dead = O.sort_key(g, p.i1, p.i2, np.ones(n), 8)
    cells = p.i1.astype(np.int64) * g.n2 + p.i2
    assert len(np.unique(key)) == len(np.unique(cells)) and key.max() < dead
