"""Pins for oracle S1-S3 (metric, derivatives, tetrads) — nothing here re-types the oracle's
formula for the quantity it pins: inverses, determinants, limits and finite differences."""
import numpy as np
import pytest

PTS = [(3.2, 7.9), (60.5, 31.7), (100.1, 3.3), (10.0, 60.2), (120.9, 32.0)]


@pytest.fixture(scope="module", params=["log_uniform", "offset_stretched", "linear_r"])
def g(O, request):
    """The map of the five configs (A.3 with r0 = 0, h0 = 0) and the full A.3 map: radial offset
    r0 = 0.6 and polar stretch h0 = 0.35; every pin below that does not name the map holds for both."""
    if request.param == "log_uniform":
        return O.Grid(128, 64, 0.95, 0.9 * (1 + np.sqrt(1 - 0.95 ** 2)), 20.0)
    if request.param == "linear_r":                     # spherical Kerr-Schild of App. A.2
        return O.Grid(128, 64, 0.95, 0.9 * (1 + np.sqrt(1 - 0.95 ** 2)), 20.0, linear_r=1)
    return O.Grid(128, 64, 0.95, 0.9 * (1 + np.sqrt(1 - 0.95 ** 2)), 20.0, r0=0.6, h0=0.35)


def _mat(m, k, up):
    p = "hu" if up else "hd"
    return np.array([[m[p + "11"][k], 0, m[p + "13"][k]], [0, m[p + "22"][k], 0], [m[p + "13"][k], 0, m[p + "33"][k]]])


def test_inverse_and_determinant(O, g):
    x1, x2 = np.array(PTS).T
    m = O.metric(g, x1, x2)
    for k in range(len(PTS)):
        hd, hu = _mat(m, k, False), _mat(m, k, True)
        assert np.allclose(hd @ hu, np.eye(3), atol=1e-13)
        assert np.isclose(m["sqrt_h"][k], np.sqrt(np.linalg.det(hd)), rtol=1e-13)


def test_four_metric_relations(O, g):
    """g^00 = -1/alpha^2 = -(1+z); g^01 = beta^1/alpha^2 = z; g^11 = h^11 - (beta^1)^2/alpha^2 = Delta/Sigma (A1)."""
    x1, x2 = np.array(PTS).T
    m = O.metric(g, x1, x2)
    assert np.allclose(1 / m["alpha"] ** 2, 1 + m["z"], rtol=1e-14)
    assert np.allclose(m["beta1"] * m["s1"] / m["alpha"] ** 2, m["z"], rtol=1e-14)
    g11 = (m["hu11"] - m["beta1"] ** 2 / m["alpha"] ** 2) * m["s1"] ** 2
    assert np.allclose(g11, m["Delta"] / m["Sigma"], rtol=1e-12, atol=1e-14)
    # beta_i beta^i = z^2/(1+z)
    assert np.allclose(m["hd11"] * m["beta1"] ** 2, m["z"] ** 2 / (1 + m["z"]), rtol=1e-13)


def test_schwarzschild_limit(O):
    g0 = O.Grid(64, 32, 0.0, 1.5, 30.0)
    x1 = np.array([1.0, 20.5, 60.0]); x2 = np.array([3.3, 16.0, 29.1])
    m = O.metric(g0, x1, x2)
    r = m["r"]
    assert np.allclose(m["hd11"] / m["s1"] ** 2, 1 + 2 / r, rtol=1e-14)
    assert np.allclose(m["alpha"], (1 + 2 / r) ** -0.5, rtol=1e-14)
    assert np.allclose(m["beta1"] * m["s1"], 2 / (r + 2), rtol=1e-14)
    assert np.allclose(m["hd22"] / m["s2"] ** 2, r * r, rtol=1e-14)
    assert np.allclose(m["hd33"], r * r * np.sin(m["th"]) ** 2, rtol=1e-14)
    assert np.all(m["hd13"] == 0) and np.all(m["hu13"] == 0)


def test_coordinate_map(O, g):
    m = O.metric(g, np.array([0.0, 128.0, 64.0]), np.array([32.0, 32.0, 16.0]))
    # xi = log(r - r0) is uniform in x1: the middle of the grid is the geometric mean of (r - r0); A.2: the arithmetic mean
    mid = 0.5 * (g.r_min + g.r_max) if g.linear_r else g.r0 + np.sqrt((g.r_min - g.r0) * (g.r_max - g.r0))
    assert np.allclose(m["r"], [g.r_min, g.r_max, mid], rtol=1e-14)
    # theta(eta) of P:821 at eta = pi/2 and pi/4: pi/2 (fixed point of the stretch) and pi/4 + 2 h0 (pi/4)(pi/2)(3pi/4)/pi^2
    assert np.allclose(m["th"], [np.pi / 2, np.pi / 2, np.pi / 4 * (1 + 0.75 * g.h0)], rtol=1e-14)


def test_scale_factors_are_the_map_derivatives(O, g):
    """s1 = dr/dx1 and s2 = dtheta/dx2 (what "dr", "dtheta" of the code basis mean):
    finite differences of the map itself; and the stretch keeps theta symmetric about the equator,
    monotonic, with theta(0) = 0, theta(pi) = pi."""
    x1, x2 = np.array(PTS).T
    h = 1e-3
    f = lambda a, b, k: O.metric(g, a, b, derivs=False)[k]
    s1_fd = (-f(x1 + 2 * h, x2, "r") + 8 * f(x1 + h, x2, "r") - 8 * f(x1 - h, x2, "r") + f(x1 - 2 * h, x2, "r")) / (12 * h)
    s2_fd = (-f(x1, x2 + 2 * h, "th") + 8 * f(x1, x2 + h, "th") - 8 * f(x1, x2 - h, "th") + f(x1, x2 - 2 * h, "th")) / (12 * h)
    m = O.metric(g, x1, x2, derivs=False)
    assert np.allclose(m["s1"], s1_fd, rtol=1e-10) and np.allclose(m["s2"], s2_fd, rtol=1e-10)
    gg = O.Grid(g.n1, g.n2, g.a, g.r_min, g.r_max, small_angle=0.0, r0=g.r0, h0=g.h0)
    x = np.linspace(0.0, g.n2, 257)
    th = O.metric(gg, np.full_like(x, 5.0), x, derivs=False)["th"]
    assert abs(th[0]) < 1e-15 and abs(th[-1] - np.pi) < 1e-14
    assert np.all(np.diff(th) > 0) and np.allclose(th + th[::-1], np.pi, atol=1e-14)


def test_small_angle_clamp(O, g):
    m = O.metric(g, np.array([10.0] * 4), np.array([0.0, -0.3, 64.0, 64.2]))
    assert np.allclose(m["th"], [1e-5, 1e-5, np.pi - 1e-5, np.pi - 1e-5], rtol=0, atol=1e-18)
    assert np.all(np.isfinite(m["hu33"]))


def test_derivatives_vs_finite_differences(O, g):
    """Central differences of the metric itself (4th order, h = 1e-2 cell)."""
    x1, x2 = np.array(PTS).T
    m = O.metric(g, x1, x2)
    h = 1e-2

    def fd(name, axis):
        def f(s):
            return O.metric(g, x1 + (s if axis == 0 else 0), x2 + (s if axis == 1 else 0), derivs=False)[name]
        return (-f(2 * h) + 8 * f(h) - 8 * f(-h) + f(-2 * h)) / (12 * h)

    for name in ("hu11", "hu22", "hu33", "hu13", "alpha", "beta1"):
        for axis in (0, 1):
            an = m["d%d_%s" % (axis + 1, name)]
            nu = fd(name, axis)
            scale = np.abs(m[name]) * (0.02 if axis == 0 else 0.05) + 1e-300
            assert np.all(np.abs(an - nu) <= 1e-8 * scale + 1e-9 * np.abs(nu)), (name, axis, an, nu)


def test_tetrad_roundtrip_and_orthonormality(O, g):
    rng = np.random.default_rng(1)
    for (x1, x2) in PTS:
        m = O.metric(g, x1, x2)
        hd, hu = _mat(m, 0, False), _mat(m, 0, True)
        v = rng.normal(size=3)
        vh = O.cntrv_to_tetrad(g, x1, x2, v)
        assert np.isclose(vh @ vh, v @ hd @ v, rtol=1e-13)              # e^T h e = 1
        assert np.allclose(O.tetrad_to_cntrv(g, x1, x2, vh), v, rtol=1e-12, atol=1e-14)
        w = rng.normal(size=3)
        wh = O.cov_to_tetrad(g, x1, x2, w)
        assert np.isclose(wh @ wh, w @ hu @ w, rtol=1e-13)
        assert np.allclose(O.tetrad_to_cov(g, x1, x2, wh), w, rtol=1e-12, atol=1e-14)
        assert np.isclose(vh @ wh, v @ w, rtol=1e-12)                    # contraction is frame independent
