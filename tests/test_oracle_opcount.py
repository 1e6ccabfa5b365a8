"""The operation count of the method as the oracle states it ("an exact count from an operation-counting
scalar type in the oracle"): oracle/grpic_oracle.c compiled on oracle/orc_count.hpp.  The counting build must BE the
oracle (bit-identical results), its loop stages must scale with n_iter exactly, and the table is printed."""
import numpy as np

from helpers import grid_from_domain, oracle_particles


def _sample(O, W, n_iter=10):
    wl = W.config_large(shrink=64)
    g = grid_from_domain(O, wl.dom, n_iter=n_iter)
    p = oracle_particles(O, wl.species[0], np.float32)
    return wl, g, p


def test_counting_build_is_the_oracle_and_counts_scale_with_n_iter(O, W):
    wl, g, p = _sample(O, W)
    c10 = O.count_ops(g, p, wl.fields, wl.dt)
    assert c10["particles"] == int(p.tag.sum()) and c10["n_iter"] == 10
    # same arithmetic: the counting type wraps a double and does the same operations in the same order
    import ctypes as C
    L = C.CDLL(O.build_count())
    q, r = p.copy(), p.copy()
    O.push(g, q, wl.fields, wl.dt)
    Jq, _ = O.deposit(g, q, wl.dt)
    gc, rc = g.c(), r.c()
    Jr = {k: np.zeros(g.shape) for k in ("J1", "J2", "J3")}
    jc = O._Current(*[O._ptr(Jr[k], O._dp) for k in ("J1", "J2", "J3")])
    fc, keep = O._fields_c(wl.fields)
    out = np.zeros((len(O.COUNT_STAGES), len(O.COUNT_KINDS)), np.int64); n = C.c_int64(0); dt = C.c_double(wl.dt)
    L.orc_count_step(C.byref(gc), C.byref(rc), C.byref(fc), C.byref(jc), C.byref(dt), out.ctypes.data_as(C.c_void_p), C.byref(n))
    for k in ("i1", "i2", "dx1", "dx2", "u1", "u2", "u3", "phi", "tag"):
        assert np.array_equal(getattr(q, k), getattr(r, k)), k
    for k in Jq:                                     # the plain build sums per-thread partial grids: same up to the order
        assert np.allclose(Jq[k], Jr[k], rtol=0, atol=1e-12 * np.abs(Jq[k]).max()), k
    # the two fixed-point loops execute exactly n_iter (+1 for phi) applications of their maps
    _, g5, _ = _sample(O, W, n_iter=5)
    c5 = O.count_ops(g5, p, wl.fields, wl.dt)
    su, sx = O.COUNT_STAGES[3], O.COUNT_STAGES[4]
    per_u = (c10["per_stage"][su] - c5["per_stage"][su]) / 5
    per_x = (c10["per_stage"][sx] - c5["per_stage"][sx]) / 5
    assert abs(c10["per_stage"][su] - 10 * per_u) < 1e-9 * c10["per_stage"][su] + 1.0
    assert abs(c10["per_stage"][sx] - 11 * per_x) < 0.02 * c10["per_stage"][sx]      # + phi: one more metric evaluation
    for st in O.COUNT_STAGES:
        if st not in (su, sx):
            assert abs(c10["per_stage"][st] - c5["per_stage"][st]) < 0.5 + 1e-3 * c10["per_stage"][st], st
    print()
    print(f"operations per particle update, oracle as written, n_iter = 10 ({c10['particles']} particles):")
    for st in O.COUNT_STAGES:
        kinds = ", ".join(f"{k} {v:.1f}" for k, v in c10["per_update"][st].items() if v > 0)
        print(f"  {st:52s} {c10['per_stage'][st]:8.1f}   ({kinds})")
    print(f"  {'total':52s} {c10['total_per_update']:8.1f}   (per momentum iteration {per_u:.1f}, per coordinate iteration {per_x:.1f})")
    assert 2000 < c10["total_per_update"] < 5000
