"""ctypes binding of oracle/grpic_oracle.c — TEST INFRASTRUCTURE, not the product path.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It never imports the CUDA package.

The C file is the oracle (plain FP64 statement of PAPER.md Sec. 3.1-3.2); this module
only marshals numpy arrays.  Written in numpy here: `sort_reference` (the sort is not in
the paper, its key is defined by include/grpic.h, DESIGN.md R-S9), the time-level sequencing
`fields_prepare` / `fields_advance` (Sec. 3.4) around the C field operators, and the boundary
side `field_bc`, `filter_current`, `field_match` (Sec. 3.3.3).
Parity unpinned (forms the paper defers to paper I; only their behaviour is pinned): the choice
of digital filter in `filter_current` (R-F5) and the profile of `field_match` (R-F6).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "grpic_oracle.c")
_LIB = os.path.join(_HERE, "libgrpic_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_LIB_COUNT = os.path.join(_HERE, "libgrpic_oracle_count.so")
COUNT_STAGES = ("interpolation (S4)", "metric + 12 derivatives at x^n (S1, S2)", "tetrad projections + 2 Boris halves (S3, S5)",
                "momentum loop Eq. 26-27 (S6)", "coordinate loop Eq. 28-29 + phi Eq. 30 (S7, S8)",
                "renormalise + particle BCs (S9)", "deposit incl. v^3 at the path midpoint (S10)", "other")
COUNT_KINDS = ("add/sub", "mul", "div", "sqrt", "exp/log", "sin/cos", "floor", "min/max", "compare", "neg/abs")


def build_count(force: bool = False) -> str:
    """The same C source compiled as C++ on the operation-counting stand-in for double (oracle/orc_count.hpp)."""
    deps = [_SRC, os.path.join(_HERE, "orc_count.hpp")]
    if force or not os.path.exists(_LIB_COUNT) or any(os.path.getmtime(_LIB_COUNT) < os.path.getmtime(d) for d in deps):
        cmd = ["g++", "-x", "c++", "-O1", "-std=gnu++17", "-ffp-contract=off", "-DORC_COUNT", "-shared", "-fPIC", _SRC,
               "-o", _LIB_COUNT, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB_COUNT


def count_ops(g: "Grid", p: "Particles", fields, dt: float) -> dict:
    """Operations the oracle, as written, executes for one push + deposit of the alive particles of a COPY of `p`:
    {"per_update": {stage: {kind: count per particle}}, "total_per_update": float, "particles": n}.
    Every +, -, *, /, sqrt, exp, log, sin, cos, floor, fmin/fmax, comparison and negation on a real number counts 1."""
    L = C.CDLL(build_count())
    q = p.copy()
    gc = g.c(); pc = q.c()
    J = {k: np.zeros(g.shape) for k in ("J1", "J2", "J3")}
    jc = _Current(*[_ptr(J[k], _dp) for k in ("J1", "J2", "J3")])
    out = np.zeros((len(COUNT_STAGES), len(COUNT_KINDS)), np.int64)
    n = C.c_int64(0)
    dtc = C.c_double(dt)
    if fields is None:
        L.orc_count_step(C.byref(gc), C.byref(pc), None, C.byref(jc), C.byref(dtc), out.ctypes.data_as(C.c_void_p), C.byref(n))
    else:
        fc, keep = _fields_c(fields)
        L.orc_count_step(C.byref(gc), C.byref(pc), C.byref(fc), C.byref(jc), C.byref(dtc), out.ctypes.data_as(C.c_void_p), C.byref(n))
    npart = max(1, int(n.value))
    per = {st: {kd: out[i, j] / npart for j, kd in enumerate(COUNT_KINDS)} for i, st in enumerate(COUNT_STAGES)}
    return {"per_update": per, "per_stage": {st: float(out[i].sum()) / npart for i, st in enumerate(COUNT_STAGES)},
            "total_per_update": float(out.sum()) / npart, "particles": int(n.value), "n_iter": g.n_iter}


class _Grid(C.Structure):
    _fields_ = [("n1", C.c_int32), ("n2", C.c_int32), ("ng", C.c_int32), ("n_iter", C.c_int32),
                ("a", C.c_double), ("r_min", C.c_double), ("r_max", C.c_double), ("small_angle", C.c_double),
                ("r0", C.c_double), ("h0", C.c_double), ("linear_r", C.c_int32),
                ("mass", C.c_double)]


_METRIC_NAMES = ["r", "th", "sth", "cth", "Sigma", "Delta", "A", "z", "s1", "s2", "alpha", "beta1",
                 "hu11", "hu22", "hu33", "hu13", "hd11", "hd22", "hd33", "hd13", "sqrt_h", "dls2"]
_DMETRIC_NAMES = ["hu11", "hu22", "hu33", "hu13", "alpha", "beta1"]

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_bp = C.POINTER(C.c_uint8)


class _Fields(C.Structure):
    _fields_ = [(k, _dp) for k in ("D1", "D2", "D3", "B1", "B2", "B3")]


class _Current(C.Structure):
    _fields_ = [(k, _dp) for k in ("J1", "J2", "J3")]


class _Particles(C.Structure):
    _fields_ = [("n", C.c_int64), ("i1", _ip), ("i2", _ip), ("dx1", _dp), ("dx2", _dp),
                ("u1", _dp), ("u2", _dp), ("u3", _dp), ("phi", _dp),
                ("i1_prev", _ip), ("i2_prev", _ip), ("dx1_prev", _dp), ("dx2_prev", _dp),
                ("weight", _dp), ("tag", _bp),
                ("q_over_m", C.c_double), ("charge", C.c_double), ("massive", C.c_int32)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_num_threads.restype = C.c_int
    return _lib


@dataclass
class Grid:
    n1: int
    n2: int
    a: float
    r_min: float
    r_max: float
    ng: int = 2
    n_iter: int = 10
    small_angle: float = 1e-5
    r0: float = 0.0          # A.3 radial offset, xi = log(r - r0)
    h0: float = 0.0          # A.3 polar stretch
    linear_r: int = 0        # 1: A.2 map, r uniform in x1
    mass: float = 1.0        # M/r_g; 0 (with a = 0) = flat spherical kerr_schild_0 of A.1

    def c(self) -> _Grid:
        return _Grid(self.n1, self.n2, self.ng, self.n_iter, self.a, self.r_min, self.r_max, self.small_angle,
                     self.r0, self.h0, self.linear_r, self.mass)

    @property
    def shape(self):
        return (self.n1 + 2 * self.ng, self.n2 + 2 * self.ng)


def _f64(x):
    return np.ascontiguousarray(x, dtype=np.float64)


def _ptr(a, t):
    return a.ctypes.data_as(t)


@dataclass
class Particles:
    """FP64 SoA particle columns (same columns as include/grpic.h)."""
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
    i1_prev: np.ndarray = field(default=None)
    i2_prev: np.ndarray = field(default=None)
    dx1_prev: np.ndarray = field(default=None)
    dx2_prev: np.ndarray = field(default=None)
    q_over_m: float = 0.0
    charge: float = 0.0
    massive: int = 1

    def __post_init__(self):
        for k in ("i1", "i2"):
            setattr(self, k, np.ascontiguousarray(getattr(self, k), dtype=np.int32).copy())
        for k in ("dx1", "dx2", "u1", "u2", "u3", "weight"):
            setattr(self, k, _f64(getattr(self, k)).copy())
        self.tag = np.ascontiguousarray(self.tag, dtype=np.uint8).copy()
        if self.phi is not None:
            self.phi = _f64(self.phi).copy()
        n = self.i1.size
        self.i1_prev = np.zeros(n, np.int32) if self.i1_prev is None else np.ascontiguousarray(self.i1_prev, np.int32).copy()
        self.i2_prev = np.zeros(n, np.int32) if self.i2_prev is None else np.ascontiguousarray(self.i2_prev, np.int32).copy()
        self.dx1_prev = np.zeros(n) if self.dx1_prev is None else _f64(self.dx1_prev).copy()
        self.dx2_prev = np.zeros(n) if self.dx2_prev is None else _f64(self.dx2_prev).copy()

    @property
    def n(self):
        return self.i1.size

    def copy(self) -> "Particles":
        return Particles(**{k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in self.__dict__.items()})

    def c(self) -> _Particles:
        return _Particles(self.n, _ptr(self.i1, _ip), _ptr(self.i2, _ip), _ptr(self.dx1, _dp), _ptr(self.dx2, _dp),
                          _ptr(self.u1, _dp), _ptr(self.u2, _dp), _ptr(self.u3, _dp),
                          _ptr(self.phi, _dp) if self.phi is not None else None,
                          _ptr(self.i1_prev, _ip), _ptr(self.i2_prev, _ip), _ptr(self.dx1_prev, _dp),
                          _ptr(self.dx2_prev, _dp), _ptr(self.weight, _dp), _ptr(self.tag, _bp),
                          float(self.q_over_m), float(self.charge), int(self.massive))


def _fields_c(fields):
    arrs = [_f64(fields[k]) for k in ("D1", "D2", "D3", "B1", "B2", "B3")]
    return _Fields(*[_ptr(a, _dp) for a in arrs]), arrs


def metric(g: Grid, x1, x2, derivs: bool = True):
    """All S1 quantities (and S2 derivatives) at code coordinates (x1, x2)."""
    x1 = _f64(np.atleast_1d(x1)); x2 = _f64(np.atleast_1d(x2))
    n = x1.size
    m = np.zeros((n, len(_METRIC_NAMES)))
    d = np.zeros((n, len(_DMETRIC_NAMES), 2))
    gc = g.c()
    lib().orc_metric_many(C.byref(gc), C.c_int64(n), _ptr(x1, _dp), _ptr(x2, _dp), _ptr(m, _dp),
                          _ptr(d, _dp) if derivs else None)
    out = {k: m[:, j].copy() for j, k in enumerate(_METRIC_NAMES)}
    if derivs:
        for j, k in enumerate(_DMETRIC_NAMES):
            out["d1_" + k] = d[:, j, 0].copy()
            out["d2_" + k] = d[:, j, 1].copy()
    return out


def _vec3(fn, g, x1, x2, v):
    gc = g.c()
    out = np.zeros(3)
    m = (C.c_double * len(_METRIC_NAMES))()
    lib().orc_metric(C.byref(gc), C.c_double(x1), C.c_double(x2), m)
    vin = _f64(v)
    getattr(lib(), fn)(m, _ptr(vin, _dp), _ptr(out, _dp))
    return out


def cntrv_to_tetrad(g, x1, x2, v): return _vec3("orc_cntrv_to_tetrad", g, x1, x2, v)
def cov_to_tetrad(g, x1, x2, v): return _vec3("orc_cov_to_tetrad", g, x1, x2, v)
def tetrad_to_cov(g, x1, x2, v): return _vec3("orc_tetrad_to_cov", g, x1, x2, v)
def tetrad_to_cntrv(g, x1, x2, v): return _vec3("orc_tetrad_to_cntrv", g, x1, x2, v)


def interp(g: Grid, fields, i1, i2, dx1, dx2):
    fc, keep = _fields_c(fields)
    i1 = np.ascontiguousarray(i1, np.int32); i2 = np.ascontiguousarray(i2, np.int32)
    dx1 = _f64(dx1); dx2 = _f64(dx2)
    n = i1.size
    D = np.zeros((n, 3)); B = np.zeros((n, 3))
    gc = g.c()
    lib().orc_interp_many(C.byref(gc), C.byref(fc), C.c_int64(n), _ptr(i1, _ip), _ptr(i2, _ip),
                          _ptr(dx1, _dp), _ptr(dx2, _dp), _ptr(D, _dp), _ptr(B, _dp))
    return D, B


def push(g: Grid, p: Particles, fields, dt: float, diag: dict | None = None):
    """In-place step 1-11 + BCs on `p`.  Returns (alive, absorbed_in, absorbed_out).
    If `diag` is a dict it receives 'del1', 'del2': the raw displacement of Eq. 28-29 per particle."""
    gc = g.c(); pc = p.c()
    cnt = (C.c_int64 * 3)()
    if diag is not None:
        diag["del1"] = np.zeros(p.n); diag["del2"] = np.zeros(p.n)
        lib().orc_set_diag(_ptr(diag["del1"], _dp), _ptr(diag["del2"], _dp))
    try:
        return _push(gc, pc, p, fields, dt, cnt)
    finally:
        if diag is not None:
            lib().orc_set_diag(None, None)


def _push(gc, pc, p, fields, dt, cnt):
    if fields is None:
        assert p.q_over_m == 0.0 or not p.massive, "charged particles need fields"
        lib().orc_push(C.byref(gc), C.byref(pc), None, C.c_double(dt), cnt)
    else:
        fc, keep = _fields_c(fields)
        lib().orc_push(C.byref(gc), C.byref(pc), C.byref(fc), C.c_double(dt), cnt)
    return tuple(int(x) for x in cnt)


def push_given_fields(g: Grid, p: Particles, Dp, Bp, dt: float):
    """Same update with contravariant D,B at each particle supplied ([n,3])."""
    gc = g.c(); pc = p.c()
    Dp = _f64(Dp).reshape(p.n, 3); Bp = _f64(Bp).reshape(p.n, 3)
    lib().orc_push_given_fields(C.byref(gc), C.byref(pc), _ptr(Dp, _dp), _ptr(Bp, _dp), C.c_double(dt))


def deposit(g: Grid, p: Particles, dt: float, J=None):
    """Accumulate into J = dict(J1,J2,J3) (created zeroed if None). Returns (J, n_overstep)."""
    if J is None:
        J = {k: np.zeros(g.shape) for k in ("J1", "J2", "J3")}
    for k in ("J1", "J2", "J3"):
        assert J[k].dtype == np.float64 and J[k].flags.c_contiguous and J[k].shape == g.shape
    jc = _Current(*[_ptr(J[k], _dp) for k in ("J1", "J2", "J3")])
    gc = g.c(); pc = p.c()
    over = C.c_int64(0)
    lib().orc_deposit(C.byref(gc), C.byref(pc), C.c_double(dt), C.byref(jc), C.byref(over))
    return J, int(over.value)


# ----------------------------------------------------------------------------------------------
# Field-solver half: Eq. 42-44 auxiliary fields, Eq. 40 Faraday, Eq. 41/45 Ampere
# ----------------------------------------------------------------------------------------------
def _grid_arr(g, a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.shape == g.shape
    return a


def aux_fields(g: Grid, fields: dict) -> dict:
    """E1,E2,E3 (at the D^i locations) and H1,H2,H3 (at the B^i locations) from D^i, B^i."""
    f = {k: _grid_arr(g, fields[k]) for k in ("D1", "D2", "D3", "B1", "B2", "B3")}
    fc = _Fields(*[_ptr(f[k], _dp) for k in ("D1", "D2", "D3", "B1", "B2", "B3")])
    out = {k: np.zeros(g.shape) for k in ("E1", "E2", "E3", "H1", "H2", "H3")}
    gc = g.c()
    lib().orc_aux_fields(C.byref(gc), C.byref(fc), *[_ptr(out[k], _dp) for k in ("E1", "E2", "E3", "H1", "H2", "H3")])
    return out


def faraday(g: Grid, B: dict, E: dict, dt: float) -> dict:
    """B^i updated in place (dict B1,B2,B3 of float64 arrays) with E_i; returns B."""
    for k in ("B1", "B2", "B3"):
        assert B[k].dtype == np.float64 and B[k].flags.c_contiguous and B[k].shape == g.shape
    gc = g.c()
    lib().orc_faraday(C.byref(gc), *[_ptr(B[k], _dp) for k in ("B1", "B2", "B3")],
                      *[_ptr(_grid_arr(g, E[k]), _dp) for k in ("E1", "E2", "E3")], C.c_double(dt))
    return B


def ampere(g: Grid, D: dict, H: dict, J, dt: float, kJ: float = 4.0 * np.pi) -> dict:
    """D^i updated in place with H_i and the conformal currents J (dict or None); returns D."""
    for k in ("D1", "D2", "D3"):
        assert D[k].dtype == np.float64 and D[k].flags.c_contiguous and D[k].shape == g.shape
    Hs = [_grid_arr(g, H[k]) for k in ("H1", "H2", "H3")]
    Js = [None] * 3 if J is None else [_grid_arr(g, J[k]) for k in ("J1", "J2", "J3")]
    gc = g.c()
    lib().orc_ampere(C.byref(gc), *[_ptr(D[k], _dp) for k in ("D1", "D2", "D3")], *[_ptr(h, _dp) for h in Hs],
                     *[None if j is None else _ptr(j, _dp) for j in Js], C.c_double(kJ), C.c_double(dt))
    return D


def sqrt_h(g: Grid, x1, x2):
    """sqrt(h) at arbitrary code positions, axis not clamped (field side)."""
    gg = Grid(g.n1, g.n2, g.a, g.r_min, g.r_max, g.ng, g.n_iter, 0.0, g.r0, g.h0, g.linear_r, g.mass)
    m = metric(gg, x1, x2, derivs=False)
    return m["sqrt_h"]


def num_threads() -> int:
    return int(lib().orc_num_threads())


def set_num_threads(n: int):
    lib().orc_set_num_threads(C.c_int(n))


# ----------------------------------------------------------------------------------------------
# Sort reference (not in the paper; key defined in include/grpic.h, DESIGN.md R-S9).
# ----------------------------------------------------------------------------------------------
def sort_key(g: Grid, i1, i2, tag, tile: int):
    """Tile-major cell key; dead particles get the key one past the last cell."""
    i1 = np.asarray(i1, np.int64); i2 = np.asarray(i2, np.int64)
    nt2 = (g.n2 + tile - 1) // tile
    nt1 = (g.n1 + tile - 1) // tile
    t1, l1 = i1 // tile, i1 % tile
    t2, l2 = i2 // tile, i2 % tile
    key = ((t1 * nt2 + t2) * tile + l1) * tile + l2
    dead_key = nt1 * nt2 * tile * tile
    return np.where(np.asarray(tag) != 0, key, dead_key), dead_key


def sort_reference(g: Grid, p: Particles, tile: int):
    """Stable sort of all columns by sort_key. Returns (sorted copy, permutation, keys_sorted)."""
    key, _ = sort_key(g, p.i1, p.i2, p.tag, tile)
    perm = np.argsort(key, kind="stable")
    q = p.copy()
    for k, v in p.__dict__.items():
        if isinstance(v, np.ndarray):
            setattr(q, k, v[perm].copy())
    return q, perm, key[perm]


# ----------------------------------------------------------------------------------------------
# Field side of one PIC timestep (Sec. 3.4), plain numpy around the three operations above.
# state = dict(B_prev = (n-3/2)B, B = (n-1/2)B, D_prev = (n-1)D, D = (n)D), each a dict of three float64 arrays.
# ----------------------------------------------------------------------------------------------
def _avg(x, y, keys):
    return {k: 0.5 * (x[k] + y[k]) for k in keys}


def fields_prepare(g: Grid, state: dict, dt: float) -> dict:
    """Step 2 (Eq. 46-48): returns (n)B, the magnetic field aligned with (n)D for the particle push."""
    kb, kd = ("B1", "B2", "B3"), ("D1", "D2", "D3")
    B_nm1 = _avg(state["B_prev"], state["B"], kb)                       # (n-1)B
    D_half = _avg(state["D_prev"], state["D"], kd)                      # (n-1/2)D
    E_half = aux_fields(g, {**state["B"], **D_half})                    # (n-1/2)E from (n-1/2)B, (n-1/2)D
    B_n = {k: np.array(v) for k, v in B_nm1.items()}
    faraday(g, B_n, E_half, dt)                                         # (n-1)B -> (n)B
    # Boundary conditions are imposed on the evolved field components, and the ghost zones next to the axis satisfy
    # reflection symmetry: the push reads the ghost columns of (n)B, which Faraday does not write
    if g.n2 >= g.ng:
        _axis_reflect(g, B_n)
    return B_n


def fields_advance(g: Grid, state: dict, B_n: dict, J_prev, J, dt: float, kJ: float = 4.0 * np.pi) -> dict:
    """Steps 5-7 (Eq. 51-56): state at (n+1); J_prev = (n-1/2)J, J = (n+1/2)J (dicts or None for vacuum)."""
    kb, kd = ("B1", "B2", "B3"), ("D1", "D2", "D3")
    J_n = None if J is None else _avg(J_prev, J, ("J1", "J2", "J3"))    # Eq. 51
    aux_n = aux_fields(g, {**B_n, **state["D"]})                        # Eq. 52
    B_new = {k: np.array(v) for k, v in state["B"].items()}
    faraday(g, B_new, aux_n, dt)                                        # Eq. 53: (n-1/2)B -> (n+1/2)B
    D_half = _avg(state["D_prev"], state["D"], kd)                      # (n-1/2)D
    ampere(g, D_half, aux_n, J_n, dt, kJ)                               # Eq. 54: -> (n+1/2)D
    aux_h = aux_fields(g, {**B_new, **D_half})                          # Eq. 55
    D_new = {k: np.array(v) for k, v in state["D"].items()}
    ampere(g, D_new, aux_h, J, dt, kJ)                                  # Eq. 56: (n)D -> (n+1)D
    return dict(B_prev=state["B"], B=B_new, D_prev=state["D"], D=D_new)


# ----------------------------------------------------------------------------------------------
# Field boundary conditions (Sec. 3.3.3; reading R-F4 of DESIGN.md): reflection across the polar axes of the
# ghost columns, zero for the components that vanish on the axes, constant layer inside the horizon.
# Parity of the contravariant code-basis components under theta -> -theta: r-components even, theta-components odd
# (Fig. 1); phi-components even (not stated; what the analytic continuation of an axisymmetric field gives).
# ----------------------------------------------------------------------------------------------
_AXIS_PARITY = {"D1": (+1, 0.0), "D2": (-1, 0.5), "D3": (+1, 0.0), "B1": (+1, 0.5), "B2": (-1, 0.0), "B3": (+1, 0.5)}


def field_bc(g: Grid, fields: dict, n_const: int = -1) -> dict:
    """In place on dict(D1..B3) of float64 arrays; n_const >= 0: rows i1 in [-ng, n_const] take the values of row
    n_const + 1 (n_const = number of current-filter passes n_f)."""
    _axis_reflect(g, fields)
    if n_const >= 0:
        for A in fields.values():
            A[: g.ng + n_const + 1, :] = A[g.ng + n_const + 1, :]
    return fields


def _axis_reflect(g: Grid, fields: dict) -> None:
    """ghost columns beyond the two polar axes of whichever of D1..B3 are in `fields`, and the zeros on the axes"""
    G, n2 = g.ng, g.n2
    for k, (par, off) in _AXIS_PARITY.items():
        if k not in fields:
            continue
        A = fields[k]
        for m in range(1, G + 1):
            if off == 0.0:                       # samples at integer j: ghost j = -m mirrors j = +m; j = n2+m mirrors n2-m
                A[:, G - m] = par * A[:, G + m]
                if G + n2 + m < A.shape[1]:
                    A[:, G + n2 + m] = par * A[:, G + n2 - m]
            else:                                # samples at j+1/2: ghost j = -m (+1/2) mirrors j = m-1 (+1/2)
                A[:, G - m] = par * A[:, G + m - 1]
                A[:, G + n2 + m - 1] = par * A[:, G + n2 - m]
    for k in ("B2", "D3"):                       # vanish on the axes by symmetry
        if k in fields:
            fields[k][:, G] = 0.0
            fields[k][:, G + n2] = 0.0


# ----------------------------------------------------------------------------------------------
# Absorbing layer at the outer radial boundary ("the fields are matched to their initial values using an
# absorbing layer"; "In the absorbing layer, we smoothly match the field components with the analytic
# solution").  The paper defers the profile to paper I.  Reading R-F6 of DESIGN.md: in the layer r_abs < r the field
# relaxes toward the target with the weight
#     s(r) = tanh(4 (r_max - r) / (r_max - r_abs)),   F <- F_target + s (F - F_target),
# every component at its own Yee radius (D^1, B^2, B^3 at i+1/2; D^2, D^3, B^1 at i); rows beyond r_max take the
# target; rows with r <= r_abs are not touched.  The PROFILE is parity unpinned (paper I); the pins check what any
# such layer must do: a fixed point at the target, untouched interior, monotone weight, and that an outgoing pulse
# is absorbed instead of reflected.
# ----------------------------------------------------------------------------------------------
_X1_OFFSET = {"D1": 0.5, "D2": 0.0, "D3": 0.0, "B1": 0.0, "B2": 0.5, "B3": 0.5}


def radius(g: Grid, x1):
    """r(x1) of the radial map (App. A.2 / A.3)"""
    x1 = np.asarray(x1, np.float64)
    if g.linear_r:
        return g.r_min + x1 * ((g.r_max - g.r_min) / g.n1)
    lo = np.log(g.r_min - g.r0)
    return g.r0 + np.exp(lo + x1 * ((np.log(g.r_max - g.r0) - lo) / g.n1))


def match_weight(g: Grid, r, r_abs: float):
    r = np.asarray(r, np.float64)
    d = np.clip((g.r_max - r) / (g.r_max - r_abs), 0.0, None)
    return np.tanh(4.0 * d)


def field_match(g: Grid, fields: dict, target: dict, r_abs: float) -> dict:
    """In place on dict(D1..B3) of float64 arrays [n1+2ng][n2+2ng]; target: the same keys (initial / analytic fields)."""
    G = g.ng
    for k, off in _X1_OFFSET.items():
        r = radius(g, np.arange(-G, g.n1 + G, dtype=np.float64) + off)
        rows = np.nonzero(r > r_abs)[0]
        s = match_weight(g, r[rows], r_abs)[:, None]
        A, T = fields[k], np.asarray(target[k], np.float64)
        A[rows, :] = T[rows, :] + s * (A[rows, :] - T[rows, :])
    return fields


# ----------------------------------------------------------------------------------------------
# Current filter ("n_f passes of a digital filter", details deferred to paper I).  Reading R-F5: the
# standard binomial 1-2-1 smoothing of PIC codes, separable in x1 and x2, one pass = [1 2 1]/4 along each axis, on
# each component's own Yee lattice; beyond the polar axes the neighbour is the mirror sample with the component's
# parity (J^1, J^3 even, J^2 odd, as D^i); the first and last array rows are left as they are.
# The CHOICE of filter is parity unpinned (any symmetric normalised stencil commutes with the continuity equation).
# ----------------------------------------------------------------------------------------------
_J_PARITY = {"J1": (+1, 0.0), "J2": (-1, 0.5), "J3": (+1, 0.0)}


def filter_current(g: Grid, J: dict, n_passes: int = 1) -> dict:
    G, n2 = g.ng, g.n2
    for _ in range(int(n_passes)):
        for k, (par, off) in _J_PARITY.items():
            A = J[k]
            ncol = n2 + 1 if off == 0.0 else n2                 # physical samples in theta
            P = np.zeros((A.shape[0], ncol + 2))
            P[:, 1:-1] = A[:, G:G + ncol]
            if off == 0.0:                                      # node-sampled: j = -1 mirrors j = +1, n2+1 mirrors n2-1
                P[:, 0] = par * A[:, G + 1]; P[:, -1] = par * A[:, G + n2 - 1]
            else:                                               # half-sampled: -1/2 mirrors +1/2, n2+1/2 mirrors n2-1/2
                P[:, 0] = par * A[:, G]; P[:, -1] = par * A[:, G + n2 - 1]
            T = 0.25 * (P[:, :-2] + 2.0 * P[:, 1:-1] + P[:, 2:])               # along x2
            out = T.copy()
            out[1:-1] = 0.25 * (T[:-2] + 2.0 * T[1:-1] + T[2:])                # along x1, edge rows unchanged in x1
            A[:, G:G + ncol] = out
    return J
