"""Thin ctypes binding of include/grpic.h — argument marshalling only.

Every step of the path runs in the CUDA kernels of libgrpic_f32.so / libgrpic_f64.so; this module
only turns torch CUDA tensors into raw device pointers and checks status codes.  There is no CPU
fallback: if the shared library is missing the import of a precision raises, and every compute call
on a machine without a CUDA device raises GrpicError (GRPIC_ECUDA).

Names follow the C ABI: Context.interp_push / deposit / step / sort / counters / step_host.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

GRPIC_OK, GRPIC_EINVAL, GRPIC_ENOMEM, GRPIC_ECUDA, GRPIC_ESTATE = 0, -1, -2, -3, -4

EXPORTS = ["grpic_real_bytes", "grpic_create", "grpic_destroy", "grpic_set_int", "grpic_set_real",
           "grpic_interp_push", "grpic_deposit", "grpic_step", "grpic_sort", "grpic_tile_size",
           "grpic_counters", "grpic_updates_total", "grpic_step_host", "grpic_last_error",
           "grpic_aux_fields", "grpic_faraday", "grpic_ampere", "grpic_fields_prepare", "grpic_fields_advance",
           "grpic_field_bc", "grpic_sorted_alive", "grpic_filter_current", "grpic_sort_into", "grpic_field_match",
           "grpic_probe", "grpic_forget"]


class GrpicError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"grpic status {code}: {msg}")
        self.code = code


class _Grid(C.Structure):
    _fields_ = [("n1", C.c_int32), ("n2", C.c_int32), ("nghost", C.c_int32), ("r_map", C.c_int32)]


_vp = C.c_void_p


class _Particles(C.Structure):
    _fields_ = [("n", C.c_int64), ("i1", _vp), ("i2", _vp), ("dx1", _vp), ("dx2", _vp),
                ("u1", _vp), ("u2", _vp), ("u3", _vp), ("phi", _vp),
                ("i1_prev", _vp), ("i2_prev", _vp), ("dx1_prev", _vp), ("dx2_prev", _vp),
                ("weight", _vp), ("tag", _vp),
                ("q_over_m", C.c_double), ("charge", C.c_double), ("massive", C.c_int32)]


class _Fields(C.Structure):
    _fields_ = [(k, _vp) for k in ("D1", "D2", "D3", "B1", "B2", "B3")]


class _Vec3(C.Structure):
    _fields_ = [(k, _vp) for k in ("F1", "F2", "F3")]


class _FieldState(C.Structure):
    _fields_ = [("B_prev", _Vec3), ("B", _Vec3), ("D_prev", _Vec3), ("D", _Vec3)]


class _Current(C.Structure):
    _fields_ = [(k, _vp) for k in ("J1", "J2", "J3")]


_libs = {}


def load(precision: str, build_if_missing: bool = False):
    """dlopen libgrpic_<precision>.so (precision 'f32' or 'f64').  Fails loudly if it is not built."""
    if precision in _libs:
        return _libs[precision]
    path = _build.lib_path(precision)
    if not os.path.exists(path):
        if not build_if_missing:
            raise ImportError(f"{path} is missing: run `python -m paper_2511_17701_b200.build` "
                              f"(there is no fallback path)")
        _build.build()
    lib = C.CDLL(path)
    lib.grpic_last_error.restype = C.c_char_p
    lib.grpic_last_error.argtypes = [_vp]
    lib.grpic_create.argtypes = [C.POINTER(_Grid), C.c_double, C.c_double, C.c_double, C.POINTER(_vp)]
    lib.grpic_destroy.argtypes = [_vp]
    lib.grpic_set_int.argtypes = [_vp, C.c_char_p, C.c_int64]
    lib.grpic_set_real.argtypes = [_vp, C.c_char_p, C.c_double]
    lib.grpic_interp_push.argtypes = [_vp, C.POINTER(_Particles), C.POINTER(_Fields), C.c_double, _vp]
    lib.grpic_deposit.argtypes = [_vp, C.POINTER(_Particles), C.POINTER(_Current), _vp]
    lib.grpic_step.argtypes = [_vp, C.POINTER(_Particles), C.POINTER(_Fields), C.POINTER(_Current), C.c_double, _vp]
    lib.grpic_sort.argtypes = [_vp, C.POINTER(_Particles), _vp]
    lib.grpic_sort_into.argtypes = [_vp, C.POINTER(_Particles), C.POINTER(_Particles), _vp]
    lib.grpic_counters.argtypes = [_vp] + [C.POINTER(C.c_int64)] * 4 + [_vp]
    lib.grpic_updates_total.argtypes = [_vp, C.POINTER(C.c_int64), _vp]
    lib.grpic_probe.argtypes = [_vp, C.c_char_p, C.c_int64, C.POINTER(C.c_int64), _vp]
    lib.grpic_step_host.argtypes = [_vp, C.POINTER(_Particles), C.POINTER(_Fields), C.POINTER(_Current), C.c_double,
                                    C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    lib.grpic_aux_fields.argtypes = [_vp, C.POINTER(_Fields), C.POINTER(_Vec3), C.POINTER(_Vec3), _vp]
    lib.grpic_faraday.argtypes = [_vp, C.POINTER(_Vec3), C.POINTER(_Vec3), C.c_double, _vp]
    lib.grpic_ampere.argtypes = [_vp, C.POINTER(_Vec3), C.POINTER(_Vec3), C.POINTER(_Current), C.c_double, _vp]
    lib.grpic_sorted_alive.argtypes = [_vp, C.POINTER(_Particles), C.POINTER(C.c_int64)]
    lib.grpic_forget.argtypes = [_vp, C.POINTER(_Particles)]
    lib.grpic_filter_current.argtypes = [_vp, C.POINTER(_Current), C.c_int32, _vp]
    lib.grpic_field_bc.argtypes = [_vp, C.POINTER(_Vec3), C.POINTER(_Vec3), C.c_int32, _vp]
    lib.grpic_field_match.argtypes = [_vp] + [C.POINTER(_Vec3)] * 4 + [C.c_double, _vp]
    lib.grpic_fields_prepare.argtypes = [_vp, C.POINTER(_FieldState), C.POINTER(_Vec3), C.c_double, _vp]
    lib.grpic_fields_advance.argtypes = [_vp, C.POINTER(_FieldState), C.POINTER(_Vec3), C.POINTER(_Current),
                                         C.POINTER(_Current), C.c_double, _vp]
    want = 4 if precision == "f32" else 8
    if lib.grpic_real_bytes() != want:
        raise ImportError(f"{path} reports grpic_real of {lib.grpic_real_bytes()} bytes, expected {want}")
    _libs[precision] = lib
    return lib


def _torch():
    import torch
    return torch


def _np_real(precision):
    return np.float32 if precision == "f32" else np.float64


def torch_real(precision):
    torch = _torch()
    return torch.float32 if precision == "f32" else torch.float64


_REAL_COLS = ("dx1", "dx2", "u1", "u2", "u3", "phi", "dx1_prev", "dx2_prev", "weight")
_INT_COLS = ("i1", "i2", "i1_prev", "i2_prev")
ALL_COLS = ("i1", "i2", "dx1", "dx2", "u1", "u2", "u3", "phi", "i1_prev", "i2_prev", "dx1_prev", "dx2_prev",
            "weight", "tag")


class ParticleSet:
    """One species: SoA columns held as torch tensors (device or pinned host), plus species constants."""

    def __init__(self, cols: dict, q_over_m: float, charge: float, massive: int = 1):
        self.cols = cols
        self.q_over_m, self.charge, self.massive = float(q_over_m), float(charge), int(massive)

    @property
    def n(self):
        return int(self.cols["i1"].numel())

    @classmethod
    def from_host(cls, sp, precision: str, device="cuda", with_phi=None, pinned=False):
        """sp: any object with numpy columns i1,i2,dx1,dx2,u1,u2,u3,weight,tag[,phi] and q_over_m, charge, massive
        (workloads.Species or oracle Particles).  Values are rounded once to the build's precision."""
        torch = _torch()
        rt = _np_real(precision)
        has_phi = (getattr(sp, "phi", None) is not None) if with_phi is None else with_phi
        n = int(np.asarray(sp.i1).size)

        def put(a, dt):
            t = torch.from_numpy(np.ascontiguousarray(a, dtype=dt))
            if device == "cpu":
                return t.pin_memory() if pinned else t.clone()
            return t.to(device)

        cols = {"i1": put(sp.i1, np.int32), "i2": put(sp.i2, np.int32), "tag": put(sp.tag, np.uint8)}
        for k in ("dx1", "dx2", "u1", "u2", "u3", "weight"):
            cols[k] = put(getattr(sp, k), rt)
        cols["phi"] = put(sp.phi, rt) if has_phi else None
        for k, dt in (("i1_prev", np.int32), ("i2_prev", np.int32), ("dx1_prev", rt), ("dx2_prev", rt)):
            src = getattr(sp, k, None)
            cols[k] = put(src if src is not None else np.zeros(n, dt), dt)
        return cls(cols, sp.q_over_m, sp.charge, sp.massive)

    def drop_prev(self):
        """forget the four *_prev columns (the fused step and the sort do without them)"""
        for k in ("i1_prev", "i2_prev", "dx1_prev", "dx2_prev"):
            self.cols[k] = None
        return self

    def empty_like(self):
        """a second column set of the same shape (uninitialised): the other half of a sort_into ping-pong"""
        torch = _torch()
        return ParticleSet({k: (None if v is None else torch.empty_like(v)) for k, v in self.cols.items()},
                           self.q_over_m, self.charge, self.massive)

    def clone(self):
        return ParticleSet({k: (None if v is None else v.clone()) for k, v in self.cols.items()},
                           self.q_over_m, self.charge, self.massive)

    def to_numpy(self) -> dict:
        return {k: (None if v is None else v.detach().cpu().numpy().copy()) for k, v in self.cols.items()}

    def c_struct(self, with_prev: bool = True) -> _Particles:
        c = self.cols
        if not with_prev:
            c = dict(c, i1_prev=None, i2_prev=None, dx1_prev=None, dx2_prev=None)
        ptr = lambda t: None if t is None else t.data_ptr()
        return _Particles(self.n, ptr(c["i1"]), ptr(c["i2"]), ptr(c["dx1"]), ptr(c["dx2"]), ptr(c["u1"]),
                          ptr(c["u2"]), ptr(c["u3"]), ptr(c["phi"]), ptr(c["i1_prev"]), ptr(c["i2_prev"]),
                          ptr(c["dx1_prev"]), ptr(c["dx2_prev"]), ptr(c["weight"]), ptr(c["tag"]),
                          self.q_over_m, self.charge, self.massive)


def grid_tensors(arrays: dict, names, precision: str, device="cuda", pinned=False):
    torch = _torch()
    out = {}
    for k in names:
        t = torch.from_numpy(np.ascontiguousarray(arrays[k], dtype=_np_real(precision)))
        out[k] = (t.pin_memory() if pinned else t.clone()) if device == "cpu" else t.to(device)
    return out


def _fields_struct(fields):
    if fields is None:
        return None
    return _Fields(*[fields[k].data_ptr() for k in ("D1", "D2", "D3", "B1", "B2", "B3")])


def _current_struct(J):
    if J is None:
        return None
    return _Current(*[J[k].data_ptr() for k in ("J1", "J2", "J3")])


def _stream_ptr(stream):
    if stream is None:
        torch = _torch()
        if torch.cuda.is_available():
            return torch.cuda.current_stream().cuda_stream
        return None
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


class Context:
    """grpic_ctx* with the ABI's calls as methods (same names, same order of arguments)."""

    def __init__(self, n1, n2, a, r_min, r_max, nghost=2, precision="f32", n_iter=None, small_angle=None,
                 r0=None, h0=None, r_map=1, mass=None):
        self.precision = precision
        self.lib = load(precision)
        self.n1, self.n2, self.nghost = int(n1), int(n2), int(nghost)
        g = _Grid(self.n1, self.n2, self.nghost, int(r_map))
        h = _vp()
        rc = self.lib.grpic_create(C.byref(g), float(a), float(r_min), float(r_max), C.byref(h))
        if rc != GRPIC_OK:
            raise GrpicError(rc, self.lib.grpic_last_error(None).decode())
        self.h = h
        if n_iter is not None:
            self.set_int("n_iter", n_iter)
        if small_angle is not None:
            self.set_real("small_angle", small_angle)
        if r0 is not None:
            self.set_real("r0", r0)        # A.3 radial offset
        if h0 is not None:
            self.set_real("h0", h0)        # A.3 polar stretch
        if mass is not None:
            self.set_real("mass", mass)    # 0 with a = 0: flat kerr_schild_0 (App. A.1)

    @property
    def shape(self):
        return (self.n1 + 2 * self.nghost, self.n2 + 2 * self.nghost)

    def _ck(self, rc):
        if rc != GRPIC_OK:
            raise GrpicError(rc, self.lib.grpic_last_error(self.h).decode())

    def close(self):
        if getattr(self, "h", None):
            self.lib.grpic_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_int(self, key, v):
        self._ck(self.lib.grpic_set_int(self.h, key.encode(), int(v)))

    def set_real(self, key, v):
        self._ck(self.lib.grpic_set_real(self.h, key.encode(), float(v)))

    def interp_push(self, p: ParticleSet, fields, dt, stream=None):
        ps = p.c_struct(); fs = _fields_struct(fields)
        self._ck(self.lib.grpic_interp_push(self.h, C.byref(ps), C.byref(fs) if fs else None, float(dt),
                                            _stream_ptr(stream)))

    def deposit(self, p: ParticleSet, J, stream=None):
        ps = p.c_struct(); js = _current_struct(J)
        self._ck(self.lib.grpic_deposit(self.h, C.byref(ps), C.byref(js) if js else None, _stream_ptr(stream)))

    def step(self, p: ParticleSet, fields, J, dt, stream=None):
        ps = p.c_struct(); fs = _fields_struct(fields); js = _current_struct(J)
        self._ck(self.lib.grpic_step(self.h, C.byref(ps), C.byref(fs) if fs else None,
                                     C.byref(js) if js else None, float(dt), _stream_ptr(stream)))

    def sort(self, p: ParticleSet, stream=None):
        ps = p.c_struct()
        self._ck(self.lib.grpic_sort(self.h, C.byref(ps), _stream_ptr(stream)))

    def sort_into(self, src: ParticleSet, dst: ParticleSet, stream=None):
        """out-of-place sort: src -> dst (two column sets that the caller swaps), no snapshot inside"""
        a = src.c_struct(); b = dst.c_struct()
        self._ck(self.lib.grpic_sort_into(self.h, C.byref(a), C.byref(b), _stream_ptr(stream)))

    def forget(self, p: ParticleSet):
        """drop the tile table of this species (before its storage is freed or reused)"""
        ps = p.c_struct()
        self._ck(self.lib.grpic_forget(self.h, C.byref(ps)))

    def sorted_alive(self, p: ParticleSet) -> int:
        """alive particles of the species at its last sort; they occupy the slots [0, n_alive)"""
        ps = p.c_struct(); v = C.c_int64(0)
        self._ck(self.lib.grpic_sorted_alive(self.h, C.byref(ps), C.byref(v)))
        return int(v.value)

    def counters(self, stream=None):
        v = [C.c_int64(0) for _ in range(4)]
        self._ck(self.lib.grpic_counters(self.h, *[C.byref(x) for x in v], _stream_ptr(stream)))
        return dict(zip(("alive", "absorbed_in", "absorbed_out", "overstep"), (int(x.value) for x in v)))

    def probe(self, what: str, iters: int, stream=None) -> int:
        """enqueue one throughput-probe launch ("ffma", "dfma", "mufu", "smem_rmw"); returns its operation count"""
        v = C.c_int64(0)
        self._ck(self.lib.grpic_probe(self.h, what.encode(), int(iters), C.byref(v), _stream_ptr(stream)))
        return int(v.value)

    def updates_total(self, stream=None) -> int:
        v = C.c_int64(0)
        self._ck(self.lib.grpic_updates_total(self.h, C.byref(v), _stream_ptr(stream)))
        return int(v.value)

    def step_host(self, p: ParticleSet, fields, J, dt, with_prev: bool = True):
        """All tensors are HOST tensors (pinned or not).  Returns (h2d_bytes, d2h_bytes).
        with_prev=False passes NULL for the four *_prev columns (they are then not copied back)."""
        ps = p.c_struct(with_prev); fs = _fields_struct(fields); js = _current_struct(J)
        up, down = C.c_int64(0), C.c_int64(0)
        self._ck(self.lib.grpic_step_host(self.h, C.byref(ps), C.byref(fs) if fs else None,
                                          C.byref(js) if js else None, float(dt), C.byref(up), C.byref(down)))
        return int(up.value), int(down.value)

    # ---- field-solver half (Sec. 3.3): dicts of torch CUDA tensors, keys as named ----
    def aux_fields(self, fields, E=None, H=None, stream=None):
        """E = dict(E1,E2,E3) and/or H = dict(H1,H2,H3) are written from fields = dict(D1..B3)."""
        fs = _fields_struct(fields)
        e = None if E is None else _Vec3(*[E[k].data_ptr() for k in ("E1", "E2", "E3")])
        h = None if H is None else _Vec3(*[H[k].data_ptr() for k in ("H1", "H2", "H3")])
        self._ck(self.lib.grpic_aux_fields(self.h, C.byref(fs), C.byref(e) if e else None, C.byref(h) if h else None,
                                           _stream_ptr(stream)))

    def faraday(self, B, E, dt, stream=None):
        b = _Vec3(*[B[k].data_ptr() for k in ("B1", "B2", "B3")])
        e = _Vec3(*[E[k].data_ptr() for k in ("E1", "E2", "E3")])
        self._ck(self.lib.grpic_faraday(self.h, C.byref(b), C.byref(e), float(dt), _stream_ptr(stream)))

    def ampere(self, D, H, J, dt, stream=None):
        d = _Vec3(*[D[k].data_ptr() for k in ("D1", "D2", "D3")])
        h = _Vec3(*[H[k].data_ptr() for k in ("H1", "H2", "H3")])
        js = _current_struct(J)
        self._ck(self.lib.grpic_ampere(self.h, C.byref(d), C.byref(h), C.byref(js) if js else None, float(dt),
                                       _stream_ptr(stream)))

    def filter_current(self, J, n_passes=1, stream=None):
        js = _current_struct(J)
        self._ck(self.lib.grpic_filter_current(self.h, C.byref(js), int(n_passes), _stream_ptr(stream)))

    def field_bc(self, fields, n_const=-1, stream=None):
        """Axis reflection of the ghost columns, zeros on the axes, constant layer inside the horizon (in place)."""
        d = _Vec3(*[fields[k].data_ptr() for k in ("D1", "D2", "D3")])
        b = _Vec3(*[fields[k].data_ptr() for k in ("B1", "B2", "B3")])
        self._ck(self.lib.grpic_field_bc(self.h, C.byref(d), C.byref(b), int(n_const), _stream_ptr(stream)))

    def field_match(self, fields, target, r_abs, stream=None):
        """Absorbing layer r_abs < r <= r_max: fields relax toward `target` (dict D1..B3), in place (reading R-F6)."""
        v = lambda d, ks: _Vec3(*[d[k].data_ptr() for k in ks])
        kb, kd = ("B1", "B2", "B3"), ("D1", "D2", "D3")
        d, b, d0, b0 = v(fields, kd), v(fields, kb), v(target, kd), v(target, kb)
        self._ck(self.lib.grpic_field_match(self.h, C.byref(d), C.byref(b), C.byref(d0), C.byref(b0), float(r_abs),
                                            _stream_ptr(stream)))

    @staticmethod
    def _state_struct(state):
        v = lambda d, ks: _Vec3(*[d[k].data_ptr() for k in ks])
        kb, kd = ("B1", "B2", "B3"), ("D1", "D2", "D3")
        return _FieldState(v(state["B_prev"], kb), v(state["B"], kb), v(state["D_prev"], kd), v(state["D"], kd))

    def fields_prepare(self, state, B_n, dt, stream=None):
        """state = dict(B_prev, B, D_prev, D) of dicts of tensors; B_n = dict(B1,B2,B3) receives (n)B (Eq. 46-48)."""
        ss = self._state_struct(state)
        bn = _Vec3(*[B_n[k].data_ptr() for k in ("B1", "B2", "B3")])
        self._ck(self.lib.grpic_fields_prepare(self.h, C.byref(ss), C.byref(bn), float(dt), _stream_ptr(stream)))

    def fields_advance(self, state, B_n, J_prev, J, dt, stream=None):
        """Eq. 51-56; the tensors of `state` are updated in place to (n-1/2)B, (n+1/2)B, (n)D, (n+1)D."""
        ss = self._state_struct(state)
        bn = _Vec3(*[B_n[k].data_ptr() for k in ("B1", "B2", "B3")])
        jp, jn = _current_struct(J_prev), _current_struct(J)
        self._ck(self.lib.grpic_fields_advance(self.h, C.byref(ss), C.byref(bn), C.byref(jp) if jp else None,
                                               C.byref(jn) if jn else None, float(dt), _stream_ptr(stream)))

    def tile_size(self):
        return int(self.lib.grpic_tile_size())
