"""ctypes binding of the CPU oracle (oracle/libmco.so).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
may import this module.  It never imports the product package's CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)


class FieldParams(C.Structure):
    _fields_ = [("kind", C.c_int32), ("sigma", C.c_float), ("radius", C.c_int32),
                ("coupling", C.c_float), ("n_sources", C.c_int32), ("sources", _fp)]


class WorldParams(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("dt", C.c_float), ("nu", C.c_float),
                ("trt_lambda", C.c_float), ("rho0", C.c_float), ("k_el", C.c_float),
                ("pbd_iters", C.c_int32), ("n_fields", C.c_int32), ("fields", FieldParams * 4),
                ("max_beads", C.c_int64), ("coupling", C.c_int32), ("mdf_iters", C.c_int32),
                ("pbd_order", C.c_int32), ("pbd_project", C.c_int32), ("two_layer", C.c_int32),
                ("layer_offset", C.c_float)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.mco_phi.restype = C.c_double
        L.mco_phi.argtypes = [C.c_double]
        L.mco_last_error.restype = C.c_char_p
        L.mco_last_error.argtypes = [C.c_void_p]
        L.mco_destroy.restype = None
        L.mco_destroy.argtypes = [C.c_void_p]
        L.mco_radius.restype = C.c_int32
        L.mco_radius.argtypes = [C.c_double, C.c_int32]
        _lib = L
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f(a):
    return None if a is None else a.ctypes.data_as(_fp)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def make_params(p: dict):
    """dict (worlds.py) -> (WorldParams, keepalive list)."""
    wp = WorldParams()
    keep = []
    for k in ("nx", "ny", "pbd_iters"):
        setattr(wp, k, int(p[k]))
    for k in ("dt", "nu", "trt_lambda", "rho0", "k_el"):
        setattr(wp, k, float(p[k]))
    wp.n_fields = len(p["fields"])
    wp.max_beads = int(p["max_beads"])
    wp.coupling = int(p.get("coupling", 0))
    wp.mdf_iters = int(p.get("mdf_iters", 0))
    wp.pbd_order = int(p.get("pbd_order", 0))
    wp.pbd_project = int(p.get("pbd_project", 0))
    wp.two_layer = int(p.get("two_layer", 0))
    wp.layer_offset = float(p.get("layer_offset", 0.0))
    for i, fd in enumerate(p["fields"]):
        fp = wp.fields[i]
        fp.kind = int(fd["kind"])
        fp.sigma = float(fd["sigma"])
        fp.radius = int(fd["radius"])
        fp.coupling = float(fd["coupling"])
        src = fd.get("sources")
        if src is not None:
            src = _f32(src).reshape(-1, 4)
            keep.append(src)
            fp.n_sources = src.shape[0]
            fp.sources = _f(src)
        else:
            fp.n_sources = 0
            fp.sources = None
    return wp, keep


class World:
    """Oracle world: mco_create + mco_load_filaments from a worlds.py dict."""

    def __init__(self, world: dict, fp32_state: bool = False, threads: int = 0):
        L = lib()
        self.p = world["params"]
        self.nx, self.ny = int(self.p["nx"]), int(self.p["ny"])
        self.n_fields = len(self.p["fields"])
        wp, self._keep = make_params(self.p)
        h = C.c_void_p()
        rc = L.mco_create(C.byref(wp), C.byref(h))
        if rc != 0:
            raise ValueError(f"mco_create failed: {rc}")
        self.h = h
        off = np.ascontiguousarray(world["offsets"], dtype=np.int32)
        self.N = int(off[-1])
        arrs = [_f32(world[k]) for k in ("xy", "L_rest", "theta_rest", "k_bend", "k_shear",
                                        "k_stretch", "act_amp", "act_phase", "act_period")]
        rc = L.mco_load_filaments(h, C.c_int32(len(off) - 1), off.ctypes.data_as(_ip),
                                  *[_f(a) for a in arrs])
        if rc != 0:
            msg = L.mco_last_error(h).decode()
            L.mco_destroy(h)
            self.h = None
            raise ValueError(f"mco_load_filaments failed: {rc} {msg}")
        if world.get("act_L_amp") is not None:
            la = _f32(world["act_L_amp"])
            assert la.shape == (self.N,)
            L.mco_set_length_actuation(h, _f(la))
        if fp32_state:
            L.mco_set_fp32_state(h, 1)
        L.mco_set_threads(h, int(threads))

    def close(self):
        if getattr(self, "h", None):
            lib().mco_destroy(self.h)
            self.h = None

    def __del__(self):
        self.close()

    def set_state(self, step: int, xy=None, fdev=None):
        xy = None if xy is None else _f64(xy)
        fdev = None if fdev is None else _f64(fdev)
        rc = lib().mco_set_state(self.h, C.c_int64(step), _d(xy), _d(fdev))
        if rc != 0:
            raise ValueError(f"mco_set_state failed: {rc}")

    def set_threads(self, k: int):
        lib().mco_set_threads(self.h, int(k))

    def step(self, n: int = 1):
        rc = lib().mco_step(self.h, C.c_int32(n))
        if rc != 0:
            raise RuntimeError(f"mco_step failed: {rc} {lib().mco_last_error(self.h).decode()}")

    def read_state(self) -> dict:
        ny, nx, N = self.ny, self.nx, self.N
        out = dict(xy=np.empty((N, 2)), u=np.empty((2, ny, nx)), rho=np.empty((ny, nx)),
                   fdev=np.empty((9, ny, nx)), field=np.empty((self.n_fields, ny, nx)),
                   force=np.empty((N, 2)), sense=np.empty(N))
        st = C.c_int64()
        rc = lib().mco_read_state(self.h, C.byref(st), _d(out["xy"]), _d(out["u"]), _d(out["rho"]),
                                  _d(out["fdev"]), _d(out["field"]), _d(out["force"]),
                                  _d(out["sense"]))
        if rc != 0:
            raise RuntimeError(f"mco_read_state failed: {rc}")
        out["step"] = int(st.value)
        return out

    def read_intermediates(self) -> dict:
        ny, nx, N = self.ny, self.nx, self.N
        out = dict(D=np.empty((N, 2)), rho_b=np.empty((ny, nx)), G=np.empty((2, ny, nx)))
        lib().mco_read_intermediates(self.h, _d(out["D"]), _d(out["rho_b"]), _d(out["G"]))
        return out


# ---- stateless components ----
def phi(r: float) -> float:
    return float(lib().mco_phi(float(r)))


def support(x: float):
    i0 = C.c_int32()
    w = (C.c_double * 4)()
    lib().mco_support(C.c_double(x), C.byref(i0), w)
    return int(i0.value), np.array(w[:])


def elastic(offsets, xy, L_rest, theta_rest, k_bend, k_shear, k_stretch, act_amp, act_phase,
            act_period, dt: float, n: int) -> np.ndarray:
    off = np.ascontiguousarray(offsets, dtype=np.int32)
    xy = _f64(xy)
    N = int(off[-1])
    arrs = [_f32(a) for a in (L_rest, theta_rest, k_bend, k_shear, k_stretch, act_amp, act_phase,
                              act_period)]
    D = np.empty((N, 2))
    rc = lib().mco_elastic(C.c_int32(len(off) - 1), off.ctypes.data_as(_ip), _d(xy),
                           *[_f(a) for a in arrs], C.c_double(dt), C.c_int64(n), _d(D))
    if rc != 0:
        raise ValueError(f"mco_elastic failed: {rc}")
    return D


def pbd(offsets, xy, L_rest, theta_rest, k_bend, k_shear, k_stretch, act_amp, act_phase, act_period,
        dt: float, n: int, iters: int = 1, order: int = 0, act_L_amp=None) -> np.ndarray:
    """Literal PBD (reading 27): net displacement of `iters` iterations, Jacobi (0) or red-black GS (1)."""
    off = np.ascontiguousarray(offsets, dtype=np.int32)
    xy = _f64(xy)
    N = int(off[-1])
    arrs = [_f32(a) for a in (L_rest, theta_rest, k_bend, k_shear, k_stretch, act_amp, act_phase,
                              act_period)]
    la = None if act_L_amp is None else _f32(act_L_amp)
    D = np.empty((N, 2))
    rc = lib().mco_pbd(C.c_int32(len(off) - 1), off.ctypes.data_as(_ip), _d(xy),
                       *[_f(a) for a in arrs], _f(la), C.c_double(dt), C.c_int64(n), C.c_int32(iters),
                       C.c_int32(order), _d(D))
    if rc != 0:
        raise ValueError(f"mco_pbd failed: {rc}")
    return D


def markers(offsets, xy, h: float) -> np.ndarray:
    """Two-layer markers (reading 28): [2N, 2], rows 2i / 2i+1 = X_i +- h n_i."""
    off = np.ascontiguousarray(offsets, dtype=np.int32)
    xy = _f64(xy)
    out = np.empty((2 * len(xy), 2))
    lib().mco_markers(C.c_int32(len(off) - 1), off.ctypes.data_as(_ip), _d(xy), C.c_double(h), _d(out))
    return out


def deposit(nx, ny, xy) -> np.ndarray:
    xy = _f64(xy)
    out = np.empty((ny, nx))
    lib().mco_deposit(C.c_int32(nx), C.c_int32(ny), C.c_int64(len(xy)), _d(xy), _d(out))
    return out


def spread(nx, ny, xy, F) -> np.ndarray:
    xy, F = _f64(xy), _f64(F)
    out = np.empty((2, ny, nx))
    lib().mco_spread(C.c_int32(nx), C.c_int32(ny), C.c_int64(len(xy)), _d(xy), _d(F), _d(out))
    return out


def interp(planes, xy) -> np.ndarray:
    planes, xy = _f64(planes), _f64(xy)
    nch, ny, nx = planes.shape
    out = np.empty((len(xy), nch))
    lib().mco_interp(C.c_int32(nx), C.c_int32(ny), C.c_int32(nch), _d(planes), C.c_int64(len(xy)),
                     _d(xy), _d(out))
    return out


def radius(sigma: float, r: int = 0) -> int:
    return int(lib().mco_radius(float(sigma), int(r)))


def gauss_taps(sigma: float, R: int) -> np.ndarray:
    t = np.empty(2 * R + 1)
    lib().mco_gauss_taps(C.c_double(sigma), C.c_int32(R), _d(t))
    return t


def blur(a, sigma: float, R: int) -> np.ndarray:
    a = _f64(a)
    ny, nx = a.shape
    out = np.empty((ny, nx))
    lib().mco_blur(C.c_int32(nx), C.c_int32(ny), _d(a), C.c_double(sigma), C.c_int32(R), _d(out))
    return out


def grad(a):
    a = _f64(a)
    ny, nx = a.shape
    gx, gy = np.empty((ny, nx)), np.empty((ny, nx))
    lib().mco_grad(C.c_int32(nx), C.c_int32(ny), _d(a), _d(gx), _d(gy))
    return gx, gy


def static_field(nx, ny, sources) -> np.ndarray:
    s = _f32(sources).reshape(-1, 4)
    out = np.empty((ny, nx))
    lib().mco_static_field(C.c_int32(nx), C.c_int32(ny), C.c_int32(len(s)), _f(s), _d(out))
    return out


def lattice_constants(nu: float, dt: float, lam: float):
    a, b = C.c_double(), C.c_double()
    lib().mco_lattice_constants(C.c_double(nu), C.c_double(dt), C.c_double(lam), C.byref(a),
                                C.byref(b))
    return float(a.value), float(b.value)


def lbm_step(f, G, omega_plus: float, omega_minus: float):
    """f [9,ny,nx] un-shifted (modified copy returned), G [2,ny,nx] or None -> (f', u)."""
    f = _f64(f).copy()
    _, ny, nx = f.shape
    G = None if G is None else _f64(G)
    u = np.empty((2, ny, nx))
    lib().mco_lbm_step(C.c_int32(nx), C.c_int32(ny), _d(f), _d(G), C.c_double(omega_plus),
                       C.c_double(omega_minus), _d(u))
    return f, u


def moments(f):
    """f [9,ny,nx] un-shifted -> (rho [ny,nx], ustar [2,ny,nx])."""
    f = _f64(f)
    _, ny, nx = f.shape
    rho, us = np.empty((ny, nx)), np.empty((2, ny, nx))
    lib().mco_moments(C.c_int32(nx), C.c_int32(ny), _d(f), _d(rho), _d(us))
    return rho, us


def mdf(xy, V, ustar, rho, rho0: float, iters: int):
    """Multi-Direct Forcing -> dict(F [N,2], G [2,ny,nx], u [2,ny,nx], resid [iters+1])."""
    xy, V, ustar, rho = _f64(xy), _f64(V), _f64(ustar), _f64(rho)
    _, ny, nx = ustar.shape
    N = len(xy)
    out = dict(F=np.empty((N, 2)), G=np.empty((2, ny, nx)), u=np.empty((2, ny, nx)),
               resid=np.empty(iters + 1))
    lib().mco_mdf(C.c_int32(nx), C.c_int32(ny), C.c_int64(N), _d(xy), _d(V), _d(ustar), _d(rho),
                  C.c_double(rho0), C.c_int32(iters), _d(out["F"]), _d(out["G"]), _d(out["u"]),
                  _d(out["resid"]))
    return out


def mdf_layers(P, layers: int, V, ustar, rho, rho0: float, iters: int):
    """MDF through `layers` points per bead (P [N*layers, 2]) -> dict like mdf()."""
    P, V, ustar, rho = _f64(P), _f64(V), _f64(ustar), _f64(rho)
    _, ny, nx = ustar.shape
    N = len(V)
    assert len(P) == N * layers
    out = dict(F=np.empty((N, 2)), G=np.empty((2, ny, nx)), u=np.empty((2, ny, nx)),
               resid=np.empty(iters + 1))
    lib().mco_mdf_layers(C.c_int32(nx), C.c_int32(ny), C.c_int64(N), C.c_int32(layers), _d(P), _d(V), _d(ustar),
                         _d(rho), C.c_double(rho0), C.c_int32(iters), _d(out["F"]), _d(out["G"]), _d(out["u"]),
                         _d(out["resid"]))
    return out
