"""ctypes binding of the CPU oracle (oracle/ugkso.c).  Test infrastructure only.

``build()`` compiles ``libugkso.so`` next to the source with gcc
(``-O2 -ffp-contract=off -fopenmp``).  ``Oracle(problem)`` wraps one context; ``problem``
is a ``workloads.Problem`` (plain data: mesh, velocity nodes/weights, gas, BCs, CFL).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libugkso.so")
_SRC = [os.path.join(_HERE, "ugkso.c"), os.path.join(_HERE, "ugkso.h")]
_lock = threading.Lock()
_lib = None

_dp = C.POINTER(C.c_double)


class _Mesh(C.Structure):
    _fields_ = [("I", C.c_int), ("J", C.c_int), ("x0", C.c_double), ("x1", C.c_double),
                ("y0", C.c_double), ("y1", C.c_double)]


class _VGrid(C.Structure):
    _fields_ = [("Nu", C.c_int), ("Nv", C.c_int), ("u", _dp), ("wu", _dp), ("v", _dp), ("wv", _dp)]


class _Gas(C.Structure):
    _fields_ = [("omega", C.c_double), ("mu_ref", C.c_double), ("Kn", C.c_double), ("Pr", C.c_double),
                ("K_int", C.c_int)]


class _BC(C.Structure):
    _fields_ = [("type", C.c_int), ("rho", C.c_double), ("U", C.c_double), ("V", C.c_double),
                ("T", C.c_double)]


class _BCs(C.Structure):
    _fields_ = [("xmin", _BC), ("xmax", _BC), ("ymin", _BC), ("ymax", _BC)]


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than its sources."""
    with _lock:
        stale = force or not os.path.exists(_SO) or any(
            os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
        if stale:
            tmp = _SO + f".tmp{os.getpid()}"
            cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                   _SRC[0], "-o", tmp, "-lm"]
            subprocess.run(cmd, check=True, cwd=_HERE)
            os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp = C.c_void_p
        L.ugkso_init.argtypes = [C.POINTER(vp), C.POINTER(_Mesh), C.POINTER(_VGrid), C.POINTER(_Gas),
                                 C.POINTER(_BCs), C.c_double]
        L.ugkso_set_state.argtypes = [vp, _dp, _dp]
        L.ugkso_step.argtypes = [vp, C.c_int]
        L.ugkso_moments.argtypes = [vp, _dp, _dp]
        L.ugkso_get_f.argtypes = [vp, _dp]
        L.ugkso_residual.argtypes = [vp, _dp]
        L.ugkso_dt.argtypes = [vp]; L.ugkso_dt.restype = C.c_double
        L.ugkso_mu_ref.argtypes = [vp]; L.ugkso_mu_ref.restype = C.c_double
        L.ugkso_step_count.argtypes = [vp]; L.ugkso_step_count.restype = C.c_long
        L.ugkso_set_threads.argtypes = [vp, C.c_int]; L.ugkso_set_threads.restype = None
        L.ugkso_set_tangential.argtypes = [vp, C.c_int]; L.ugkso_set_tangential.restype = None
        L.ugkso_destroy.argtypes = [vp]; L.ugkso_destroy.restype = None
        L.ugkso_face_flux.argtypes = [vp, C.c_int, C.c_int, C.c_int, _dp, _dp, _dp]
        L.ugkso_cell_update.argtypes = [vp, C.c_int, C.c_int, _dp, _dp]
        L.ugkso_prim_of_W.argtypes = [_dp, _dp]; L.ugkso_prim_of_W.restype = None
        L.ugkso_W_of_prim.argtypes = [_dp, _dp]; L.ugkso_W_of_prim.restype = None
        L.ugkso_maxwellian.argtypes = [_dp, C.c_double, C.c_double]; L.ugkso_maxwellian.restype = C.c_double
        L.ugkso_gauss_moments.argtypes = [_dp] * 5; L.ugkso_gauss_moments.restype = None
        L.ugkso_moment_T.argtypes = [_dp, C.c_int, _dp, C.c_int, C.c_int, _dp]; L.ugkso_moment_T.restype = None
        L.ugkso_micro_slope.argtypes = [_dp, _dp, _dp]; L.ugkso_micro_slope.restype = None
        L.ugkso_time_coeffs.argtypes = [C.c_double, C.c_double, _dp]; L.ugkso_time_coeffs.restype = None
        L.ugkso_van_leer.argtypes = [C.c_double, C.c_double]; L.ugkso_van_leer.restype = C.c_double
        L.ugkso_tau.argtypes = [C.c_double] * 4; L.ugkso_tau.restype = C.c_double
        L.ugkso_mu_ref_from_kn.argtypes = [C.c_double, C.c_double]; L.ugkso_mu_ref_from_kn.restype = C.c_double
        _lib = L
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _a(x, n=None) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    if n is not None:
        assert a.size == n, (a.size, n)
    return a


# ---- stateless closed-form pieces (pins) ----
def prim_of_W(W):
    o = np.empty(4); lib().ugkso_prim_of_W(_p(_a(W, 4)), _p(o)); return o


def W_of_prim(prim):
    o = np.empty(4); lib().ugkso_W_of_prim(_p(_a(prim, 4)), _p(o)); return o


def maxwellian(prim, u, v):
    return lib().ugkso_maxwellian(_p(_a(prim, 4)), float(u), float(v))


def gauss_moments(prim):
    ML, MR, Mu, Mv = (np.empty(7) for _ in range(4))
    lib().ugkso_gauss_moments(_p(_a(prim, 4)), _p(ML), _p(MR), _p(Mu), _p(Mv))
    return ML, MR, Mu, Mv


def moment_T(prim, X, c, alpha, beta):
    o = np.empty(4)
    cc = None if c is None else _p(_a(c, 4))
    lib().ugkso_moment_T(_p(_a(prim, 4)), {"Mu": 0, "ML": 1, "MR": 2}[X], cc, alpha, beta, _p(o))
    return o


def micro_slope(prim, s):
    o = np.empty(4); lib().ugkso_micro_slope(_p(_a(prim, 4)), _p(_a(s, 4)), _p(o)); return o


def time_coeffs(dt, tau):
    o = np.empty(5); lib().ugkso_time_coeffs(float(dt), float(tau), _p(o)); return o


def van_leer(a, b):
    return lib().ugkso_van_leer(float(a), float(b))


def tau(mu_ref, omega, rho, lam):
    return lib().ugkso_tau(float(mu_ref), float(omega), float(rho), float(lam))


def mu_ref_from_kn(Kn, omega):
    return lib().ugkso_mu_ref_from_kn(float(Kn), float(omega))


class OracleError(RuntimeError):
    pass


class Oracle:
    """One oracle context.  ``problem`` is a ``workloads.Problem``."""

    def __init__(self, problem, threads: int | None = None, tangential: bool = False):
        L = lib()
        p = problem
        self.I, self.J, self.Nu, self.Nv = p.I, p.J, len(p.u), len(p.v)
        self.N = self.Nu * self.Nv
        self._keep = [_a(p.u), _a(p.wu), _a(p.v), _a(p.wv)]
        mesh = _Mesh(p.I, p.J, p.x0, p.x1, p.y0, p.y1)
        vg = _VGrid(self.Nu, self.Nv, *[_p(a) for a in self._keep])
        gas = _Gas(p.omega, p.mu_ref, p.Kn, p.Pr, p.K_int)
        bcs = _BCs(*[_BC(int(b[0]), float(b[1]), float(b[2]), float(b[3]), float(b[4])) for b in p.bcs])
        h = C.c_void_p()
        rc = L.ugkso_init(C.byref(h), C.byref(mesh), C.byref(vg), C.byref(gas), C.byref(bcs), float(p.cfl))
        if rc:
            raise OracleError(f"ugkso_init -> {rc}")
        self._h = h
        if threads:
            L.ugkso_set_threads(h, int(threads))
        if tangential:
            L.ugkso_set_tangential(h, 1)

    def _chk(self, rc, what):
        if rc:
            raise OracleError(f"{what} -> {rc}")

    def close(self):
        if getattr(self, "_h", None):
            lib().ugkso_destroy(self._h); self._h = None

    __del__ = close

    @property
    def dt(self): return lib().ugkso_dt(self._h)

    @property
    def mu_ref(self): return lib().ugkso_mu_ref(self._h)

    @property
    def step_count(self): return lib().ugkso_step_count(self._h)

    def set_threads(self, n): lib().ugkso_set_threads(self._h, int(n))

    def set_state(self, W, f):
        W = _a(W, self.I * self.J * 4); f = _a(f, self.I * self.J * self.N)
        self._chk(lib().ugkso_set_state(self._h, _p(W), _p(f)), "ugkso_set_state")

    def step(self, n=1):
        self._chk(lib().ugkso_step(self._h, int(n)), "ugkso_step")

    def W(self):
        o = np.empty((self.J, self.I, 4)); self._chk(lib().ugkso_moments(self._h, _p(o), None), "ugkso_moments"); return o

    def W_of_f(self):
        o = np.empty((self.J, self.I, 4)); self._chk(lib().ugkso_moments(self._h, None, _p(o)), "ugkso_moments"); return o

    def f(self):
        o = np.empty((self.J, self.I, self.Nv, self.Nu)); self._chk(lib().ugkso_get_f(self._h, _p(o)), "ugkso_get_f"); return o

    def residual(self):
        o = np.empty(4); self._chk(lib().ugkso_residual(self._h, _p(o)), "ugkso_residual"); return o

    def face_flux(self, direction, i, j):
        FW = np.empty(4); Ff = np.empty((self.Nv, self.Nu)); st = np.empty(40)
        self._chk(lib().ugkso_face_flux(self._h, int(direction), int(i), int(j), _p(FW), _p(Ff), _p(st)),
                  "ugkso_face_flux")
        return FW, Ff, st

    def cell_update(self, i, j):
        Wn = np.empty(4); fn = np.empty((self.Nv, self.Nu))
        self._chk(lib().ugkso_cell_update(self._h, int(i), int(j), _p(Wn), _p(fn)), "ugkso_cell_update")
        return Wn, fn
