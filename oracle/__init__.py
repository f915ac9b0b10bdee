"""CPU ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT.

ctypes binding of ``oracle/ref_dg.cpp`` (see ``ref_dg.h``).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_1805_01443_b200``.

Two builds of the same source: ``libref_dg.so`` (single-threaded: the definition) and
``libref_dg_omp.so`` (``-fopenmp``: one ``parallel for`` over cell rows; results are
bitwise identical because cells are independent inside a stage).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ref_dg.cpp")
_FLAGS = ["-O2", "-ffp-contract=off", "-std=c++17", "-fPIC", "-shared", "-Wall", "-Wno-unknown-pragmas"]


def build(force: bool = False) -> None:
    """Compile both oracle libraries with g++ (no fast-math, no FMA contraction)."""
    for name, extra in (("libref_dg.so", []), ("libref_dg_omp.so", ["-fopenmp"])):
        out = os.path.join(_HERE, name)
        if (not force and os.path.exists(out)
                and os.path.getmtime(out) >= max(os.path.getmtime(_SRC),
                                                 os.path.getmtime(os.path.join(_HERE, "ref_dg.h")))):
            continue
        subprocess.check_call(["g++", *_FLAGS, *extra, _SRC, "-o", out])


class RefParams(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32),
        ("x0", C.c_double), ("x1", C.c_double), ("y0", C.c_double), ("y1", C.c_double),
        ("order", C.c_int32), ("rk", C.c_int32), ("bc", C.c_int32), ("eos", C.c_int32),
        ("gamma", C.c_double), ("h_aspect", C.c_double),
        ("gm_star", C.c_double), ("eps_star", C.c_double),
        ("q_planet", C.c_double), ("r_planet", C.c_double), ("eps_planet", C.c_double),
        ("omega_planet", C.c_double), ("phase0", C.c_double),
        ("damp_r0", C.c_double), ("damp_r1", C.c_double), ("t0", C.c_double),
        ("limiter", C.c_int32), ("lim_eps", C.c_double),
        ("flux", C.c_int32),
        ("damp_in_r0", C.c_double), ("damp_in_r1", C.c_double),
        ("damp_mode", C.c_int32),
    ]


def _to_struct(p: dict) -> RefParams:
    s = RefParams()
    for name, _ in RefParams._fields_:
        setattr(s, name, p[name])
    return s


_PD = C.POINTER(C.c_double)
_ODE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_double, _PD, _PD)
_libs: dict = {}


def _lib(omp: bool):
    key = bool(omp)
    if key in _libs:
        return _libs[key]
    build()
    L = C.CDLL(os.path.join(_HERE, "libref_dg_omp.so" if omp else "libref_dg.so"))
    vp, d, i = C.c_void_p, C.c_double, C.c_int
    PP = C.POINTER(RefParams)
    sig = {
        "ref_init": (i, [PP, C.POINTER(vp)]),
        "ref_set_state": (i, [vp, _PD]), "ref_get_state": (i, [vp, _PD]),
        "ref_rhs": (i, [vp, d, _PD]), "ref_cfl_dt": (i, [vp, d, _PD]),
        "ref_step": (i, [vp, d]), "ref_step_debug": (i, [vp, d, _PD]),
        "ref_time": (d, [vp]), "ref_set_time": (i, [vp, d]), "ref_destroy": (None, [vp]),
        "ref_tables": (i, [i, _PD, _PD, _PD, _PD, _PD, _PD]),
        "ref_point_flux": (i, [PP, _PD, d, d, i, _PD, _PD, _PD]),
        "ref_llf": (i, [PP, _PD, _PD, d, d, i, _PD]),
        "ref_hllc": (i, [PP, _PD, _PD, d, d, i, _PD]),
        "ref_gravity": (i, [PP, d, d, d, _PD]),
        "ref_rhs_parts": (i, [vp, d, i, _PD]), "ref_damp": (i, [vp, d]),
        "ref_load_working_state": (i, [vp, _PD]),
        "ref_rk_step": (i, [i, C.c_long, _PD, d, d, _ODE_FN, vp, _PD]),
        "ref_threads": (i, []), "ref_set_threads": (None, [i]),
        "ref_rk_stages": (i, [i]), "ref_limit": (i, [vp]), "ref_torque": (i, [vp, d, _PD]),
        "ref_torque_normalised": (i, [vp, d, d, _PD]),
        "ref_lobatto": (i, [i, _PD, _PD]), "ref_limit_cell": (i, [PP, _PD, _PD]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _libs[key] = L
    return L


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(_PD)


def _chk(e: int, what: str):
    if e != 0:
        raise RuntimeError(f"oracle: {what} failed ({e})")


class RefDG:
    """Host-memory twin of ``paper_1805_01443_b200.DG`` (names prefixed ``ref_`` in C)."""

    def __init__(self, params: dict, omp: bool = False, threads: int | None = None):
        self.L = _lib(omp)
        if omp and threads:
            self.L.ref_set_threads(int(threads))
        self.params = dict(params)
        self.m = params["order"]
        self.shape = (params["ny"], params["nx"], 4, self.m, self.m)
        self._h = C.c_void_p()
        _chk(self.L.ref_init(C.byref(_to_struct(params)), C.byref(self._h)), "ref_init")

    def close(self):
        if self._h:
            self.L.ref_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def threads(self) -> int:
        return int(self.L.ref_threads())

    def set_state(self, U: np.ndarray):
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.shape == self.shape
        _chk(self.L.ref_set_state(self._h, _p(U)), "ref_set_state")

    def load_working_state(self, U: np.ndarray):
        """Replace the working state; the snapshot U0 taken by set_state stays."""
        U = np.ascontiguousarray(U, dtype=np.float64)
        assert U.shape == self.shape
        _chk(self.L.ref_load_working_state(self._h, _p(U)), "ref_load_working_state")

    def get_state(self) -> np.ndarray:
        U = np.empty(self.shape)
        _chk(self.L.ref_get_state(self._h, _p(U)), "ref_get_state")
        return U

    def rhs(self, t: float, parts: int = 7) -> np.ndarray:
        out = np.empty(self.shape)
        _chk(self.L.ref_rhs_parts(self._h, float(t), int(parts), _p(out)), "ref_rhs")
        return out

    def cfl_dt(self, cfl: float) -> float:
        dt = C.c_double()
        _chk(self.L.ref_cfl_dt(self._h, float(cfl), C.byref(dt)), "ref_cfl_dt")
        return dt.value

    def step(self, dt: float):
        _chk(self.L.ref_step(self._h, float(dt)), "ref_step")

    def step_debug(self, dt: float) -> np.ndarray:
        st = np.empty((rk_stages(self.params["rk"]),) + self.shape)
        _chk(self.L.ref_step_debug(self._h, float(dt), _p(st)), "ref_step_debug")
        return st

    def limit(self):
        _chk(self.L.ref_limit(self._h), "ref_limit")

    def torque(self, t: float) -> float:
        g = C.c_double()
        _chk(self.L.ref_torque(self._h, float(t), C.byref(g)), "ref_torque")
        return g.value

    def torque_normalised(self, t: float, sigma_p: float) -> float:
        """gamma Gamma / Gamma_0."""
        g = C.c_double()
        _chk(self.L.ref_torque_normalised(self._h, float(t), float(sigma_p), C.byref(g)), "ref_torque_normalised")
        return g.value

    def damp(self, dt: float):
        _chk(self.L.ref_damp(self._h, float(dt)), "ref_damp")

    @property
    def time(self) -> float:
        return float(self.L.ref_time(self._h))

    @time.setter
    def time(self, t: float):
        _chk(self.L.ref_set_time(self._h, float(t)), "ref_set_time")


# ---- pieces, for the pin tests ----------------------------------------------------------------
def rk_stages(rk: int) -> int:
    """Sub-steps per time step: 2, 3, 5 (rk 4: SSP-RK(5,4)), 6 (rk 5: Cash-Karp)."""
    return int(_lib(False).ref_rk_stages(int(rk)))


def lobatto(m: int):
    """Gauss-Lobatto nodes on [-1,1] and weights normalised to sum 1 used by the limiter of order m."""
    xh, wh = np.empty(4), np.empty(4)
    n = _lib(False).ref_lobatto(int(m), _p(xh), _p(wh))
    if n < 0:
        raise RuntimeError("oracle: ref_lobatto failed")
    return xh[:n].copy(), wh[:n].copy()


def limit_cell(params: dict, u: np.ndarray):
    """C12 on one cell u[4][m][m]; returns (limited copy, theta1, theta2)."""
    u = np.array(u, dtype=np.float64).copy()
    th = np.empty(2)
    _chk(_lib(False).ref_limit_cell(C.byref(_to_struct(params)), _p(u), _p(th)), "ref_limit_cell")
    return u, float(th[0]), float(th[1])


def tables(m: int) -> dict:
    L = _lib(False)
    xi, w, Ep, Em = (np.empty(m) for _ in range(4))
    B, D = np.empty((m, m)), np.empty((m, m))
    _chk(L.ref_tables(m, _p(xi), _p(w), _p(B), _p(D), _p(Ep), _p(Em)), "ref_tables")
    return dict(xi=xi, w=w, B=B, D=D, Ep=Ep, Em=Em)


def point_flux(params: dict, U4, x: float, y: float, direction: int):
    L = _lib(False)
    U4 = np.ascontiguousarray(U4, dtype=np.float64)
    F = np.empty(4)
    vn, c = C.c_double(), C.c_double()
    _chk(L.ref_point_flux(C.byref(_to_struct(params)), _p(U4), x, y, direction, _p(F),
                          C.byref(vn), C.byref(c)), "ref_point_flux")
    return F, vn.value, c.value


def llf(params: dict, UL, UR, x: float, y: float, direction: int) -> np.ndarray:
    L = _lib(False)
    UL = np.ascontiguousarray(UL, dtype=np.float64)
    UR = np.ascontiguousarray(UR, dtype=np.float64)
    H = np.empty(4)
    _chk(L.ref_llf(C.byref(_to_struct(params)), _p(UL), _p(UR), x, y, direction, _p(H)), "ref_llf")
    return H


def hllc(params: dict, UL, UR, x: float, y: float, direction: int) -> np.ndarray:
    """C5b: HLLC (eos 0) / HLL (eos 1) flux across a face with normal +direction."""
    L = _lib(False)
    UL = np.ascontiguousarray(UL, dtype=np.float64)
    UR = np.ascontiguousarray(UR, dtype=np.float64)
    H = np.empty(4)
    _chk(L.ref_hllc(C.byref(_to_struct(params)), _p(UL), _p(UR), x, y, direction, _p(H)), "ref_hllc")
    return H


def gravity(params: dict, t: float, x: float, y: float) -> np.ndarray:
    L = _lib(False)
    g = np.empty(2)
    _chk(L.ref_gravity(C.byref(_to_struct(params)), t, x, y, _p(g)), "ref_gravity")
    return g


def rk_step(rk: int, y: np.ndarray, t: float, dt: float, f, want_stages: bool = False):
    """One SSP-RK step of y' = f(t, y) with the oracle's own integrator (C8)."""
    L = _lib(False)
    y = np.array(y, dtype=np.float64).ravel().copy()
    n = y.size

    def cb(_user, tt, yp, dp):
        yy = np.ctypeslib.as_array(yp, shape=(n,))
        np.ctypeslib.as_array(dp, shape=(n,))[:] = f(tt, yy.copy())

    st = np.empty((rk_stages(rk), n)) if want_stages else None
    _chk(L.ref_rk_step(rk, n, _p(y), t, dt, _ODE_FN(cb), None,
                       _p(st) if want_stages else None), "ref_rk_step")
    return (y, st) if want_stages else y
