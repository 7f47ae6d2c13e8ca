"""ctypes binding of the ORACLE (oracle/cholla_ref.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares no code with paper_1410_4194_b200 and never imports it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cholla_ref.cpp")
_LIB = os.path.join(_HERE, "libcholla_ref.so")

PERIODIC, REFLECTIVE, OUTFLOW, NOH = 1, 2, 3, 4
PPMC, PLMC, PCM, PPMP, PLMP = 0, 1, 2, 3, 4


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, no FMA contraction).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", _SRC, "-o", _LIB + ".tmp%d" % os.getpid()]
        subprocess.check_call(cmd)
        os.replace(cmd[-1], _LIB)
    return _LIB


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.ref_init.restype = C.c_void_p
        L.ref_init.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.POINTER(C.c_int)]
        L.ref_free.argtypes = [C.c_void_p]
        L.ref_set_spacing.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_double]
        L.ref_padded_cells.restype = C.c_long
        L.ref_padded_cells.argtypes = [C.c_void_p]
        for name in ("ref_set_state", "ref_get_state", "ref_set_padded", "ref_get_padded"):
            getattr(L, name).argtypes = [C.c_void_p, dp]
        L.ref_compute_dt.restype = C.c_double
        L.ref_compute_dt.argtypes = [C.c_void_p, C.c_double]
        L.ref_step.argtypes = [C.c_void_p, C.c_double]
        L.ref_last_error.restype = C.c_char_p
        L.ref_cons_to_prim.argtypes = [C.c_double, dp, dp]
        L.ref_prim_to_cons.argtypes = [C.c_double, dp, dp]
        L.ref_char_project.argtypes = [C.c_double, C.c_double, dp, dp]
        L.ref_char_backproject.argtypes = [C.c_double, C.c_double, dp, dp]
        L.ref_limited_slope.argtypes = [C.c_double, dp, dp, dp, dp]
        L.ref_ppmc_cell.argtypes = [C.c_double, C.c_double, dp, dp]
        L.ref_riemann_exact.argtypes = [C.c_double, dp, dp, dp, dp]
        L.ref_riemann_roe.argtypes = [C.c_double, dp, dp, dp]
        L.ref_riemann_roe.restype = C.c_int
        L.ref_set_solver.argtypes = [C.c_void_p, C.c_int]
        L.ref_set_reconstruction.argtypes = [C.c_void_p, C.c_int]
        L.ref_set_hcorrection.argtypes = [C.c_void_p, C.c_int]
        L.ref_riemann_roe_eta.argtypes = [C.c_double, dp, dp, C.c_double, dp]
        L.ref_riemann_roe_eta.restype = C.c_int
        L.ref_plmc_cell.argtypes = [C.c_double, C.c_double, dp, dp]
        L.ref_ppmp_cell.argtypes = [C.c_double, C.c_double, dp, dp]
        L.ref_plmp_cell.argtypes = [C.c_double, C.c_double, dp, dp]
        L.ref_set_noh.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.ref_set_time.argtypes = [C.c_void_p, C.c_double]
        L.ref_get_time.argtypes = [C.c_void_p]
        L.ref_get_time.restype = C.c_double
        L.ref_fill_ghosts.argtypes = [C.c_void_p]
        _lib = L
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _arr(x) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(x, dtype=np.float64))


class RefGrid:
    """Same call surface as the product's Grid (init / set_state / compute_dt / step / get_state)."""

    def __init__(self, nx, ny, nz, nghost=3, gamma=1.4, bc=(PERIODIC,) * 6):
        bc_arr = (C.c_int * 6)(*[int(b) for b in bc])
        self._h = lib().ref_init(nx, ny, nz, nghost, gamma, bc_arr)
        if not self._h:
            raise ValueError("ref_init: " + lib().ref_last_error().decode())
        self.shape = (nz, ny, nx)
        self.nghost = nghost
        g = [nghost if n > 1 else 0 for n in (nz, ny, nx)]
        self.padded_shape = tuple(n + 2 * gg for n, gg in zip(self.shape, g))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().ref_free(self._h)
            self._h = None

    def set_spacing(self, dx, dy, dz):
        if lib().ref_set_spacing(self._h, dx, dy, dz) != 0:
            raise ValueError(lib().ref_last_error().decode())

    def set_state(self, u):
        u = _arr(u)
        assert u.shape == (5,) + self.shape, u.shape
        lib().ref_set_state(self._h, _p(u))

    def get_state(self) -> np.ndarray:
        u = np.empty((5,) + self.shape)
        if lib().ref_get_state(self._h, _p(u)) != 0:
            raise RuntimeError(lib().ref_last_error().decode())
        return u

    def set_padded(self, up):
        up = _arr(up)
        assert up.shape == (5,) + self.padded_shape, (up.shape, self.padded_shape)
        lib().ref_set_padded(self._h, _p(up))

    def get_padded(self) -> np.ndarray:
        up = np.empty((5,) + self.padded_shape)
        lib().ref_get_padded(self._h, _p(up))
        return up

    def compute_dt(self, cfl) -> float:
        return float(lib().ref_compute_dt(self._h, cfl))

    def set_solver(self, solver):
        """0 = exact (default), 1 = Roe with the HLLE failsafe (the solver is selectable)."""
        if lib().ref_set_solver(self._h, int(solver)) != 0:
            raise ValueError("ref_set_solver: " + lib().ref_last_error().decode())

    def set_hcorrection(self, on):
        """H correction (Appendix C): Roe solver only, nghost >= 4."""
        if lib().ref_set_hcorrection(self._h, int(bool(on))) != 0:
            raise ValueError("ref_set_hcorrection: " + lib().ref_last_error().decode())

    def set_reconstruction(self, recon):
        """0 = PPMC (default), 1 = PLMC, 2 = PCM, 3 = PPMP (nghost >= 4), 4 = PLMP."""
        if lib().ref_set_reconstruction(self._h, int(recon)) != 0:
            raise ValueError("ref_set_reconstruction: " + lib().ref_last_error().decode())

    def set_noh(self, rho0=1.0, p0=1e-6):
        """Ambient state of the analytic Noh boundary (faces with bc code NOH)."""
        if lib().ref_set_noh(self._h, rho0, p0) != 0:
            raise ValueError("ref_set_noh: " + lib().ref_last_error().decode())

    def set_time(self, t):
        lib().ref_set_time(self._h, float(t))

    def get_time(self) -> float:
        return float(lib().ref_get_time(self._h))

    def fill_ghosts(self):
        lib().ref_fill_ghosts(self._h)

    def step(self, dt):
        if lib().ref_step(self._h, dt) != 0:
            raise ValueError("ref_step: " + lib().ref_last_error().decode())


# ---- unit-level functions (primitive variables, direction-local order) -----------------------
def cons_to_prim(gamma, u):
    u = _arr(u); w = np.empty(5)
    lib().ref_cons_to_prim(gamma, _p(u), _p(w))
    return w


def prim_to_cons(gamma, w):
    w = _arr(w); u = np.empty(5)
    lib().ref_prim_to_cons(gamma, _p(w), _p(u))
    return u


def char_project(rho, a, dw):
    dw = _arr(dw); out = np.empty(5)
    lib().ref_char_project(rho, a, _p(dw), _p(out))
    return out


def char_backproject(rho, a, dxi):
    dxi = _arr(dxi); out = np.empty(5)
    lib().ref_char_backproject(rho, a, _p(dxi), _p(out))
    return out


def limited_slope(gamma, wm, w0, wp):
    wm, w0, wp = _arr(wm), _arr(w0), _arr(wp); out = np.empty(5)
    lib().ref_limited_slope(gamma, _p(wm), _p(w0), _p(wp), _p(out))
    return out


def ppmc_cell(gamma, dtdx, w):
    """w[5 cells i-2..i+2][5 comps] -> (WL, WR, WLstar, WRstar)."""
    w = _arr(w); assert w.shape == (5, 5)
    out = np.empty((4, 5))
    lib().ref_ppmc_cell(gamma, dtdx, _p(w), _p(out))
    return out[0], out[1], out[2], out[3]


def ppmp_cell(gamma, dtdx, w):
    """w[7 cells i-3..i+3][5 comps] -> (WL, WR, WLstar, WRstar), A.4."""
    w = _arr(w); assert w.shape == (7, 5)
    out = np.empty((4, 5))
    lib().ref_ppmp_cell(gamma, dtdx, _p(w), _p(out))
    return out[0], out[1], out[2], out[3]


def plmp_cell(gamma, dtdx, w):
    """w[7 cells][5 comps] (only i-1..i+1 are read) -> (WL, WR, WLstar, WRstar), A.1."""
    w = _arr(w); assert w.shape == (7, 5)
    out = np.empty((4, 5))
    lib().ref_plmp_cell(gamma, dtdx, _p(w), _p(out))
    return out[0], out[1], out[2], out[3]


def riemann_exact(gamma, WL, WR):
    """-> (flux[5], dict(pm, um, rho, u, p, iters, region))."""
    WL, WR = _arr(WL), _arr(WR)
    f = np.empty(5); d = np.empty(7)
    lib().ref_riemann_exact(gamma, _p(WL), _p(WR), _p(f), _p(d))
    return f, dict(pm=d[0], um=d[1], rho=d[2], u=d[3], p=d[4], iters=int(d[5]), region=int(d[6]))


ROE_PATHS = ("F_L", "F_R", "roe", "hlle")


def riemann_roe(gamma, WL, WR):
    """Roe solver with the HLLE failsafe (B.2) -> (flux[5], path) with path in ROE_PATHS."""
    WL, WR = _arr(WL), _arr(WR)
    f = np.empty(5)
    path = lib().ref_riemann_roe(gamma, _p(WL), _p(WR), _p(f))
    return f, ROE_PATHS[path]


def plmc_cell(gamma, dtdx, w):
    """PLMC (A.2): w[5 cells i-2..i+2][5 comps] (only i-1..i+1 used) -> (WL, WR, WLstar, WRstar)."""
    w = _arr(w); assert w.shape == (5, 5)
    out = np.empty((4, 5))
    lib().ref_plmc_cell(gamma, dtdx, _p(w), _p(out))
    return out[0], out[1], out[2], out[3]


def riemann_roe_eta(gamma, WL, WR, eta_h):
    """Roe solver with |lambda| -> max(|lambda|, eta_h) in B28 (H correction, C3) -> (flux[5], path)."""
    WL, WR = _arr(WL), _arr(WR)
    f = np.empty(5)
    path = lib().ref_riemann_roe_eta(gamma, _p(WL), _p(WR), float(eta_h), _p(f))
    return f, ROE_PATHS[path]
