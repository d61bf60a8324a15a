"""ctypes wrapper of the CPU ORACLE (oracle/mmo.h).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It shares nothing with the CUDA
library or its binding (paper_2401_15233_b200/); neither imports the other.

`build()` compiles oracle/*.c with gcc (-O2 -ffp-contract=off: no FMA contraction, IEEE
evaluation order as written) into oracle/libmmo.so.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_LIB_PATH = _HERE / "libmmo.so"
_SOURCES = ["mmo_moments.c", "mmo_scheme.c"]

SYS5_1D, SYS14_2D = 5, 14
TAU_NONE, TAU_CONST, TAU_KN = 0, 1, 2
BC_TRANSMISSIVE, BC_PERIODIC, BC_DIRICHLET = 0, 1, 2
LIM_NONE, LIM_MINMOD, LIM_VANALBADA = 0, 1, 2
FLUX_HLL, FLUX_RUSANOV = 0, 1
SRC_EXPLICIT, SRC_POINT_IMPLICIT = 0, 1      # BGK source: forward Euler | point-implicit
TIME_EULER, TIME_MIDPOINT = 0, 1             # forward Euler | midpoint (2nd-order RK)
OK, EINVAL, ENONFINITE = 0, -1, -4


def build(force: bool = False) -> Path:
    srcs = [_HERE / s for s in _SOURCES] + [_HERE / "mmo.h"]
    if not force and _LIB_PATH.exists() and all(
            _LIB_PATH.stat().st_mtime >= s.stat().st_mtime for s in srcs):
        return _LIB_PATH
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-fPIC", "-shared", "-Wall", "-Wextra", "-o", str(_LIB_PATH)]
    cmd += [str(_HERE / s) for s in _SOURCES] + ["-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB_PATH


class _Grid(C.Structure):
    _fields_ = [("system", C.c_int), ("nx", C.c_int), ("ny", C.c_int),
                ("x0", C.c_double), ("x1", C.c_double), ("y0", C.c_double), ("y1", C.c_double)]


class _Collision(C.Structure):
    _fields_ = [("model", C.c_int), ("tau", C.c_double), ("Kn", C.c_double),
                ("L_ref", C.c_double), ("rho_ref", C.c_double)]


class _BC(C.Structure):
    _fields_ = [("type", C.c_int), ("nbands", C.c_int),
                ("band_lo", C.POINTER(C.c_double)), ("band_hi", C.POINTER(C.c_double)),
                ("band_W", C.POINTER(C.c_double)), ("default_W", C.POINTER(C.c_double))]


class _Options(C.Structure):
    _fields_ = [("sigma_lim", C.c_double), ("ws_scale", C.c_double), ("limiter", C.c_int),
                ("shared_limiter", C.c_int), ("flux", C.c_int), ("source_scheme", C.c_int),
                ("time_scheme", C.c_int), ("nthreads", C.c_int)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is not None:
        return _lib
    _lib = bind(C.CDLL(str(build())))
    return _lib


def bind(L):
    """Attach the argument / result types of oracle/mmo.h to a loaded library."""
    d, i, p = C.c_double, C.c_int, _dp
    sig = {
        "mmo_cons2prim5": (None, [p, p]), "mmo_prim2cons5": (None, [p, p]),
        "mmo_sigma5": (d, [d, d]), "mmo_sstar5": (d, [d, d]),
        "mmo_closure5": (d, [p, d, p, p]),
        "mmo_flux5_given_s": (None, [p, d, p]), "mmo_flux5": (None, [p, d, p]),
        "mmo_wavespeed5": (None, [p, d, d, p, p]), "mmo_source5": (None, [p, d, p]),
        "mmo_cons2prim14": (None, [p, p]), "mmo_prim2cons14": (None, [p, p]),
        "mmo_sigma14": (d, [p]),
        "mmo_closure14": (None, [p, d, p, p, p, p, p]),
        "mmo_flux14_given_closure": (None, [p, p, p, p, i, p]),
        "mmo_flux14": (None, [p, i, d, p]),
        "mmo_wavespeed14_star": (d, [d, d, d, d]),
        "mmo_wavespeed14": (None, [p, i, d, d, p, p]),
        "mmo_source14": (None, [p, d, p]),
        "mmo_tau": (d, [i, d, d, d, d, d, d]),
        "mmo_limiter_psi": (d, [i, d, d]), "mmo_limited_slope": (d, [i, d, d]),
        "mmo_numflux": (None, [i, i, p, p, p, p, d, d, d, d, p]),
        "mmo_face_states": (None, [i, i, i, p, p, p, p, p]),
        "mmo_create": (i, [C.POINTER(C.c_void_p), C.POINTER(_Grid), C.POINTER(_Collision),
                           C.POINTER(_BC), C.POINTER(_Options)]),
        "mmo_set_state": (i, [C.c_void_p, p]), "mmo_set_state_prim": (i, [C.c_void_p, p]),
        "mmo_get_state": (i, [C.c_void_p, p]), "mmo_get_state_prim": (i, [C.c_void_p, p]),
        "mmo_cfl_dt": (d, [C.c_void_p, d]),
        "mmo_step": (i, [C.c_void_p, i, d]), "mmo_step_fixed_dt": (i, [C.c_void_p, i, d]),
        "mmo_advance_to": (i, [C.c_void_p, d, d, i]),
        "mmo_get_info": (i, [C.c_void_p, p, C.POINTER(C.c_longlong), p, p]),
        "mmo_threads_used": (i, [C.c_void_p]),
        "mmo_destroy": (None, [C.c_void_p]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    return L


def _arr(x, n=None):
    a = np.ascontiguousarray(x, dtype=np.float64)
    if n is not None:
        assert a.size == n, (a.size, n)
    return a


def _ptr(a):
    return a.ctypes.data_as(_dp)


# ------------------------------------------------------------------ pointwise functions
def cons2prim(U):
    U = _arr(U); W = np.empty_like(U)
    (lib().mmo_cons2prim5 if U.size == 5 else lib().mmo_cons2prim14)(_ptr(U), _ptr(W))
    return W


def prim2cons(W):
    W = _arr(W); U = np.empty_like(W)
    (lib().mmo_prim2cons5 if W.size == 5 else lib().mmo_prim2cons14)(_ptr(W), _ptr(U))
    return U


def sigma5(qs, rs):
    return lib().mmo_sigma5(qs, rs)


def sstar5(qs, sb):
    return lib().mmo_sstar5(qs, sb)


def closure5(W, sigma_lim):
    W = _arr(W, 5); sg = C.c_double(); sb = C.c_double()
    s = lib().mmo_closure5(_ptr(W), sigma_lim, C.byref(sg), C.byref(sb))
    return s, sg.value, sb.value


def flux5(W, sigma_lim):
    W = _arr(W, 5); F = np.empty(5)
    lib().mmo_flux5(_ptr(W), sigma_lim, _ptr(F))
    return F


def flux5_given_s(W, s):
    W = _arr(W, 5); F = np.empty(5)
    lib().mmo_flux5_given_s(_ptr(W), s, _ptr(F))
    return F


def wavespeed5(W, sigma_lim, k=1.0):
    W = _arr(W, 5); a = C.c_double(); b = C.c_double()
    lib().mmo_wavespeed5(_ptr(W), sigma_lim, k, C.byref(a), C.byref(b))
    return a.value, b.value


def source5(W, tau):
    W = _arr(W, 5); Cc = np.empty(5)
    lib().mmo_source5(_ptr(W), tau, _ptr(Cc))
    return Cc


def sigma14(W):
    return lib().mmo_sigma14(_ptr(_arr(W, 14)))


def closure14(W, sigma_lim):
    """-> sigma, sigma_bar, Q[3,3,3], R2[3,3], S[3] (dimensional)."""
    W = _arr(W, 14); sg = C.c_double(); sb = C.c_double()
    Q = np.empty((3, 3, 3)); R2 = np.empty((3, 3)); S = np.empty(3)
    lib().mmo_closure14(_ptr(W), sigma_lim, C.byref(sg), C.byref(sb), _ptr(Q), _ptr(R2), _ptr(S))
    return sg.value, sb.value, Q, R2, S


def flux14_given_closure(W, Q, R2, S, k):
    W = _arr(W, 14); Q = _arr(Q, 27); R2 = _arr(R2, 9); S = _arr(S, 3); F = np.empty(14)
    lib().mmo_flux14_given_closure(_ptr(W), _ptr(Q), _ptr(R2), _ptr(S), k, _ptr(F))
    return F


def flux14(W, k, sigma_lim):
    W = _arr(W, 14); F = np.empty(14)
    lib().mmo_flux14(_ptr(W), k, sigma_lim, _ptr(F))
    return F


def wavespeed14_star(Pdd, qd, qt, sb):
    return lib().mmo_wavespeed14_star(Pdd, qd, qt, sb)


def wavespeed14(W, d, sigma_lim, k=1.0):
    W = _arr(W, 14); a = C.c_double(); b = C.c_double()
    lib().mmo_wavespeed14(_ptr(W), d, sigma_lim, k, C.byref(a), C.byref(b))
    return a.value, b.value


def source14(W, tau):
    W = _arr(W, 14); Cc = np.empty(14)
    lib().mmo_source14(_ptr(W), tau, _ptr(Cc))
    return Cc


def tau(model, tau_const, Kn, L_ref, rho_ref, rho, P):
    return lib().mmo_tau(model, tau_const, Kn, L_ref, rho_ref, rho, P)


def limiter_psi(limiter, dm, dp):
    return lib().mmo_limiter_psi(limiter, dm, dp)


def limited_slope(limiter, dm, dp):
    return lib().mmo_limited_slope(limiter, dm, dp)


def face_states(limiter, shared, Wm, W0, Wp):
    """MUSCL face states (low, high) of the middle cell (L262-266)."""
    Wm, W0, Wp = _arr(Wm), _arr(W0), _arr(Wp)
    n = W0.size
    lo, hi = np.empty(n), np.empty(n)
    lib().mmo_face_states(n, limiter, int(shared), _ptr(Wm), _ptr(W0), _ptr(Wp), _ptr(lo), _ptr(hi))
    return lo, hi


def numflux(flux, FL, FR, UL, UR, lminL, lmaxL, lminR, lmaxR):
    FL, FR, UL, UR = map(_arr, (FL, FR, UL, UR)); out = np.empty_like(FL)
    lib().mmo_numflux(flux, FL.size, _ptr(FL), _ptr(FR), _ptr(UL), _ptr(UR),
                      lminL, lmaxL, lminR, lmaxR, _ptr(out))
    return out


# ------------------------------------------------------------------------------- solver
class Solver:
    """Oracle solver object.  `bcs` is a list of 4 dicts (xlo, xhi, ylo, yhi):
    {"type": BC_*, "bands": [(lo, hi, W), ...], "default": W or None}."""

    def __init__(self, system, nx, ny=1, extent=(0.0, 1.0, 0.0, 1.0), collision=None, bcs=None,
                 sigma_lim=1e-4, ws_scale=1.0, limiter=LIM_MINMOD, shared_limiter=0,
                 flux=FLUX_HLL, source_scheme=0, time_scheme=0, nthreads=0):
        L = lib()
        self.nm, self.nx, self.ny = system, nx, ny
        g = _Grid(system, nx, ny, *extent)
        col = collision or {"model": TAU_NONE}
        c = _Collision(col.get("model", TAU_NONE), col.get("tau", 0.0), col.get("Kn", 0.0),
                       col.get("L_ref", 1.0), col.get("rho_ref", 1.0))
        bcs = bcs or [{"type": BC_TRANSMISSIVE}] * 4
        keep = []
        arr = (_BC * 4)()
        for k in range(4):
            b = bcs[k] if k < len(bcs) else {"type": BC_TRANSMISSIVE}
            bands = b.get("bands", [])
            lo = _arr([x[0] for x in bands]); hi = _arr([x[1] for x in bands])
            bw = _arr([x[2] for x in bands]).reshape(-1)
            dflt = b.get("default")
            dw = _arr(dflt, system) if dflt is not None else None
            keep += [lo, hi, bw, dw]
            arr[k] = _BC(b["type"], len(bands), _ptr(lo), _ptr(hi), _ptr(bw),
                         _ptr(dw) if dw is not None else None)
        o = _Options(sigma_lim, ws_scale, limiter, shared_limiter, flux, source_scheme, time_scheme, nthreads)
        h = C.c_void_p()
        rc = L.mmo_create(C.byref(h), C.byref(g), C.byref(c), arr, C.byref(o))
        if rc != OK:
            raise ValueError(f"mmo_create failed: {rc}")
        self._h = h
        self._L = L

    def _chk(self, rc):
        if rc != OK:
            raise RuntimeError(f"oracle error {rc}")

    def set_state(self, U):
        self._chk(self._L.mmo_set_state(self._h, _ptr(_arr(U, self.nm * self.ny * self.nx))))

    def set_state_prim(self, W):
        self._chk(self._L.mmo_set_state_prim(self._h, _ptr(_arr(W, self.nm * self.ny * self.nx))))

    def get_state(self):
        U = np.empty((self.nm, self.ny, self.nx))
        self._chk(self._L.mmo_get_state(self._h, _ptr(U)))
        return U

    def get_state_prim(self):
        W = np.empty((self.nm, self.ny, self.nx))
        self._chk(self._L.mmo_get_state_prim(self._h, _ptr(W)))
        return W

    def cfl_dt(self, cfl):
        return self._L.mmo_cfl_dt(self._h, cfl)

    def step(self, n, cfl):
        self._chk(self._L.mmo_step(self._h, n, cfl))

    def step_fixed_dt(self, n, dt):
        self._chk(self._L.mmo_step_fixed_dt(self._h, n, dt))

    def advance_to(self, t_end, cfl, max_steps=0):
        self._chk(self._L.mmo_advance_to(self._h, t_end, cfl, max_steps))

    def info(self, with_speed=False):
        t = C.c_double(); n = C.c_longlong(); dt = C.c_double(); sp = C.c_double()
        self._chk(self._L.mmo_get_info(self._h, C.byref(t), C.byref(n), C.byref(dt),
                                       C.byref(sp) if with_speed else None))
        return {"t": t.value, "steps": n.value, "last_dt": dt.value,
                "max_speed": sp.value if with_speed else None}

    @property
    def threads(self):
        return self._L.mmo_threads_used(self._h)

    def close(self):
        if self._h:
            self._L.mmo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
