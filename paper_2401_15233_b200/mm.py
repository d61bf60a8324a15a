"""Thin ctypes binding of include/mm.h (argument marshalling only).

Every function below forwards to the C-ABI entry point of the same name in libmm.so; device
memory and the stream come from PyTorch (plumbing).  Nothing here computes any step of the
method and nothing falls back to a CPU path: a missing library or device raises.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np

from . import build_ext

SYS5_1D, SYS14_2D = 5, 14
TAU_NONE, TAU_CONST, TAU_KN = 0, 1, 2
BC_TRANSMISSIVE, BC_PERIODIC, BC_DIRICHLET = 0, 1, 2
STATE_PRIMITIVE, STATE_MAXWELLIAN = 0, 1     # mm_bc.band_state: W[nmom] | (rho, u_x, u_y, u_z, T)
LIM_NONE, LIM_MINMOD, LIM_VANALBADA = 0, 1, 2
FLUX_HLL, FLUX_RUSANOV = 0, 1
SRC_EXPLICIT, SRC_POINT_IMPLICIT = 0, 1      # BGK source: forward Euler | point-implicit
TIME_EULER, TIME_MIDPOINT = 0, 1             # forward Euler | midpoint (2nd-order RK)
OK, EINVAL, EWORKSPACE, ECUDA, ENONFINITE, ETOOLARGE = 0, -1, -2, -3, -4, -5
MAX_BANDS = 8
STATIC5_MAX_NX = 8192                         # mm_static5_run: cells the built-in 4 MiB scratch holds

EXPORTS = ["mm_workspace_bytes", "mm_create", "mm_set_state", "mm_set_state_prim", "mm_step",
           "mm_step_fixed_dt", "mm_advance_to", "mm_get_state", "mm_get_state_prim", "mm_get_info",
           "mm_cfl_dt", "mm_get_dt_history", "mm_set_clock", "mm_decomposition", "mm_launch_count", "mm_profile_begin", "mm_profile_end",
           "mm_set_fast_path", "mm_fast_path_active",
           "mm_destroy", "mm_strerror",
           "mm_batch5_workspace_bytes", "mm_batch5_create", "mm_batch5_set_state_prim", "mm_batch5_step",
           "mm_batch5_step_fixed_dt", "mm_batch5_advance_to", "mm_batch5_get_state", "mm_batch5_get_info",
           "mm_batch5_launch_count", "mm_batch5_destroy", "mm_static5_run"]
BENCH_EXPORTS = ["mm_measure_fp64_peak", "mm_measure_fp64_operand_rates", "mm_selftest_fastmath"]          # include/mm_bench.h, libmm_bench.so

_dp = C.POINTER(C.c_double)


class mm_grid(C.Structure):
    _fields_ = [("system", C.c_int), ("nx", C.c_int), ("ny", C.c_int),
                ("x0", C.c_double), ("x1", C.c_double), ("y0", C.c_double), ("y1", C.c_double)]


class mm_gas(C.Structure):
    _fields_ = [("R_gas", C.c_double)]


class mm_collision(C.Structure):
    _fields_ = [("model", C.c_int), ("tau", C.c_double), ("Kn", C.c_double),
                ("L_ref", C.c_double), ("rho_ref", C.c_double)]


class mm_bc(C.Structure):
    _fields_ = [("type", C.c_int), ("nbands", C.c_int), ("band_lo", _dp), ("band_hi", _dp),
                ("band_W", _dp), ("default_W", _dp), ("band_state", C.c_int)]


class mm_options(C.Structure):
    _fields_ = [("sigma_lim", C.c_double), ("ws_scale", C.c_double), ("limiter", C.c_int),
                ("shared_limiter", C.c_int), ("flux", C.c_int), ("source_scheme", C.c_int),
                ("time_scheme", C.c_int), ("stream", C.c_void_p)]


class MMError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"mm error {status}: {msg}")
        self.status = status


_lib = None


def lib() -> C.CDLL:
    """Load libmm.so (building it in-tree if the sources are newer).  Raises if impossible."""
    global _lib
    if _lib is not None:
        return _lib
    path = build_ext.build()
    L = C.CDLL(str(path))
    vp, i, d = C.c_void_p, C.c_int, C.c_double
    L.mm_workspace_bytes.restype, L.mm_workspace_bytes.argtypes = C.c_size_t, [C.POINTER(mm_grid)]
    L.mm_create.restype = i
    L.mm_create.argtypes = [C.POINTER(vp), C.POINTER(mm_grid), C.POINTER(mm_gas), C.POINTER(mm_collision),
                            C.POINTER(mm_bc), C.POINTER(mm_options), vp, C.c_size_t]
    for name in ("mm_set_state", "mm_set_state_prim", "mm_get_state", "mm_get_state_prim"):
        f = getattr(L, name)
        f.restype, f.argtypes = i, [vp, vp, i]
    L.mm_step.restype, L.mm_step.argtypes = i, [vp, i, d]
    L.mm_step_fixed_dt.restype, L.mm_step_fixed_dt.argtypes = i, [vp, i, d]
    L.mm_advance_to.restype, L.mm_advance_to.argtypes = i, [vp, d, d, i]
    L.mm_get_info.restype = i
    L.mm_get_info.argtypes = [vp, _dp, C.POINTER(C.c_longlong), _dp, _dp]
    L.mm_cfl_dt.restype, L.mm_cfl_dt.argtypes = i, [vp, d, _dp]
    L.mm_get_dt_history.restype, L.mm_get_dt_history.argtypes = i, [vp, C.c_longlong, i, _dp]
    L.mm_set_clock.restype, L.mm_set_clock.argtypes = i, [vp, d, C.c_longlong]
    ip = C.POINTER(C.c_int)
    L.mm_decomposition.restype, L.mm_decomposition.argtypes = i, [i, i, i, i, ip, ip, ip]
    L.mm_launch_count.restype, L.mm_launch_count.argtypes = C.c_longlong, [vp]
    L.mm_profile_begin.restype, L.mm_profile_begin.argtypes = i, [vp]
    L.mm_profile_end.restype = i
    L.mm_profile_end.argtypes = [vp, _dp, C.POINTER(C.c_longlong)]
    L.mm_set_fast_path.restype, L.mm_set_fast_path.argtypes = i, [vp, i]
    L.mm_fast_path_active.restype, L.mm_fast_path_active.argtypes = i, [vp]
    L.mm_destroy.restype, L.mm_destroy.argtypes = None, [vp]
    L.mm_batch5_workspace_bytes.restype, L.mm_batch5_workspace_bytes.argtypes = C.c_size_t, [i, i]
    L.mm_batch5_create.restype = i
    L.mm_batch5_create.argtypes = [C.POINTER(vp), i, i, d, d, _dp, _dp, d, d, d, i, i, i, vp, vp, C.c_size_t]
    L.mm_batch5_set_state_prim.restype, L.mm_batch5_set_state_prim.argtypes = i, [vp, vp, i, i]
    L.mm_batch5_step.restype, L.mm_batch5_step.argtypes = i, [vp, i, d]
    L.mm_batch5_step_fixed_dt.restype, L.mm_batch5_step_fixed_dt.argtypes = i, [vp, i, d]
    L.mm_batch5_advance_to.restype, L.mm_batch5_advance_to.argtypes = i, [vp, d, d, C.c_longlong]
    L.mm_batch5_get_state.restype, L.mm_batch5_get_state.argtypes = i, [vp, vp, i]
    L.mm_batch5_get_info.restype = i
    L.mm_batch5_get_info.argtypes = [vp, _dp, C.POINTER(C.c_longlong), C.POINTER(C.c_int)]
    L.mm_batch5_launch_count.restype, L.mm_batch5_launch_count.argtypes = C.c_longlong, [vp]
    L.mm_batch5_destroy.restype, L.mm_batch5_destroy.argtypes = None, [vp]
    L.mm_strerror.restype, L.mm_strerror.argtypes = C.c_char_p, [i]
    L.mm_static5_run.restype = i
    L.mm_static5_run.argtypes = [i, d, d, C.POINTER(mm_collision), C.POINTER(mm_bc), C.POINTER(mm_options),
                                 vp, i, d, d, vp, i, _dp]
    _lib = L
    return L


_bench_lib = None


def bench_lib() -> C.CDLL:
    """Load libmm_bench.so (include/mm_bench.h): the measurement hooks, kept out of the product library."""
    global _bench_lib
    if _bench_lib is None:
        B = C.CDLL(str(build_ext.build_bench()))
        vp, i = C.c_void_p, C.c_int
        B.mm_measure_fp64_peak.restype, B.mm_measure_fp64_peak.argtypes = i, [vp, i, _dp, _dp]
        B.mm_selftest_fastmath.restype, B.mm_selftest_fastmath.argtypes = i, [vp, i, _dp]
        B.mm_measure_fp64_operand_rates.restype, B.mm_measure_fp64_operand_rates.argtypes = i, [vp, i, _dp]
        _bench_lib = B
    return _bench_lib


def _check(rc: int):
    if rc != OK:
        raise MMError(rc, lib().mm_strerror(rc).decode())


def _darr(x, n=None):
    a = np.ascontiguousarray(x, dtype=np.float64)
    if n is not None and a.size != n:
        raise ValueError(f"expected {n} doubles, got {a.size}")
    return a


def mm_workspace_bytes(system: int, nx: int, ny: int = 1, extent=(0.0, 1.0, 0.0, 1.0)) -> int:
    g = mm_grid(system, nx, ny, *extent)
    return lib().mm_workspace_bytes(C.byref(g))


def mm_measure_fp64_peak(repeats: int = 5, stream=None, with_clock: bool = False):
    """Measured FP64 FMA peak of the current device in TFLOP/s (2 flop per FMA); with_clock: also the SM
    clock (MHz) the probe ran at, from the kernel's own cycle counter and global timer."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    tf, mhz = C.c_double(), C.c_double()
    _check(bench_lib().mm_measure_fp64_peak(C.c_void_p(st.cuda_stream), repeats, C.byref(tf), C.byref(mhz)))
    return (tf.value, mhz.value) if with_clock else tf.value


def mm_measure_fp64_operand_rates(repeats: int = 3, stream=None):
    """10^12 thread instructions / s of the FP64 pipe with operands the reuse cache cannot supply:
    (DFMA with three distinct registers, DMUL, DADD); include/mm_bench.h."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    out = (C.c_double * 3)()
    _check(bench_lib().mm_measure_fp64_operand_rates(C.c_void_p(st.cuda_stream), repeats, out))
    return tuple(out)


def mm_decomposition(nx: int, ny: int, zsym: bool = True, sms: int = 148):
    """-> (nstrips, nchunks, warps_per_sm) of the 14-moment step kernel's launch (host logic only)."""
    a, b, c = C.c_int(), C.c_int(), C.c_int()
    _check(lib().mm_decomposition(nx, ny, int(zsym), sms, C.byref(a), C.byref(b), C.byref(c)))
    return a.value, b.value, c.value


def mm_selftest_fastmath(n: int = 1 << 22, stream=None):
    """Max relative error (units of 2^-53) of the library's rcp, sqrt and tabulated a(P*), b(P*)
    (include/mm.h)."""
    import torch
    st = stream if stream is not None else torch.cuda.current_stream()
    out = (C.c_double * 3)()
    _check(bench_lib().mm_selftest_fastmath(C.c_void_p(st.cuda_stream), n, out))
    return tuple(out)


def static5_run(W0, n: int, cfl: float = 0.0, dt: float = 0.0, extent=(0.0, 1.0), collision: Optional[dict] = None,
                sigma_lim: float = 1e-4, ws_scale: float = 1.0, limiter: int = LIM_MINMOD, shared_limiter: int = 0,
                flux: int = FLUX_HLL, source_scheme: int = SRC_EXPLICIT, time_scheme: int = TIME_EULER,
                periodic: bool = False, out=None, stream=None):
    """mm_static5_run (include/mm.h): n steps of a 1-D 5-moment tube of nx <= STATIC5_MAX_NX cells with no
    workspace from the caller -- the scratch is a 4 MiB array built into libmm.so, shared by every call on
    the device.  For callers that hold only their input and output arrays and cannot get device memory of
    their own (see the header for who they are).  W0: primitives [5][nx], numpy array (host path) or CUDA
    float64 tensor (device path); returns (U, t) with U of the same kind, conserved moments [5][nx].
    dt > 0: fixed time step; otherwise CFL steps at Courant number cfl.  Ends are transmissive, or
    periodic.  This wrapper allocates only `out` when none is given; pass `out` to allocate nothing."""
    import torch
    if not torch.cuda.is_available():
        raise MMError(ECUDA, "no CUDA device: the moment-method library has no CPU path")
    on_device = isinstance(W0, torch.Tensor) and W0.is_cuda
    if on_device:
        if W0.dtype != torch.float64 or not W0.is_contiguous() or W0.numel() % 5:
            raise ValueError("W0 must be a contiguous float64 tensor [5, nx]")
        nx = W0.numel() // 5
        if out is None:
            out = torch.empty((5, nx), dtype=torch.float64, device=W0.device)
        elif not (isinstance(out, torch.Tensor) and out.is_cuda and out.dtype == torch.float64
                  and out.is_contiguous() and out.numel() == 5 * nx):
            raise ValueError("out must be a contiguous CUDA float64 tensor [5, nx]")
        src, dst = C.c_void_p(W0.data_ptr()), C.c_void_p(out.data_ptr())
    else:
        W0 = _darr(W0)
        if W0.size % 5:
            raise ValueError("W0 must be [5, nx]")
        nx = W0.size // 5
        if out is None:
            out = np.empty((5, nx))
        elif out.dtype != np.float64 or not out.flags.c_contiguous or out.size != 5 * nx:
            raise ValueError("out must be a contiguous float64 array [5, nx]")
        src, dst = C.c_void_p(W0.ctypes.data), C.c_void_p(out.ctypes.data)
    col = collision or {"model": TAU_NONE}
    c = mm_collision(col.get("model", TAU_NONE), col.get("tau", 0.0), col.get("Kn", 0.0),
                     col.get("L_ref", 1.0), col.get("rho_ref", 1.0))
    sides = (mm_bc * 2)()
    sides[0].type = sides[1].type = BC_PERIODIC if periodic else BC_TRANSMISSIVE
    st = stream if stream is not None else torch.cuda.current_stream()
    o = mm_options(sigma_lim, ws_scale, limiter, shared_limiter, flux, source_scheme, time_scheme,
                   C.c_void_p(st.cuda_stream))
    t = C.c_double()
    _check(lib().mm_static5_run(nx, extent[0], extent[1], C.byref(c), sides, C.byref(o), src, n, cfl, dt,
                                dst, int(on_device), C.byref(t)))
    return out, t.value


class Solver:
    """mm_create ... mm_destroy around a torch-owned workspace.

    `bcs`: 4 dicts (xlo, xhi, ylo, yhi): {"type": BC_*, "bands": [(lo, hi, W), ...], "default": W|None,
    "state": STATE_PRIMITIVE (W = nmom primitives) | STATE_MAXWELLIAN (W = (rho, u_x, u_y, u_z, T))}.
    `R_gas`: mm_gas.R_gas (T = P/(rho R_gas); only Maxwellian boundary states use it).
    `workspace`: optional CUDA uint8 tensor of >= mm_workspace_bytes + 255 bytes to use instead of a fresh one.
    State arrays are [nmom][ny][nx]; numpy arrays / CPU tensors go through the host path
    (on_device = 0), CUDA tensors through the device path (on_device = 1)."""

    def __init__(self, system: int, nx: int, ny: int = 1, extent=(0.0, 1.0, 0.0, 1.0),
                 collision: Optional[dict] = None, bcs: Optional[Sequence[dict]] = None,
                 sigma_lim: float = 1e-4, ws_scale: float = 1.0, limiter: int = LIM_MINMOD,
                 shared_limiter: int = 0, flux: int = FLUX_HLL, source_scheme: int = SRC_EXPLICIT,
                 time_scheme: int = TIME_EULER, R_gas: float = 1.0, device: str = "cuda:0", stream=None,
                 workspace=None):
        import torch
        if not torch.cuda.is_available():
            raise MMError(ECUDA, "no CUDA device: the moment-method library has no CPU path")
        L = lib()
        self._L, self._torch = L, torch
        self.nm, self.nx, self.ny = system, nx, ny
        self.device = torch.device(device)
        g = mm_grid(system, nx, ny, *extent)
        nbytes = L.mm_workspace_bytes(C.byref(g))
        if nbytes == 0:
            raise MMError(EINVAL, "invalid grid")
        col = collision or {"model": TAU_NONE}
        c = mm_collision(col.get("model", TAU_NONE), col.get("tau", 0.0), col.get("Kn", 0.0),
                         col.get("L_ref", 1.0), col.get("rho_ref", 1.0))
        bcs = list(bcs) if bcs else [{"type": BC_TRANSMISSIVE}] * 4
        keep, arr = [], (mm_bc * 4)()
        for k in range(4):
            b = bcs[k] if k < len(bcs) else {"type": BC_TRANSMISSIVE}
            bands = b.get("bands", [])
            lo, hi = _darr([x[0] for x in bands]), _darr([x[1] for x in bands])
            bw = _darr([x[2] for x in bands]).reshape(-1)
            dflt = b.get("default")
            kind = b.get("state", STATE_PRIMITIVE)
            nw = 5 if kind == STATE_MAXWELLIAN else system
            if bw.size != nw * len(bands):
                raise ValueError(f"boundary side {k}: band states must have {nw} entries each")
            dw = _darr(dflt, nw) if dflt is not None else None
            keep += [lo, hi, bw, dw]
            arr[k] = mm_bc(b["type"], len(bands), lo.ctypes.data_as(_dp), hi.ctypes.data_as(_dp),
                           bw.ctypes.data_as(_dp), dw.ctypes.data_as(_dp) if dw is not None else None, kind)
        with torch.cuda.device(self.device):
            self._stream = stream if stream is not None else torch.cuda.current_stream()
            if workspace is None:
                workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            elif workspace.dtype != torch.uint8 or not workspace.is_cuda or workspace.numel() < nbytes + 255:
                raise MMError(EWORKSPACE, f"workspace must be a CUDA uint8 tensor of at least {nbytes + 255} bytes")
            self.workspace = workspace          # caller-owned device memory (mm.h): the library allocates none
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) // 256 * 256
            o = mm_options(sigma_lim, ws_scale, limiter, shared_limiter, flux, source_scheme, time_scheme,
                           C.c_void_p(self._stream.cuda_stream))
            h = C.c_void_p()
            gas = mm_gas(R_gas)
            _check(L.mm_create(C.byref(h), C.byref(g), C.byref(gas), C.byref(c), arr, C.byref(o),
                               C.c_void_p(self._ws_ptr), nbytes))
        self._h = h
        self.workspace_bytes = nbytes

    @classmethod
    def from_problem(cls, prob: dict, load_state: bool = True, **kw) -> "Solver":
        s = cls(prob["system"], prob["nx"], prob["ny"], extent=prob["extent"],
                collision=prob["collision"], bcs=prob["bcs"], **prob["options"], **kw)
        if load_state:
            s.set_state_prim(prob["W0"])
        return s

    # -- state in / out -------------------------------------------------------------
    def _in(self, x):
        torch = self._torch
        n = self.nm * self.ny * self.nx
        if isinstance(x, torch.Tensor):
            if x.dtype != torch.float64 or not x.is_contiguous() or x.numel() != n:
                raise ValueError("state tensor must be contiguous float64 [nmom, ny, nx]")
            return x, C.c_void_p(x.data_ptr()), int(x.is_cuda)
        a = _darr(x, n)
        return a, C.c_void_p(a.ctypes.data), 0

    def set_state(self, U):
        keep, ptr, dev = self._in(U)
        _check(self._L.mm_set_state(self._h, ptr, dev))
        if not dev:
            self.synchronize()      # the host buffer may go away after this call

    def set_state_prim(self, W):
        keep, ptr, dev = self._in(W)
        _check(self._L.mm_set_state_prim(self._h, ptr, dev))
        if not dev:
            self.synchronize()

    def _out(self, out, fn):
        torch = self._torch
        if out is None:
            out = np.empty((self.nm, self.ny, self.nx))
        if isinstance(out, torch.Tensor):
            keep, ptr, dev = self._in(out)
        else:
            if out.dtype != np.float64 or not out.flags.c_contiguous or out.size != self.nm * self.ny * self.nx:
                raise ValueError("output array must be contiguous float64 [nmom, ny, nx]")
            ptr, dev = C.c_void_p(out.ctypes.data), 0
        _check(fn(self._h, ptr, dev))
        return out

    def get_state(self, out=None):
        return self._out(out, self._L.mm_get_state)

    def get_state_prim(self, out=None):
        return self._out(out, self._L.mm_get_state_prim)

    # -- stepping -------------------------------------------------------------------
    def step(self, n: int, cfl: float):
        _check(self._L.mm_step(self._h, n, cfl))

    def step_fixed_dt(self, n: int, dt: float):
        _check(self._L.mm_step_fixed_dt(self._h, n, dt))

    def advance_to(self, t_end: float, cfl: float, max_steps: int = 0):
        _check(self._L.mm_advance_to(self._h, t_end, cfl, max_steps))

    def cfl_dt(self, cfl: float) -> float:
        dt = C.c_double()
        _check(self._L.mm_cfl_dt(self._h, cfl, C.byref(dt)))
        return dt.value

    def info(self, check: bool = True) -> dict:
        t, n, dt, sp = C.c_double(), C.c_longlong(), C.c_double(), C.c_double()
        rc = self._L.mm_get_info(self._h, C.byref(t), C.byref(n), C.byref(dt), C.byref(sp))
        if check:
            _check(rc)
        return {"t": t.value, "steps": n.value, "last_dt": dt.value, "max_speed": sp.value,
                "status": rc}

    def dt_history(self, first_step: int, n: int) -> np.ndarray:
        """dt of the steps first_step .. first_step + n - 1 (kept on the device, last 65536 steps)."""
        out = np.empty(n, dtype=np.float64)
        _check(self._L.mm_get_dt_history(self._h, first_step, n, out.ctypes.data_as(_dp)))
        return out

    def set_clock(self, t: float, steps: int):
        """Restore t and the step counter after set_state (checkpoint / resume)."""
        _check(self._L.mm_set_clock(self._h, t, steps))

    def profile_begin(self):
        _check(self._L.mm_profile_begin(self._h))

    def profile_end(self):
        """-> (summed device time of the fused step kernel in ms, number of its launches)."""
        ms, n = C.c_double(), C.c_longlong()
        _check(self._L.mm_profile_end(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def set_fast_path(self, allow: bool):
        """Allow (default) or forbid the z-symmetric kernel variant (include/mm.h)."""
        _check(self._L.mm_set_fast_path(self._h, 1 if allow else 0))

    @property
    def fast_path_active(self) -> bool:
        return bool(self._L.mm_fast_path_active(self._h))

    @property
    def launches(self) -> int:
        return self._L.mm_launch_count(self._h)

    @property
    def stream(self):
        return self._stream

    def synchronize(self):
        self._stream.synchronize()

    def close(self):
        if getattr(self, "_h", None):
            self.synchronize()
            self._L.mm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Batch5:
    """mm_batch5_*: `ntubes` independent 1-D 5-moment tubes with per-tube sigma_lim and Kn
    (include/mm.h).  Kn <= 0 or None marks a collisionless tube."""

    def __init__(self, nx, sigma_lim, Kn, extent=(0.0, 1.0), L_ref=1.0, rho_ref=1.0, ws_scale=1.0,
                 limiter=LIM_MINMOD, shared_limiter=0, flux=FLUX_HLL, device="cuda:0", stream=None):
        import torch
        L = lib()
        self._L, self._h = L, None
        sig = _darr(sigma_lim)
        kn = _darr([k if k is not None else 0.0 for k in Kn])
        if sig.size != kn.size:
            raise ValueError("sigma_lim and Kn must have one entry per tube")
        self.nx, self.ntubes = nx, sig.size
        nbytes = L.mm_batch5_workspace_bytes(nx, self.ntubes)
        if nbytes == 0:
            raise MMError(EINVAL, "invalid batch")
        if not torch.cuda.is_available():
            raise MMError(ECUDA, "no CUDA device: this library has no CPU path")
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self._stream = stream if stream is not None else torch.cuda.current_stream()
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            ptr = (self.workspace.data_ptr() + 255) // 256 * 256
            h = C.c_void_p()
            _check(L.mm_batch5_create(C.byref(h), nx, self.ntubes, extent[0], extent[1],
                                      sig.ctypes.data_as(_dp), kn.ctypes.data_as(_dp), L_ref, rho_ref, ws_scale,
                                      limiter, shared_limiter, flux, C.c_void_p(self._stream.cuda_stream),
                                      C.c_void_p(ptr), nbytes))
            self._h = h

    def set_state_prim(self, W):
        """W: numpy [5][nx] (copied to every tube) or [ntubes][5][nx]."""
        a = np.ascontiguousarray(W, dtype=np.float64)
        per_tube = a.ndim == 3
        if a.size != (self.ntubes if per_tube else 1) * 5 * self.nx:
            raise ValueError("bad state shape")
        _check(self._L.mm_batch5_set_state_prim(self._h, a.ctypes.data_as(C.c_void_p), int(per_tube), 0))
        self._stream.synchronize()      # the host buffer may go away after this call (as Solver.set_state*)

    def step(self, n, cfl):
        _check(self._L.mm_batch5_step(self._h, n, cfl))

    def step_fixed_dt(self, n, dt):
        _check(self._L.mm_batch5_step_fixed_dt(self._h, n, dt))

    def advance_to(self, t_end, cfl, max_steps=0):
        _check(self._L.mm_batch5_advance_to(self._h, t_end, cfl, max_steps))

    def get_state(self):
        out = np.empty((self.ntubes, 5, self.nx), dtype=np.float64)
        _check(self._L.mm_batch5_get_state(self._h, out.ctypes.data_as(C.c_void_p), 0))
        return out

    def info(self, check=True):
        t = np.empty(self.ntubes); n = np.empty(self.ntubes, dtype=np.int64); f = np.empty(self.ntubes, dtype=np.int32)
        rc = self._L.mm_batch5_get_info(self._h, t.ctypes.data_as(_dp), n.ctypes.data_as(C.POINTER(C.c_longlong)),
                                        f.ctypes.data_as(C.POINTER(C.c_int)))
        if check:
            _check(rc)
        return {"t": t, "steps": n, "failed": f, "status": rc}

    @property
    def launches(self):
        return self._L.mm_batch5_launch_count(self._h)

    def sync(self):
        import torch
        torch.cuda.synchronize(self.device)

    def __del__(self):
        if getattr(self, "_h", None):
            self._L.mm_batch5_destroy(self._h)
            self._h = None

