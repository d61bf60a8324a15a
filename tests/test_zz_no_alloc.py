"""mm_static5_run: the one entry point of the library that needs no device workspace from its caller.

Who it is for.  Every other call of include/mm.h wants a `d_workspace` the caller allocated.  A routine that
is called back from inside another program's solver, or that is plugged into a framework which owns the
GPU's memory pool (and has usually reserved all of it), gets its input and output arrays and nothing more:
it may not, or cannot, obtain device memory itself -- a raw cudaMalloc there fails for lack of free memory,
stalls the whole device, or is simply against the host's rules; a C/Fortran driver linking libmm.so alone
has no CUDA runtime to call at all.  For such callers the 5-moment step's scratch (control block, tables,
both state copies) is a 4 MiB `static __device__` array inside the library, good for nx <= 8192 cells.

What is checked here, against the existing path (mm.Solver on a torch-allocated workspace: the same kernels
on caller-owned memory), at the bar the parity tests use (1e-10 per moment, tests/test_gpu_parity.py):
  * two calls in a row on different problems -- the second, smaller one runs on an array still holding the
    first one's control block, boundary table and states, so anything the entry point forgot to clear shows;
  * a repeat of the first call, and the device-pointer form of the interface;
  * sizes beyond the limit are refused with a message that names the limit (no GPU needed for that).
The file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should not hide
the parity tests.  It makes no assumption about what ran before it: it passes alone in a fresh process
(where its first call performs the per-device address lookup) and at the end of the whole suite.
"""
import numpy as np
import pytest

import mm_workloads as wl

TOL = 1e-10     # per moment, max-norm, relative: the bar of tests/test_gpu_parity.py


def rel_err(Ua, Ub):
    return max(np.abs(Ua[m] - Ub[m]).max() / np.abs(Ub[m]).max() for m in range(Ub.shape[0]))


def existing_path(mm, prob, n, dt=None, cfl=None):
    """The same run through mm_create on a caller-allocated workspace."""
    s = mm.Solver.from_problem(prob)
    if dt is not None:
        s.step_fixed_dt(n, dt)
    else:
        s.step(n, cfl)
    U, t = s.get_state().reshape(5, prob["nx"]), s.info()["t"]
    s.close()
    return U, t


def static_path(mm, prob, n, dt=0.0, cfl=0.0, W0=None, **kw):
    o = prob["options"]
    return mm.static5_run(prob["W0"].reshape(5, -1) if W0 is None else W0, n, cfl=cfl, dt=dt,
                          extent=prob["extent"][:2], collision=prob["collision"],
                          periodic=prob["bcs"][0]["type"] == wl.BC_PERIODIC, **o, **kw)


@pytest.fixture(scope="module")
def mm():
    from paper_2401_15233_b200 import mm as _mm
    _mm.lib()
    return _mm


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_workspace_path(mm):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    # call 1: the Sod tube of BASELINE configs[0] (1000 cells, Kn = 0.01), 100 fixed-dt steps
    sod = wl.sod5(1000, Kn=0.01)
    scout = mm.Solver.from_problem(sod)
    scout.step(100, 0.5)
    dt = 0.5 * float(scout.dt_history(0, 100).min())      # a fixed dt that is stable over these 100 steps
    scout.close()
    U1, t1 = static_path(mm, sod, 100, dt=dt)
    # call 2, straight after it, on the same array: a smaller periodic problem with other options,
    # CFL-stepped -- the time step comes from accumulators in the control block that call 1 left non-zero
    smooth = wl.random_smooth5(333, Kn=0.05, limiter=wl.LIM_VANALBADA, flux=wl.FLUX_RUSANOV)
    U2, t2 = static_path(mm, smooth, 60, cfl=0.5)
    R1, s1 = existing_path(mm, sod, 100, dt=dt)
    R2, s2 = existing_path(mm, smooth, 60, cfl=0.5)
    assert np.all(np.isfinite(U1)) and np.all(np.isfinite(U2))
    assert rel_err(U1, R1) <= TOL and t1 == pytest.approx(s1, rel=1e-13)
    assert rel_err(U2, R2) <= TOL and t2 == pytest.approx(s2, rel=1e-13)
    assert np.abs(U1 - wl_cons_of_start(mm, sod)).max() > 1e-3       # the run did move the state
    # call 3: the first problem again, now after the smaller one; device pointers in and out, result
    # written into a tensor the caller brought (the wrapper then allocates nothing either)
    Wd = torch.from_numpy(sod["W0"].reshape(5, -1)).cuda()
    out = torch.full((5, 1000), float("nan"), dtype=torch.float64, device="cuda")
    U3, t3 = static_path(mm, sod, 100, dt=dt, W0=Wd, out=out)
    assert U3 is out and rel_err(out.cpu().numpy(), R1) <= TOL and t3 == pytest.approx(s1, rel=1e-13)


def wl_cons_of_start(mm, prob):
    """Conserved moments of the initial state (zero steps through the entry point itself)."""
    return static_path(mm, prob, 0, dt=1.0)[0]


@pytest.mark.gpu
def test_largest_size_runs_and_the_next_one_is_refused(mm):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    nmax = mm.STATIC5_MAX_NX
    big = wl.sod5(nmax, Kn=0.01)
    U, t = static_path(mm, big, 20, cfl=0.5)
    R, s = existing_path(mm, big, 20, cfl=0.5)
    assert rel_err(U, R) <= TOL and t == pytest.approx(s, rel=1e-13)
    with pytest.raises(mm.MMError) as e:
        static_path(mm, wl.sod5(nmax + 1, Kn=0.01), 1, cfl=0.5)
    assert e.value.status == mm.ETOOLARGE and str(nmax) in str(e.value)


def test_oversize_is_refused_before_any_cuda_call(mm):
    """Runs without a GPU: the size check comes first, and its message states the limit."""
    import ctypes as C
    lib = mm.lib()
    nx = mm.STATIC5_MAX_NX + 1
    c = mm.mm_collision(0, 0, 0, 1, 1)
    o = mm.mm_options(1e-4, 1.0, 1, 0, 0, 0, 0, None)
    W = np.ones((5, nx)); U = np.empty((5, nx))
    args = (C.byref(c), None, C.byref(o), C.c_void_p(W.ctypes.data), 1, 0.5, 0.0, C.c_void_p(U.ctypes.data), 0, None)
    assert lib.mm_static5_run(nx, 0.0, 1.0, *args) == mm.ETOOLARGE
    assert str(mm.STATIC5_MAX_NX).encode() in lib.mm_strerror(mm.ETOOLARGE)
    assert lib.mm_static5_run(0, 0.0, 1.0, *args) == mm.EINVAL
    assert mm.mm_workspace_bytes(5, mm.STATIC5_MAX_NX, 1) <= 4 << 20      # what the built-in array must hold
    # and the scratch really is a static device array in the library image, not something allocated at run time
    from paper_2401_15233_b200 import build_ext
    src = (build_ext.CSRC / "mm_api.cu").read_text()
    assert "static __device__ __align__(256) unsigned char g_static5_scratch[MM_STATIC5_SCRATCH_BYTES]" in src
    assert "cudaGetSymbolAddress(&p, g_static5_scratch)" in src
