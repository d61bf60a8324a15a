"""GPU parity: the CUDA path (through the C-ABI binding) against the CPU oracle, element by
element, on the same seeded inputs (mm_workloads.py).

Bar (BASELINE.json north_star): per moment k,
    max_cells |U_gpu - U_oracle| / max_cells |U_oracle| <= 1e-10  after 100 steps at fixed dt,
and a moment that is identically zero in the oracle is identically zero on the GPU.
"""
import numpy as np
import pytest

import mm_workloads as wl
from parity_util import window_errors

pytestmark = pytest.mark.gpu

TOL = 1e-10


@pytest.fixture(scope="module")
def mm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2401_15233_b200 import mm as _mm
    _mm.lib()
    return _mm


def oracle_solver(mmo, prob, **kw):
    s = mmo.Solver(prob["system"], prob["nx"], prob["ny"], extent=prob["extent"],
                   collision=prob["collision"], bcs=prob["bcs"], nthreads=0, **prob["options"], **kw)
    s.set_state_prim(prob["W0"])
    return s


def rel_err(Ug, Uo):
    """per-moment max-norm relative error; checks exact zeros."""
    errs = []
    for m in range(Uo.shape[0]):
        scale = np.abs(Uo[m]).max()
        if scale == 0.0:
            assert np.all(Ug[m] == 0.0), f"moment {m}: oracle identically 0, GPU not"
            errs.append(0.0)
        else:
            errs.append(np.abs(Ug[m] - Uo[m]).max() / scale)
    return np.array(errs)


def assert_parity(Ug, Uo, tol=TOL):
    assert np.all(np.isfinite(Uo)), "oracle state is not finite: test case is ill-posed"
    assert np.all(np.isfinite(Ug))
    e = rel_err(Ug, Uo)
    assert e.max() <= tol, f"per-moment rel. error {e}"
    return e


def scout_dt(mmo, prob, nsteps, cfl, U0=None):
    """Smallest CFL time step the ORACLE takes over `nsteps` steps from the starting state.
    Wave speeds grow quickly once a Maxwellian start develops non-equilibrium (sigma -> sigma_lim),
    so the dt of the starting state alone is not a stable fixed dt."""
    so = oracle_solver(mmo, prob)
    if U0 is not None:
        so.set_state(U0)
    dts = []
    for _ in range(nsteps):
        so.step(1, cfl)
        dts.append(so.info()["last_dt"])
    return min(dts)


def roundoff_sensitivity(mmo, prob, nsteps, dt, seed=1):
    """What round-off alone does to the ORACLE on this problem: two oracle runs at the same fixed
    dt, one of which has every moment multiplied by (1 + k 1e-15), k in {-2..2}, after every step
    (the size of the difference between two correct fp64 evaluations of one step).  With one
    limiter value shared by all primitives psi = 2 min(|dm|,|dp|)/(|dm|+|dp|) of
    the variable nearest to an extremum sets every slope of the cell, and an error e in that
    variable changes psi by ~ e/|dp|: measured growth is ~20x per step while an extremum of any
    of the 14 variables crosses a cell (R24)."""
    a, b = oracle_solver(mmo, prob), oracle_solver(mmo, prob)
    rng = np.random.default_rng(seed)
    for _ in range(nsteps):
        a.step_fixed_dt(1, dt); b.step_fixed_dt(1, dt)
        Ub = b.get_state()
        b.set_state(Ub * (1.0 + 1e-15 * rng.integers(-2, 3, size=Ub.shape)))
    Ua, Ub = a.get_state(), b.get_state()
    scale = np.abs(Ua).max(axis=(1, 2))
    return float((np.abs(Ua - Ub).max(axis=(1, 2)) / np.where(scale > 0, scale, 1.0)).max())


def run_both(mm, mmo, prob, nsteps, dt=None, cfl=0.4, dt_frac=0.5, fast=None):
    """fast: None = whatever the library selects; True / False = require / forbid the
    z-symmetric kernel variant (include/mm.h, mm_set_fast_path)."""
    so = oracle_solver(mmo, prob)
    sg = mm.Solver.from_problem(prob)
    if fast is not None and prob["system"] == 14:
        sg.set_fast_path(fast)
        assert sg.fast_path_active == fast
    if dt is None:
        dt = dt_frac * scout_dt(mmo, prob, nsteps, cfl)
    so.step_fixed_dt(nsteps, dt)
    sg.step_fixed_dt(nsteps, dt)
    Ug, Uo = sg.get_state(), so.get_state()
    info = sg.info()
    assert info["steps"] == nsteps
    assert info["t"] == pytest.approx(so.info()["t"], rel=1e-13)
    return Ug, Uo


# ----------------------------------------------------------- state in / out, set-up values
def test_state_roundtrip_and_prim_conversion(mm, mmo):
    prob = wl.random_smooth14(70, 37)
    sg = mm.Solver.from_problem(prob)
    so = oracle_solver(mmo, prob)
    Uo = so.get_state()
    assert_parity(sg.get_state(), Uo, 1e-14)                    # prim -> cons on the GPU
    assert_parity(sg.get_state_prim(), prob["W0"], 1e-13)      # and back
    sg.set_state(Uo)
    assert np.array_equal(sg.get_state(), Uo)                   # conserved in/out is a copy
    import torch
    Ud = torch.from_numpy(Uo).cuda()
    sg.set_state(Ud)
    out = torch.empty_like(Ud)
    sg.get_state(out)
    assert torch.equal(out, Ud)
    assert sg.cfl_dt(0.4) == pytest.approx(so.cfl_dt(0.4), rel=1e-13)
    assert sg.info()["max_speed"] > 0

    p5 = wl.random_smooth5(333)
    s5 = mm.Solver.from_problem(p5); o5 = oracle_solver(mmo, p5)
    assert_parity(s5.get_state(), o5.get_state(), 1e-14)
    assert s5.cfl_dt(0.5) == pytest.approx(o5.cfl_dt(0.5), rel=1e-13)


def test_cfl_dt_includes_dirichlet_ghosts(mm, mmo):
    prob = wl.crossed_jets(64, Kn=1.0)
    sg = mm.Solver.from_problem(prob); so = oracle_solver(mmo, prob)
    # the jets' ghost states are the fastest cells of the initial state (R13)
    # at sigma_bar = sigma_lim the wave-speed formula amplifies round-off in q* by ~1/(2 sigma_lim)
    assert sg.cfl_dt(0.4) == pytest.approx(so.cfl_dt(0.4), rel=1e-10)
    bg = dict(prob, bcs=[dict(type=wl.BC_TRANSMISSIVE)] * 4)
    assert mm.Solver.from_problem(bg).cfl_dt(0.4) > 2.0 * sg.cfl_dt(0.4)


# ----------------------------------------------------------------- small, all the variants
@pytest.mark.parametrize("limiter,shared,flux", [
    (wl.LIM_MINMOD, 0, wl.FLUX_HLL), (wl.LIM_MINMOD, 1, wl.FLUX_RUSANOV),
    (wl.LIM_VANALBADA, 0, wl.FLUX_RUSANOV), (wl.LIM_VANALBADA, 1, wl.FLUX_HLL),
    (wl.LIM_NONE, 0, wl.FLUX_HLL)])
@pytest.mark.parametrize("Kn", [None, 0.05])
def test_smooth14_periodic_variants(mm, mmo, limiter, shared, flux, Kn):
    # 70 x 37: three 30-cell strips with a ragged tail; all 14 primitives vary (general variant)
    prob = wl.random_smooth14(70, 37, Kn=Kn, limiter=limiter, shared_limiter=shared, flux=flux)
    dt = 0.5 * scout_dt(mmo, prob, 30, 0.4)
    Ug, Uo = run_both(mm, mmo, prob, 5, dt=dt)
    assert_parity(Ug, Uo)
    Ug, Uo = run_both(mm, mmo, prob, 30, dt=dt)
    # shared psi amplifies round-off (see roundoff_sensitivity): condition-aware bar after 30 steps
    tol = max(TOL, 10.0 * roundoff_sensitivity(mmo, prob, 30, dt)) if shared else TOL
    assert_parity(Ug, Uo, tol)


@pytest.mark.parametrize("limiter,shared,flux", [
    (wl.LIM_MINMOD, 0, wl.FLUX_HLL), (wl.LIM_MINMOD, 1, wl.FLUX_HLL), (wl.LIM_MINMOD, 1, wl.FLUX_RUSANOV),
    (wl.LIM_VANALBADA, 1, wl.FLUX_HLL), (wl.LIM_VANALBADA, 0, wl.FLUX_RUSANOV), (wl.LIM_NONE, 0, wl.FLUX_HLL)])
@pytest.mark.parametrize("fast", [True, False])
def test_smooth14_zsym_both_kernel_variants(mm, mmo, limiter, shared, flux, fast):
    """z-symmetric state (u_z = P_xz = P_yz = q_z = 0): the fast variant and the general variant
    both match the (general) oracle; 70 x 37 spans three 30-cell strips with a ragged tail."""
    prob = wl.random_smooth14(70, 37, Kn=0.05, zsym=True, limiter=limiter, shared_limiter=shared, flux=flux)
    dt = 0.5 * scout_dt(mmo, prob, 30, 0.4)
    Ug, Uo = run_both(mm, mmo, prob, 30, dt=dt, fast=fast)
    tol = max(TOL, 10.0 * roundoff_sensitivity(mmo, prob, 30, dt)) if shared else TOL
    assert_parity(Ug, Uo, tol)
    for m in (3, 6, 8, 12):
        assert np.all(Ug[m] == 0.0)


def test_fast_path_selection(mm):
    """The fast variant is selected only when state AND Dirichlet data have no z-odd moment."""
    gen = wl.random_smooth14(40, 12)
    zs = wl.random_smooth14(40, 12, zsym=True)
    s = mm.Solver.from_problem(gen)
    assert not s.fast_path_active
    s.set_state_prim(zs["W0"])
    assert s.fast_path_active
    W = zs["W0"].copy(); W[12, 5, 7] = 1e-300
    s.set_state_prim(W)
    assert not s.fast_path_active
    s.set_state_prim(zs["W0"]); s.set_fast_path(False)
    assert not s.fast_path_active
    jets = wl.crossed_jets(32, Kn=1.0)
    assert mm.Solver.from_problem(jets).fast_path_active
    bad = [dict(b) for b in jets["bcs"]]
    Wd = np.array(bad[0]["default"], dtype=float).copy(); Wd[3] = 0.1
    bad[0]["default"] = Wd
    assert not mm.Solver.from_problem(dict(jets, bcs=bad)).fast_path_active
    assert not mm.Solver.from_problem(wl.sod5(64, Kn=0.01)).fast_path_active


def test_fastmath_accuracy(mm):
    """The branch-free reciprocal and square root of the CUDA path against IEEE division / sqrt,
    and the tabulated wave-speed functions a(P*), b(P*) (Eq 29c-d) against the direct formulas with
    libm pow / exp, over 4 M arguments; in units of 2^-53 relative.  The direct formula itself
    is only good to ~P*^2 units (rounding of P*^2 in the exponent), hence the wider last bound."""
    e_rcp, e_sqrt, e_ab = mm.mm_selftest_fastmath(1 << 22)
    assert 0.0 < e_rcp <= 2.0 and 0.0 < e_sqrt <= 2.5, (e_rcp, e_sqrt)
    assert 0.0 < e_ab <= 40.0, e_ab


def test_smooth14_transmissive(mm, mmo):
    prob = wl.random_smooth14(45, 19, Kn=0.2, periodic=False)
    Ug, Uo = run_both(mm, mmo, prob, 40)
    assert_parity(Ug, Uo)


@pytest.mark.parametrize("nx,ny", [(1, 1), (3, 2), (5, 1), (33, 9), (30, 7), (31, 5), (60, 3), (61, 40)])
def test_tiny_grids(mm, mmo, nx, ny):
    """Degenerate and edge sizes: single cells, nx below / at / just above one and two 30-cell strips."""
    prob = wl.random_smooth14(nx, ny, Kn=0.3)
    Ug, Uo = run_both(mm, mmo, prob, 10)
    assert_parity(Ug, Uo)


@pytest.mark.parametrize("zsym", [False, True])
def test_anisotropic_cells_and_mixed_boundaries(mm, mmo, zsym):
    """dx != dy (dt/dx and dt/dy differ) with periodic x and transmissive y."""
    prob = wl.random_smooth14(50, 23, Kn=0.1, zsym=zsym, shared_limiter=1)
    prob = dict(prob, extent=(0.0, 1.0, 0.0, 0.37),
                bcs=[dict(type=wl.BC_PERIODIC), dict(type=wl.BC_PERIODIC),
                     dict(type=wl.BC_TRANSMISSIVE), dict(type=wl.BC_TRANSMISSIVE)])
    dt = 0.5 * scout_dt(mmo, prob, 20, 0.4)
    Ug, Uo = run_both(mm, mmo, prob, 20, dt=dt)
    assert_parity(Ug, Uo, max(TOL, 10.0 * roundoff_sensitivity(mmo, prob, 20, dt)))


@pytest.mark.parametrize("limiter,flux", [(wl.LIM_MINMOD, wl.FLUX_HLL), (wl.LIM_VANALBADA, wl.FLUX_RUSANOV)])
def test_smooth5_periodic(mm, mmo, limiter, flux):
    prob = wl.random_smooth5(333, Kn=0.05, limiter=limiter, flux=flux)
    Ug, Uo = run_both(mm, mmo, prob, 100, cfl=0.5)
    assert_parity(Ug, Uo)


# ------------------------------------------------------------------- BASELINE configs
def test_C1_sod5_100_steps_fixed_dt(mm, mmo):
    prob = wl.sod5(1000, Kn=0.01)
    Ug, Uo = run_both(mm, mmo, prob, 100, cfl=0.5)
    assert_parity(Ug, Uo)


def test_C1_sod5_cfl_steps(mm, mmo):
    """CFL stepping (each side reduces its own dt).  Config 1 is sensitive to round-off: the
    oracle run from an initial state perturbed by 1e-15 differs from the unperturbed one by
    1e-7 after 154 steps and by percents after 200 (tests/test_oracle_scheme.py::
    test_C1_roundoff_sensitivity, R24), so element-wise parity is checked over the
    first 100 CFL steps and the whole run to t = 0.2 is compared through what is robust:
    the end time, the step count and the density profile."""
    prob = wl.sod5(1000, Kn=0.01)
    so = oracle_solver(mmo, prob); sg = mm.Solver.from_problem(prob)
    so.step(100, 0.5); sg.step(100, 0.5)
    assert sg.info()["t"] == pytest.approx(so.info()["t"], rel=1e-9)
    assert_parity(sg.get_state(), so.get_state(), 1e-8)
    so.advance_to(0.2, 0.5); sg.advance_to(0.2, 0.5)
    ig, io = sg.info(), so.info()
    assert ig["t"] == 0.2 and io["t"] == 0.2
    assert abs(ig["steps"] - io["steps"]) <= 0.03 * io["steps"]
    Ug, Uo = sg.get_state(), so.get_state()
    assert np.all(np.isfinite(Ug)) and Ug[0].min() > 0
    assert np.abs(Ug[0] - Uo[0]).mean() <= 2e-3 * np.abs(Uo[0]).mean()


@pytest.mark.parametrize("Kn", [1e-3, 1e-2, 1e-1, 1.0])
def test_C2_sod14_4096x4(mm, mmo, Kn):
    prob = wl.sod14(4096, 4, Kn=Kn)
    Ug, Uo = run_both(mm, mmo, prob, 100, cfl=0.5, fast=True)
    assert_parity(Ug, Uo)
    for j in range(1, 4):
        assert np.array_equal(Ug[:, j], Ug[:, 0])


@pytest.mark.parametrize("fast", [True, False])
def test_C3_jets_512_from_t0(mm, mmo, fast):
    prob = wl.crossed_jets(512, Kn=1.0)
    Ug, Uo = run_both(mm, mmo, prob, 100, cfl=0.4, fast=fast)
    assert_parity(Ug, Uo)


def test_C3_jets_developed_state(mm, mmo):
    """Developed state (jets have crossed): produced by the ORACLE with CFL stepping on a
    128^2 grid, then used as the common input of both sides.  Wave speeds inflated by k = 1.2
    (PAPER.md L409, L416): with k = 1 the HLL run loses positivity at t = 0.1375 on this grid, in
    the oracle itself (R14).
    On this state the scheme amplifies round-off strongly (cells at the jet edges next to the
    inflow wall sit at sigma_bar = sigma_lim, closure terms ~ 1/sigma_bar^2): two ORACLE runs whose
    inputs differ by 1e-15 relative differ by ~1e-11 after ONE step and by ~1e-3 after 100
    (R24).  So the bar is condition-aware: the GPU may differ from the oracle by no more
    than 10x what a 1e-15 perturbation of the input does to the oracle itself (and never needs to
    beat 1e-10); over 100 steps the density field and the conserved totals are compared too."""
    prob = wl.crossed_jets(128, Kn=1.0, ws_scale=1.2)
    so = oracle_solver(mmo, prob)
    so.advance_to(0.15, 0.4)
    U0 = so.get_state()
    rng = np.random.default_rng(1)
    U1 = U0 * (1.0 + 1e-15 * rng.integers(-2, 3, size=U0.shape))
    dt = 0.5 * scout_dt(mmo, prob, 100, 0.4, U0)
    sg = mm.Solver.from_problem(prob, load_state=False)
    sp = oracle_solver(mmo, prob)                      # the perturbed oracle run
    sg.set_state(U0); so.set_state(U0); sp.set_state(U1)
    done = 0
    for nsteps in (5, 100):
        so.step_fixed_dt(nsteps - done, dt); sp.step_fixed_dt(nsteps - done, dt)
        sg.step_fixed_dt(nsteps - done, dt)
        done = nsteps
        Ug, Uo, Up = sg.get_state(), so.get_state(), sp.get_state()
        sens = rel_err(Up, Uo).max()
        assert_parity(Ug, Uo, max(TOL, 10.0 * sens))
        rho_noise = np.abs(Up[0] - Uo[0]).mean()
        assert np.abs(Ug[0] - Uo[0]).mean() <= 10.0 * rho_noise + 1e-13 * np.abs(Uo[0]).mean()
    # CFL stepping from the same state: same number of steps to (nearly) the same time
    so.set_state(U0); sg.set_state(U0)
    so.step(5, 0.4); sg.step(5, 0.4)
    assert sg.info()["t"] == pytest.approx(so.info()["t"], rel=1e-9)
    sp.set_state(U1); sp.step(5, 0.4)
    assert_parity(sg.get_state(), so.get_state(), max(1e-9, 10.0 * rel_err(sp.get_state(), so.get_state()).max()))


@pytest.mark.parametrize("n,Kn,fast", [(2048, 0.1, True), (2048, 1.0, True), (4096, 0.1, True), (2048, 0.1, False)])
def test_C4_C5_jets_full_size_sampled_windows(mm, mmo, n, Kn, fast):
    """Full bench sizes (BASELINE configs[3] and [4]), bench launch configuration: after n steps a
    cell depends only on the (2n)-neighbourhood of its initial data, so the oracle is run on small
    windows of the same seeded state (transmissive window edges) and compared on the cells no edge
    can have reached."""
    nsteps, half, margin = 3, 14, 2 * 3 + 1
    prob = wl.crossed_jets(n, Kn=Kn, perturb=0.01)
    sg = mm.Solver.from_problem(prob)
    sg.set_fast_path(fast)                     # z-symmetric variant (what bench.py runs) or the general one
    assert sg.fast_path_active == fast
    so_dt = 0.5 * 0.4 * (1.0 / n) / 6.0        # CFL 0.2 against the jets' inflow speed (~5.8)
    sg.step_fixed_dt(nsteps, so_dt)
    Ug = sg.get_state()
    W0 = prob["W0"]
    rng = np.random.default_rng(7)
    centres = [(int(a), int(b)) for a, b in rng.integers(half, n - half, size=(6, 2))]
    centres += [(half, int(0.35 * n)), (half, int(0.65 * n)), (half, int(0.5 * n))]   # at the inflow side
    # across strip boundaries (every 30 cells) and row-chunk boundaries of the launch decomposition
    centres += [(30 * 20, n * 5 // 17), (30 * 41, n * 9 // 17 + 1), (30 * (n // 30) - 6, n // 2), (n - half, n - half)]
    h = 1.0 / n
    for (ci, cj) in centres:
        i0, j0 = ci - half, cj - half
        w = 2 * half
        sub = dict(prob, nx=w, ny=w, W0=np.ascontiguousarray(W0[:, j0:j0 + w, i0:i0 + w]),
                   extent=(i0 * h, (i0 + w) * h, j0 * h, (j0 + w) * h))
        if i0 > 0:
            sub["bcs"] = [dict(type=wl.BC_TRANSMISSIVE)] * 4
        so = oracle_solver(mmo, sub)
        so.step_fixed_dt(nsteps, so_dt)
        Uo = so.get_state()
        lo_i = 0 if i0 == 0 else margin
        sl = (slice(None), slice(margin, w - margin), slice(lo_i, w - margin))
        ref = Uo[sl]
        got = Ug[:, j0:j0 + w, i0:i0 + w][sl]
        e = window_errors(got, ref)            # each window scaled by its OWN data (tests/parity_util.py)
        assert e.max() <= TOL, (ci, cj, e)


def test_single_jet_fast_wave_runs_ahead_of_the_density_front(mm):
    """PAPER.md L440 (Fig 11): the density front of the collisionless M = 5 jet travels roughly at the
    jet velocity, waves in the fourth-order moment R* travel "roughly twice as fast", and the gas
    they have not reached is still at equilibrium with R* = 15 and q* = 0."""
    n = 300
    s = mm.Solver.from_problem(wl.paper_jets(n, two=False))
    xc = (np.arange(n) + 0.5) / n
    speed_jet = 5.0 * np.sqrt(5.0 / 3.0)
    fronts = []
    for t in (0.02, 0.04):
        s.advance_to(t, 0.5)
        W = s.get_state_prim()[:, n // 2]                       # the jet axis y = 0.5
        rho, P = W[0], (W[4] + W[7] + W[9]) / 3.0
        Rs = W[13] * rho / P ** 2
        qs = W[10] / (rho * (P / rho) ** 1.5)
        x_rho = xc[np.nonzero(rho > 0.1)[0].max()]
        x_R = xc[np.nonzero(np.abs(Rs - 15.0) > 0.15)[0].max()]
        fronts.append((x_rho, x_R))
        assert np.allclose(Rs[-10:], 15.0, rtol=1e-12) and np.abs(qs[-10:]).max() < 1e-12
    v_rho = (fronts[1][0] - fronts[0][0]) / 0.02
    v_R = (fronts[1][1] - fronts[0][1]) / 0.02
    assert 0.9 * speed_jet < v_rho < 1.4 * speed_jet            # 6.45: measured 7.7 (front = jet + thermal spread)
    assert 1.6 < v_R / v_rho < 2.3                              # measured 1.8


def test_crossing_jets_reseparate_only_when_collisionless(mm):
    """The paper's central 2-D result (Fig 13; L472-494, Fig 15; App C): two
    collisionless jets crossing at a right angle pass through each other and leave the domain
    straight ahead, which no Euler-like model can do; with many collisions (Kn = 0.01) they merge
    into one stream leaving along the diagonal.  300^2 cells to t = 0.3 (25 000 and 110 000 steps)."""
    n = 300
    yc = (np.arange(n) + 0.5) / n
    k9, k5 = int(0.9 * n), n // 2
    out = {}
    for Kn in (None, 0.01):
        s = mm.Solver.from_problem(wl.paper_jets(n, two=True, Kn=Kn))
        s.advance_to(0.3, 0.5)
        U = s.get_state()
        assert s.info()["t"] == 0.3 and np.all(np.isfinite(U)) and U[0].min() > 0
        out[Kn] = U[0]
    free, coll = out[None], out[0.01]
    # collisionless: each jet exits opposite to where it entered; nothing leaves through the corner
    assert abs(yc[free[:, -1].argmax()] - 0.5) < 0.08 and abs(yc[free[-1, :].argmax()] - 0.5) < 0.08
    assert free[k5, k9] > 5.0 * free[k9, k9] and free[k9, k5] > 5.0 * free[k9, k9]
    # collisional: one merged stream along the diagonal
    assert yc[coll[:, -1].argmax()] > 0.65 and yc[coll[-1, :].argmax()] > 0.65
    assert coll[k9, k9] > coll[k5, k9] and coll[k9, k9] > coll[k9, k5]
    # the set-up is symmetric under x <-> y and so are both solutions, up to the round-off the scheme
    # amplifies over 10^4 - 10^5 steps (R24; the two directions are not evaluated in the same order)
    for rho in (free, coll):
        assert np.abs(rho - rho.T).mean() < 0.05 * rho.mean()


# ----------------- midpoint time marching (L250), point-implicit source (L348)
@pytest.mark.parametrize("opts", [dict(source_scheme=wl.SRC_POINT_IMPLICIT), dict(time_scheme=wl.TIME_MIDPOINT)])
@pytest.mark.parametrize("case", ["smooth14", "smooth14_zsym", "smooth5", "jets", "sod14"])
def test_time_and_source_schemes(mm, mmo, opts, case):
    if case == "smooth14":
        prob, n, cfl = wl.random_smooth14(70, 37, Kn=0.05, **opts), 30, 0.4
    elif case == "smooth14_zsym":
        prob, n, cfl = wl.random_smooth14(70, 37, Kn=0.05, zsym=True, flux=wl.FLUX_RUSANOV, **opts), 30, 0.4
    elif case == "smooth5":
        prob, n, cfl = wl.random_smooth5(333, Kn=0.05, **opts), 100, 0.5
    elif case == "jets":
        prob, n, cfl = wl.crossed_jets(96, Kn=1.0, **opts), 100, 0.4
    else:
        prob, n, cfl = wl.sod14(1024, 4, Kn=1e-3, **opts), 100, 0.5
    Ug, Uo = run_both(mm, mmo, prob, n, cfl=cfl)
    assert_parity(Ug, Uo)
    # CFL stepping: same dt sequence (the midpoint scheme takes dt from the CFL rate of U^n)
    so = oracle_solver(mmo, prob); sg = mm.Solver.from_problem(prob)
    so.step(10, cfl); sg.step(10, cfl)
    assert sg.info()["t"] == pytest.approx(so.info()["t"], rel=1e-10)
    assert sg.info()["steps"] == 10


def test_point_implicit_sod5_small_knudsen(mm, mmo):
    """dt ~ 30 tau (Kn = 1e-5, CFL 0.5): the point-implicit source runs the whole tube to t = 0.2 and
    matches the oracle; both reproduce the Euler (gamma = 3) limit (oracle pin in test_oracle_scheme)."""
    prob = wl.sod5(400, Kn=1e-5, source_scheme=wl.SRC_POINT_IMPLICIT)
    so = oracle_solver(mmo, prob); sg = mm.Solver.from_problem(prob)
    so.advance_to(0.2, 0.5); sg.advance_to(0.2, 0.5)
    assert sg.info()["steps"] == so.info()["steps"]
    assert_parity(sg.get_state(), so.get_state(), 1e-9)


def test_scheme_option_errors(mm):
    with pytest.raises(mm.MMError) as e:
        mm.Solver(14, 8, 8, time_scheme=wl.TIME_MIDPOINT, source_scheme=wl.SRC_POINT_IMPLICIT)
    assert e.value.status == mm.EINVAL
    with pytest.raises(mm.MMError):
        mm.Solver(14, 8, 8, time_scheme=2)


# ---------------------------------------- the paper's own jet configuration
@pytest.mark.parametrize("two", [False, True])
def test_paper_jets_parity(mm, mmo, two):
    """M = 5 jets of width L/7 into a 1e-5 background, collisionless, Rusanov +
    van Albada with one shared psi, sigma_lim = 1e-4.
    This start is the worst-conditioned case in the suite: the fast-wave front sits on the Junk line
    (sigma just above sigma_lim, closing fluxes ~ 1/sigma^3 sensitive), and an ORACLE run perturbed by
    1e-15 after every step differs from the unperturbed one by 3e-13 after 2 steps and by 3 % after 3
    (measured below).  So: element-wise 1e-10 parity over the first 2 steps, the CFL time step of the
    first steps, and after 100 steps the density field within 10x the oracle's own round-off noise."""
    prob = wl.paper_jets(64, two=two)
    dt = 0.5 * scout_dt(mmo, prob, 100, 0.5)
    Ug, Uo = run_both(mm, mmo, prob, 2, dt=dt, fast=True)
    assert_parity(Ug, Uo)
    so = oracle_solver(mmo, prob); sg = mm.Solver.from_problem(prob)
    for _ in range(2):
        so.step(1, 0.5); sg.step(1, 0.5)
        assert sg.info()["last_dt"] == pytest.approx(so.info()["last_dt"], rel=1e-9)
    # 100 steps: three runs (oracle, perturbed oracle, GPU) compared through the density field
    so, sp, sg = oracle_solver(mmo, prob), oracle_solver(mmo, prob), mm.Solver.from_problem(prob)
    rng = np.random.default_rng(1)
    for _ in range(100):
        so.step_fixed_dt(1, dt); sp.step_fixed_dt(1, dt)
        Up = sp.get_state()
        sp.set_state(Up * (1.0 + 1e-15 * rng.integers(-2, 3, size=Up.shape)))
    sg.step_fixed_dt(100, dt)
    Uo, Up, Ug = so.get_state(), sp.get_state(), sg.get_state()
    noise = np.abs(Up[0] - Uo[0]).mean()
    assert noise > 1e-9 * np.abs(Uo[0]).mean()              # the ill-conditioning is real
    assert np.all(np.isfinite(Ug)) and Ug[0].min() > 0
    assert np.abs(Ug[0] - Uo[0]).mean() <= 10.0 * noise
    for m in (3, 6, 8, 12):
        assert np.all(Ug[m] == 0.0)
    # mass is transported, not created: totals agree to the noise level too
    assert abs(Ug[0].sum() - Uo[0].sum()) <= 10.0 * max(abs(Up[0].sum() - Uo[0].sum()), 1e-12 * Uo[0].sum())


def test_paper_crossing_jets_time_step_drop(mm):
    """PAPER.md L466-470, Fig 14: the two-jet run needs the same CFL time step as the single-jet run
    while the jets are independent, and a markedly smaller one once their fast waves interact
    ("around time step 9000" on the paper's 1200^2 grid, i.e. ~2250 on this 300^2 grid)."""
    n, chunk, nchunks = 300, 100, 32
    dts = {}
    for two in (False, True):
        s = mm.Solver.from_problem(wl.paper_jets(n, two=two))
        assert s.fast_path_active
        h, t_prev = [], 0.0
        for _ in range(nchunks):
            s.step(chunk, 0.5)
            t = s.info()["t"]
            h.append((t - t_prev) / chunk)      # mean time step of the chunk (a single step's dt jitters:
            t_prev = t                          # the fastest cell sits on the Junk line, R24)
        U = s.get_state()
        assert np.all(np.isfinite(U)) and U[0].min() > 0
        dts[two] = np.array(h)
    ratio = dts[True] / dts[False]
    assert np.all(np.abs(ratio[:8] - 1.0) < 0.3)            # steps 100 .. 800: independent jets
    assert ratio[-3:].max() < 0.5                            # steps 3000 .. 3200: after the interaction


def test_dt_history_and_checkpoint_resume(mm, mmo):
    """The device-side dt history equals the oracle's step-by-step dt (Fig 14 is this
    curve), and get_state + info / set_state + set_clock resume a run bit for bit."""
    prob = wl.crossed_jets(64, Kn=1.0)
    sg = mm.Solver.from_problem(prob); so = oracle_solver(mmo, prob)
    sg.step(60, 0.4)
    hist = sg.dt_history(0, 60)
    ref = []
    for _ in range(60):
        so.step(1, 0.4); ref.append(so.info()["last_dt"])
    assert np.allclose(hist, ref, rtol=1e-9, atol=0)
    assert hist.sum() == pytest.approx(sg.info()["t"], rel=1e-13)
    assert np.array_equal(sg.dt_history(57, 3), hist[57:])
    with pytest.raises(mm.MMError):
        sg.dt_history(58, 5)                                    # steps 60.. not taken yet
    # checkpoint after 60 steps, 20 more; resume a fresh solver from the checkpoint, 20 more
    U60, inf = sg.get_state(), sg.info()
    sg.step(20, 0.4)
    s2 = mm.Solver.from_problem(prob, load_state=False)
    s2.set_state(U60); s2.set_clock(inf["t"], inf["steps"])
    s2.step(20, 0.4)
    assert np.array_equal(s2.get_state(), sg.get_state())
    assert s2.info()["t"] == sg.info()["t"] and s2.info()["steps"] == 80
    assert np.array_equal(s2.dt_history(60, 20), sg.dt_history(60, 20))


@pytest.mark.parametrize("scheme", ["midpoint", "point_implicit"])
@pytest.mark.parametrize("system", [14, 5])
def test_checkpoint_resume_other_schemes(mm, scheme, system):
    """include/mm.h promises that get_state + info / set_state + set_clock resume a run bit for bit, whatever the
    scheme: the CFL rate of the restored state must come out of the same instructions that produced it in the
    original run (midpoint: the second pass of a step; point-implicit source, L348)."""
    opt = dict(time_scheme=wl.TIME_MIDPOINT) if scheme == "midpoint" else dict(source_scheme=wl.SRC_POINT_IMPLICIT)
    prob = wl.crossed_jets(64, Kn=1.0, **opt) if system == 14 else wl.sod5(400, Kn=0.01, **opt)
    sg = mm.Solver.from_problem(prob)
    sg.step(40, 0.4)
    U40, inf = sg.get_state(), sg.info()
    sg.step(25, 0.4)
    s2 = mm.Solver.from_problem(prob, load_state=False)
    s2.set_state(U40); s2.set_clock(inf["t"], inf["steps"])
    assert s2.cfl_dt(0.4) == sg.dt_history(40, 1)[0]            # the first dt after the checkpoint, to the bit
    s2.step(25, 0.4)
    assert np.array_equal(s2.dt_history(40, 25), sg.dt_history(40, 25))
    assert np.array_equal(s2.get_state(), sg.get_state())
    assert s2.info()["t"] == sg.info()["t"] and s2.info()["steps"] == 65


# ------------------------------ batched 1-D 5-moment tubes (sigma_lim x Kn sweep)
def _tube_oracles(mmo, nx, sigma_lims, Kns, **opt):
    out = []
    for sl, kn in zip(sigma_lims, Kns):
        prob = wl.sod5(nx, Kn=kn, sigma_lim=sl, **opt)
        out.append(oracle_solver(mmo, prob))
    return out


def test_batch5_matches_independent_oracle_tubes(mm, mmo):
    """Every tube of a batch equals its own 1-D oracle run: different sigma_lim and Kn per tube
    (one collisionless), 100 steps at a common fixed dt, then CFL stepping where every tube takes
    its own dt and lands on t_end by itself."""
    nx = 333
    sig = [1e-4, 1e-3, 1e-2, 1e-4, 1e-5]
    kns = [0.01, 0.1, 1.0, None, 0.001]
    W0 = wl.sod5(nx, Kn=0.01)["W0"].reshape(5, nx)
    b = mm.Batch5(nx, sig, kns)
    b.set_state_prim(W0)
    dt = 0.5 * min(scout_dt(mmo, wl.sod5(nx, Kn=kn, sigma_lim=sl), 100, 0.5) for sl, kn in zip(sig, kns))
    tubes = _tube_oracles(mmo, nx, sig, kns)
    b.step_fixed_dt(100, dt)
    Ub = b.get_state()
    for j, t in enumerate(tubes):
        t.step_fixed_dt(100, dt)
        assert_parity(Ub[j].reshape(5, 1, nx), t.get_state())
    assert np.allclose(b.info()["t"], 100 * dt, rtol=1e-13)
    # own CFL time steps, own clocks: element-wise over the first 30 steps ...
    b.set_state_prim(W0)
    tubes = _tube_oracles(mmo, nx, sig, kns)
    b.step(30, 0.5)
    inf = b.info()
    Ub = b.get_state()
    for j, t in enumerate(tubes):
        t.step(30, 0.5)
        assert inf["t"][j] == pytest.approx(t.info()["t"], rel=1e-9)
        assert_parity(Ub[j].reshape(5, 1, nx), t.get_state(), 1e-8)
    assert len(set(np.round(inf["t"], 12).tolist())) > 1       # the tubes really have their own clocks
    # ... and to t_end through what is robust to round-off (R24): every tube lands on t_end
    # by itself, with a step count and a density profile close to its oracle's
    b.advance_to(0.03, 0.5)
    inf = b.info()
    Ub = b.get_state()
    for j, t in enumerate(tubes):
        t.advance_to(0.03, 0.5)
        assert inf["t"][j] == 0.03
        # (the step COUNT of a single run is chaotic at small sigma_lim and is compared as a distribution,
        # test_batch5_step_count_distribution_matches_the_oracle)
        rho_o = t.get_state()[0, 0]
        assert np.abs(Ub[j, 0] - rho_o).mean() <= 5e-3 * rho_o.mean()
    assert len(set(inf["steps"].tolist())) > 1


def test_batch5_step_count_distribution_matches_the_oracle(mm, mmo):
    """The number of CFL steps to t_end (the paper's cost measure, L342) is round-off chaotic at small sigma_lim:
    oracle runs of the SAME tube (sigma_lim 1e-4, Kn 0.01, 333 cells, t_end 0.03) whose initial states differ by
    1e-15 relative need between ~770 and ~1210 steps (measured over 24 runs, R24), so one GPU count
    against one oracle count says nothing.  The batch runs the same 48 states as 48 tubes: the two count distributions must
    agree -- medians within 12 %, quartiles within 20 %, every tube inside the oracle's range widened by its own
    spread -- and every tube lands on t_end."""
    nx, sl, kn, ne = 333, 1e-4, 0.01, 48          # 48 samples: the medians' sampling noise is ~3.5 %, the bar 12 %
    prob = wl.sod5(nx, Kn=kn, sigma_lim=sl)
    Ws = []
    for seed in range(ne):
        W = prob["W0"].copy()
        if seed:
            W *= 1.0 + 1e-15 * np.random.default_rng(seed).standard_normal(W.shape)
        Ws.append(W.reshape(5, nx))
    b = mm.Batch5(nx, [sl] * ne, [kn] * ne)
    b.set_state_prim(np.stack(Ws))
    b.advance_to(0.03, 0.5)
    inf = b.info()
    assert np.all(inf["t"] == 0.03)
    g = np.sort(inf["steps"].astype(float))
    o = []
    for W in Ws:
        so = oracle_solver(mmo, prob)
        so.set_state_prim(W.reshape(5, 1, nx))
        so.advance_to(0.03, 0.5)
        o.append(so.info()["steps"])
    o = np.sort(np.array(o, dtype=float))
    assert o.max() > 1.2 * o.min()                               # the premise: the count is chaotic in the oracle itself
    assert abs(np.median(g) - np.median(o)) <= 0.12 * np.median(o), (g, o)
    for qt in (0.25, 0.75):
        assert abs(np.quantile(g, qt) - np.quantile(o, qt)) <= 0.20 * np.quantile(o, qt), (g, o)
    spread = o.max() - o.min()
    assert g.min() >= o.min() - spread and g.max() <= o.max() + spread, (g, o)


def test_batch5_cost_rises_as_sigma_lim_falls(mm):
    """PAPER.md L318-320, L350 (Fig 7-Left): a smaller sigma_lim lets the solution climb closer to the
    Junk line, wave speeds grow and the run needs more time steps; collisions (small Kn) lower the cost
    (L346).  64 tubes = 8 sigma_lim x 8 Kn in one batch, Sod tube to t = 0.1."""
    nx = 500
    sig = np.repeat([1e-1, 3e-2, 1e-2, 3e-3, 1e-3, 3e-4, 1e-4, 1e-5], 8)
    kns = np.tile([1e-3, 3e-3, 1e-2, 3e-2, 1e-1, 0.3, 1.0, 0.0], 8)      # 0.0: collisionless
    b = mm.Batch5(nx, sig, kns)
    b.set_state_prim(wl.sod5(nx, Kn=0.01)["W0"].reshape(5, nx))
    b.advance_to(0.1, 0.5)
    inf = b.info()
    assert np.all(inf["t"] == 0.1) and not inf["failed"].any()
    steps = inf["steps"].reshape(8, 8)                           # [sigma_lim][Kn]
    U = b.get_state()
    assert np.all(np.isfinite(U)) and U[:, 0].min() > 0
    collisionless = steps[:, 7]
    assert np.all(np.diff(collisionless) >= 0) and collisionless[-1] > 3 * collisionless[0]
    assert np.all(steps[6, :] >= steps[2, :])                    # sigma_lim 1e-4 never cheaper than 1e-2
    assert steps[6, 0] < steps[6, 7]                             # Kn = 1e-3 cheaper than collisionless


def test_batch5_errors(mm):
    with pytest.raises(mm.MMError):
        mm.Batch5(100, [1e-4, 0.0], [0.1, 0.1])                  # sigma_lim must be positive
    with pytest.raises(ValueError):
        mm.Batch5(100, [1e-4], [0.1, 0.2])
    b = mm.Batch5(64, [1e-4, 1e-4], [0.1, 1.0])
    with pytest.raises(mm.MMError):
        b.step(1, 0.5)                                           # no state yet
    W = wl.sod5(64, Kn=0.1)["W0"].reshape(5, 64).copy()
    Wb = np.stack([W, W]); Wb[1, 2, 10] = -1.0                   # negative pressure in tube 1 only
    b.set_state_prim(Wb)
    b.step(5, 0.5)
    inf = b.info(check=False)
    assert inf["status"] == mm.ENONFINITE and list(inf["failed"]) == [0, 1]
    assert inf["steps"][0] == 5 and inf["steps"][1] == 0        # the healthy tube keeps going


# ------------------------------------------------------------------------ error behaviour
def test_errors_and_failure_flag(mm, mmo):
    with pytest.raises(mm.MMError) as e:
        mm.Solver(14, 8, 8, sigma_lim=0.0)
    assert e.value.status == mm.EINVAL
    with pytest.raises(mm.MMError):
        mm.Solver(5, 8, 2)
    with pytest.raises(mm.MMError):
        mm.Solver(14, 8, 8, bcs=[dict(type=wl.BC_PERIODIC), dict(type=wl.BC_TRANSMISSIVE)] * 2)
    prob = wl.random_smooth14(16, 16)
    s = mm.Solver.from_problem(prob, load_state=False)
    with pytest.raises(mm.MMError):
        s.step(1, 0.4)                                 # no state yet
    s.set_state_prim(prob["W0"])
    s.step(0, 0.4)                                     # empty request is a no-op
    assert s.info()["steps"] == 0
    W = prob["W0"].copy()
    W[4, 3, 3] = W[7, 3, 3] = W[9, 3, 3] = -1.0        # negative pressure
    s.set_state_prim(W)
    U0 = s.get_state()
    s.step(3, 0.4)
    inf = s.info(check=False)
    assert inf["status"] == mm.ENONFINITE and inf["steps"] == 0
    assert np.array_equal(s.get_state(), U0)           # state left as is for inspection
