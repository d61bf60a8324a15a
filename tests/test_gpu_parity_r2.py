"""GPU parity, second set: the bar at the size the metric is quoted on, and element-wise evidence on
developed (ill-conditioned) states that does not depend on how the scheme amplifies round-off.

  * BASELINE configs[3] (2048^2 crossed jets): 100 steps at fixed dt on the FULL grid against the
    oracle, 1e-10 per moment (north_star; SURVEY.md section 8(d) "at 2048^2 once");
    configs[4] (4096^2): the same 100 steps on windows with a 2 x 100 + 1 cell margin, each window
    scaled by max(its own per-moment maximum, rho c^n) (reading R25; the fixed dt is reading R26).
  * Re-synchronised single steps: the oracle marches a developed state; before every step its state is
    handed to the GPU (mm_set_state), both take ONE step, every cell is compared.  Amplification across
    steps never enters, so the per-step bar is a property of one step's arithmetic.
  * Boundary: Maxwellian Dirichlet states through mm_gas (R_gas), the NaN failure path of an
    indefinite pressure tensor, the dt-history range after mm_set_clock, grids taller than 65535 rows.
"""
import numpy as np
import pytest

import mm_workloads as wl
from parity_util import moment_errors, window_errors

pytestmark = pytest.mark.gpu

TOL = 1e-10          # north_star: max relative error per moment after 100 steps at fixed dt
STEP_TOL = 1e-10     # one re-synchronised step on a developed state (derivation)


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


def inflow_scout_dt(mmo, prob, n, nsteps, cfl):
    """Smallest CFL time step the oracle takes over `nsteps` steps on a window of the SAME seeded state and
    cell size at the inflow side (96 columns from the left wall, y in [0.2, 0.8]): as the jets enter, the wave
    speeds at their fronts grow far beyond those of the starting state (sigma -> sigma_lim),
    so the starting state's own CFL step is not a stable fixed dt.  100 steps move the fronts < 40 cells."""
    h = 1.0 / n
    j0, j1, w = int(0.2 * n), int(0.8 * n), 96
    sub = dict(prob, nx=w, ny=j1 - j0, W0=np.ascontiguousarray(prob["W0"][:, j0:j1, :w]),
               extent=(0.0, w * h, j0 * h, j1 * h))
    so = oracle_solver(mmo, sub)
    dts = []
    for _ in range(nsteps):
        so.step(1, cfl)
        dts.append(so.info()["last_dt"])
    return min(dts)


# --------------------------------------------------------------- the bar at the headline size
@pytest.mark.parametrize("Kn", [0.1, 1.0])
def test_C4_full_grid_2048_100_steps(mm, mmo, Kn):
    """configs[3] as bench.py runs it (seeded +-1 % density, Kn 0.1 and 1, z-symmetric kernel variant, bench
    launch decomposition): 100 fixed-dt steps, every one of the 4 194 304 cells, all 14 moments."""
    n, nsteps = 2048, 100
    prob = wl.crossed_jets(n, Kn=Kn, perturb=0.01)
    so = oracle_solver(mmo, prob)
    sg = mm.Solver.from_problem(prob)
    assert sg.fast_path_active
    assert sg.cfl_dt(0.4) == pytest.approx(so.cfl_dt(0.4), rel=1e-10)
    dt = 0.5 * inflow_scout_dt(mmo, prob, n, nsteps, 0.4)      # half the smallest CFL-0.4 step of the 100 steps
    sg.step_fixed_dt(nsteps, dt)
    so.step_fixed_dt(nsteps, dt)
    Ug, Uo = sg.get_state(), so.get_state()
    assert np.all(np.isfinite(Uo)) and np.all(np.isfinite(Ug))
    e = moment_errors(Ug, Uo)
    assert e.max() <= TOL, f"per-moment rel. error {e}"
    # the jets have entered: the state is not the initial one
    assert Uo[0][int(0.35 * n), 0] > 0.5 and Uo[0][int(0.5 * n), 0] < 2e-3 and Uo[0].max() > 0.8


@pytest.mark.parametrize("fast", [True, False])
def test_C5_4096_100_steps_windows(mm, mmo, fast):
    """configs[4] (4096^2, Kn 0.1): 100 fixed-dt steps; a cell depends on the 2-cell stencil per step,
    so the oracle recomputes windows of the same seeded state with a 201-cell margin to every cut edge
    (and none to the true left boundary, which the window keeps) and the inner cells are compared,
    each window scaled by max(own per-moment maximum, rho c^n) (parity_util.window_errors, R25).
    Windows sit on the inflow bands, between them,
    in the far field and across strip / row-chunk boundaries of the launch decomposition."""
    n, nsteps, margin, inner = 4096, 100, 201, 48
    prob = wl.crossed_jets(n, Kn=0.1, perturb=0.01)
    sg = mm.Solver.from_problem(prob)
    sg.set_fast_path(fast)
    assert sg.fast_path_active == fast
    dt = 0.5 * inflow_scout_dt(mmo, prob, n, nsteps, 0.4)
    sg.step_fixed_dt(nsteps, dt)
    Ug = sg.get_state()
    assert np.all(np.isfinite(Ug))
    W0 = prob["W0"]
    h = 1.0 / n
    w = inner + 2 * margin
    # (i0, j0) of the window's lower-left cell; i0 = 0 keeps the Dirichlet side
    spots = [(0, int(0.35 * n) - w // 2), (0, int(0.65 * n) - w // 2), (0, int(0.5 * n) - w // 2)]
    if fast:
        spots += [(30 * 60 - margin - 7, n * 9 // 35), (n - w, n - w), (1500, 5)]
    for (i0, j0) in spots:
        sub = dict(prob, nx=w, ny=w, W0=np.ascontiguousarray(W0[:, j0:j0 + w, i0:i0 + w]),
                   extent=(i0 * h, (i0 + w) * h, j0 * h, (j0 + w) * h))
        if i0 > 0:
            sub["bcs"] = [dict(type=wl.BC_TRANSMISSIVE)] * 4
        so = oracle_solver(mmo, sub)
        so.step_fixed_dt(nsteps, dt)
        Uo = so.get_state()
        # cut edges need the margin; true domain edges (left wall at i0 = 0, top / right / bottom when the
        # window touches them) are reproduced by the window's own boundary condition
        lo_i = 0 if i0 == 0 else margin
        hi_i = w if i0 + w == n else w - margin
        lo_j = 0 if j0 == 0 else margin
        hi_j = w if j0 + w == n else w - margin
        sl = (slice(None), slice(lo_j, hi_j), slice(lo_i, hi_i))
        assert np.all(np.isfinite(Uo))
        e = window_errors(Ug[:, j0:j0 + w, i0:i0 + w][sl], Uo[sl])
        assert e.max() <= TOL, ((i0, j0), e)


# ------------------------------------------------------- re-synchronised steps, developed states
def resync_steps(mm, mmo, prob, U0, nsteps, dt, fast=None, tol=STEP_TOL):
    """Oracle marches from U0; before each step the GPU is given the oracle's state, both take one
    step of size dt, and all cells of all moments are compared.  Returns the per-step worst error."""
    so = oracle_solver(mmo, prob)
    so.set_state(U0)
    sg = mm.Solver.from_problem(prob, load_state=False)
    worst = []
    for k in range(nsteps):
        Uk = so.get_state()
        sg.set_state(Uk)
        if fast is not None and prob["system"] == 14:
            sg.set_fast_path(fast)
            assert sg.fast_path_active == fast
        so.step_fixed_dt(1, dt)
        sg.step_fixed_dt(1, dt)
        Uo, Ug = so.get_state(), sg.get_state()
        assert np.all(np.isfinite(Uo)), f"oracle state not finite at step {k}"
        e = moment_errors(Ug, Uo)
        assert e.max() <= tol, f"step {k}: per-moment rel. error {e}"
        worst.append(e.max())
    return np.array(worst)


@pytest.mark.parametrize("fast", [True, False])
def test_resync_crossed_jets_after_the_crossing(mm, mmo, fast):
    """BASELINE configs[2] shape on 128^2, HLL + shared minmod, k = 1.2 (the k = 1 run loses positivity at
    t = 0.1375 in the oracle itself, R14): state at t = 0.15, after the jets have crossed."""
    prob = wl.crossed_jets(128, Kn=1.0, ws_scale=1.2)
    so = oracle_solver(mmo, prob)
    so.advance_to(0.15, 0.4)
    U0 = so.get_state()
    dt = 0.5 * so.cfl_dt(0.4)
    resync_steps(mm, mmo, prob, U0, 50, dt, fast=fast)


@pytest.mark.parametrize("two", [False, True])
def test_resync_paper_jets_fast_wave_front(mm, mmo, two):
    """The paper's own configuration (Rusanov + van Albada, shared psi, M = 5 into 1e-5, collisionless,
    PAPER.md L426-434) on 96^2 after 150 CFL steps: the fourth-moment wave runs ahead of the density
    front with sigma just above sigma_lim (the worst-conditioned states of the suite)."""
    prob = wl.paper_jets(96, two=two)
    so = oracle_solver(mmo, prob)
    so.step(150, 0.5)
    U0 = so.get_state()
    dt = 0.5 * so.cfl_dt(0.5)
    resync_steps(mm, mmo, prob, U0, 50, dt, fast=True)


def test_resync_sod5_step_300(mm, mmo):
    """BASELINE configs[0]: the 5-moment Sod tube after 300 CFL steps (where two free-running fp64 runs
    have already diverged by > 1e-4, R24), 50 re-synchronised steps."""
    prob = wl.sod5(1000, Kn=0.01)
    so = oracle_solver(mmo, prob)
    so.step(300, 0.5)
    U0 = so.get_state()
    dt = 0.5 * so.cfl_dt(0.5)
    resync_steps(mm, mmo, prob, U0, 50, dt)


def test_resync_sod14_collisionless_front(mm, mmo):
    """BASELINE configs[1] shape at Kn = 1, after 200 CFL steps (HLL oscillations of PAPER.md L258 present)."""
    prob = wl.sod14(1024, 4, Kn=1.0)
    so = oracle_solver(mmo, prob)
    so.step(200, 0.5)
    U0 = so.get_state()
    dt = 0.5 * so.cfl_dt(0.5)
    resync_steps(mm, mmo, prob, U0, 30, dt, fast=True)


@pytest.mark.parametrize("limiter", [wl.LIM_MINMOD, wl.LIM_VANALBADA])
def test_resync_smooth14_general_variant_shared_limiter(mm, mmo, limiter):
    """The one combination that only had a condition-aware bar: fully 3-D data (non-zero u_z, P_xz, P_yz, q_z),
    the general kernel variant and ONE limiter value for all 14 primitives ("the most stringent").
    30 re-synchronised steps of random_smooth14(70, 37) at the flat 1e-10."""
    prob = wl.random_smooth14(70, 37, Kn=0.1, limiter=limiter, shared_limiter=1)
    assert all(np.abs(prob["W0"][m]).max() > 1e-3 for m in (3, 6, 8, 12))
    so = oracle_solver(mmo, prob)
    U0 = so.get_state()
    dt = 0.5 * so.cfl_dt(0.4)
    sg = mm.Solver.from_problem(prob)
    assert not sg.fast_path_active                          # z-odd moments present: the general variant runs
    resync_steps(mm, mmo, prob, U0, 30, dt)


@pytest.mark.parametrize("axis, zsym", [(0, True), (1, True), (0, False), (1, False)])
def test_anisotropic_pressure_takes_the_direct_wave_speed_path(mm, mmo, axis, zsym):
    """P_dd* < 1/32 along one direction: every face evaluation of that direction inside the step kernel leaves
    the a(P*), b(P*) table (Eq 29c-d) and redoes its wave speeds with the formulas themselves, lane by lane,
    right before the warp-collective tensor-memory instructions.  25 steps at fixed dt, both kernel variants."""
    prob = wl.anisotropic14(70, 37, axis=axis, zsym=zsym, ratio=0.02)      # collisionless: the anisotropy persists
    W0 = prob["W0"]
    Ph = (W0[4] + W0[7] + W0[9]) / 3.0
    assert (W0[(4, 7)[axis]] / Ph).max() < 1.0 / 32.0
    so = oracle_solver(mmo, prob)
    dts = []
    for _ in range(25):
        so.step(1, 0.4)
        dts.append(so.info()["last_dt"])
    Wend = so.get_state_prim()
    assert (Wend[(4, 7)[axis]] / ((Wend[4] + Wend[7] + Wend[9]) / 3.0)).max() < 1.0 / 32.0    # every cell still out of the table's range
    dt = 0.5 * min(dts)
    so = oracle_solver(mmo, prob)
    sg = mm.Solver.from_problem(prob)
    assert sg.fast_path_active == zsym
    so.step_fixed_dt(25, dt); sg.step_fixed_dt(25, dt)
    Uo, Ug = so.get_state(), sg.get_state()
    assert np.all(np.isfinite(Uo))
    e = moment_errors(Ug, Uo)
    assert e.max() <= TOL, e


# ------------------------------------------------------------------------------ boundary
def test_maxwellian_dirichlet_states_use_R_gas(mm, mmo):
    """mm_gas (include/mm.h): Dirichlet states given as (rho, u, T) are expanded on the device to the
    Maxwellian of PAPER.md L73 with P = rho R_gas T.  The oracle is given the primitive states written
    out here from that definition; both run the same 40 steps."""
    R_gas, n = 208.13, 48                                   # argon, J/(kg K)
    rho_j, T_j, rho_b, T_b = 1.0, 300.0, 1e-3, 300.0
    speed = 3.0 * np.sqrt(5.0 / 3.0 * R_gas * T_j)          # M = 3 (L428: a = sqrt(gamma R T))
    ang = np.deg2rad(20.0)

    def maxwellian_prim(rho, ux, uy, T):
        P = rho * R_gas * T
        return np.array([rho, ux, uy, 0, P, 0, 0, P, 0, P, 0, 0, 0, 15 * P * P / rho])

    bands_T = [(0.3, 0.4, [rho_j, speed * np.cos(ang), speed * np.sin(ang), 0.0, T_j]),
               (0.6, 0.7, [rho_j, speed * np.cos(ang), -speed * np.sin(ang), 0.0, T_j])]
    bands_W = [(lo, hi, maxwellian_prim(s[0], s[1], s[2], s[4])) for lo, hi, s in bands_T]
    tr = dict(type=wl.BC_TRANSMISSIVE)
    W0 = np.broadcast_to(maxwellian_prim(rho_b, 0, 0, T_b)[:, None, None], (14, n, n)).copy()
    common = dict(system=14, nx=n, ny=n, extent=(0.0, 1.0, 0.0, 1.0), W0=W0,
                  collision=dict(model=wl.TAU_KN, Kn=1.0, L_ref=0.1, rho_ref=1.0),
                  options=dict(sigma_lim=1e-4, ws_scale=1.0, limiter=wl.LIM_MINMOD, shared_limiter=1, flux=wl.FLUX_HLL))
    prob_o = dict(common, bcs=[dict(type=wl.BC_DIRICHLET, bands=bands_W, default=maxwellian_prim(rho_b, 0, 0, T_b)), tr, tr, tr])
    bcs_g = [dict(type=wl.BC_DIRICHLET, bands=bands_T, default=[rho_b, 0, 0, 0, T_b], state=mm.STATE_MAXWELLIAN), tr, tr, tr]
    so = oracle_solver(mmo, prob_o)
    sg = mm.Solver(14, n, n, extent=common["extent"], collision=common["collision"], bcs=bcs_g,
                   R_gas=R_gas, **common["options"])
    sg.set_state_prim(W0)
    assert sg.fast_path_active
    dt0 = sg.cfl_dt(0.4)
    assert dt0 == pytest.approx(so.cfl_dt(0.4), rel=1e-10)                  # the ghost states set the CFL rate
    dt = 0.5 * dt0
    so.step_fixed_dt(40, dt); sg.step_fixed_dt(40, dt)
    e = moment_errors(sg.get_state(), so.get_state())
    assert e.max() <= TOL, e
    # a different gas constant is a different problem
    s2 = mm.Solver(14, n, n, extent=common["extent"], collision=common["collision"], bcs=bcs_g,
                   R_gas=2 * R_gas, **common["options"])
    s2.set_state_prim(W0)
    assert s2.cfl_dt(0.4) < 0.95 * dt0          # hotter jets (P = rho 2R T): faster waves, u unchanged
    with pytest.raises(mm.MMError):
        mm.Solver(14, n, n, R_gas=-1.0)
    # 5-moment: (rho, u, ., ., T) -> (rho, u, P = rho R T, 0, 3 P^2/rho)  (L127)
    P = 0.5 * R_gas * 250.0
    W5 = np.array([0.5, 30.0, P, 0.0, 3 * P * P / 0.5])
    o5 = mmo.Solver(5, 64, 1, bcs=[dict(type=wl.BC_DIRICHLET, bands=[], default=W5), tr, tr, tr], collision=dict(model=wl.TAU_NONE))
    g5 = mm.Solver(5, 64, 1, bcs=[dict(type=wl.BC_DIRICHLET, bands=[], default=[0.5, 30.0, 0, 0, 250.0], state=mm.STATE_MAXWELLIAN), tr, tr, tr],
                   collision=dict(model=wl.TAU_NONE), R_gas=R_gas)
    W5_0 = np.broadcast_to(np.array([1.0, 0.0, R_gas * 300.0, 0.0, 3 * (R_gas * 300.0) ** 2])[:, None, None], (5, 1, 64)).copy()
    o5.set_state_prim(W5_0); g5.set_state_prim(W5_0)
    dt5 = 0.5 * o5.cfl_dt(0.5)
    o5.step_fixed_dt(30, dt5); g5.step_fixed_dt(30, dt5)
    assert moment_errors(g5.get_state(), o5.get_state()).max() <= TOL


def test_indefinite_pressure_tensor_fails_like_the_oracle(mm, mmo):
    """A cell whose pressure tensor is indefinite with a positive trace (P_xx = P_yy = P_zz = 1, P_xy = 2)
    and q = (1, -1, 0), R = 25 makes the radicand of Eq 21 negative: sigma is NaN.  The oracle reports a
    non-finite CFL rate for that state; the GPU must flag the same state (MM_ENONFINITE) and refuse to
    step, not carry on with sigma silently replaced by sigma_lim."""
    prob = wl.random_smooth14(33, 9, Kn=0.3, zsym=True)
    W = prob["W0"].copy()
    W[:, 4, 17] = [1.0, 0, 0, 0, 1.0, 2.0, 0, 1.0, 0, 1.0, 1.0, -1.0, 0, 25.0]
    assert np.isnan(mmo.sigma14(W[:, 4, 17]))
    so = oracle_solver(mmo, dict(prob, W0=W))
    assert not np.isfinite(so.cfl_dt(0.4))
    for fast in (True, False):
        sg = mm.Solver.from_problem(dict(prob, W0=W))
        sg.set_fast_path(fast)
        assert sg.info(check=False)["status"] == mm.ENONFINITE
        with pytest.raises(mm.MMError) as e:
            sg.cfl_dt(0.4)
        assert e.value.status == mm.ENONFINITE
        U0 = sg.get_state()
        sg.step(3, 0.4)                                   # enqueued, but every step is skipped
        assert sg.info(check=False)["steps"] == 0
        assert np.array_equal(sg.get_state(), U0, equal_nan=True)
    # the same cell one step later: a state that BECOMES indefinite is caught by the fused reduction
    good = wl.random_smooth14(33, 9, Kn=0.3, zsym=True)
    sg = mm.Solver.from_problem(good)
    sg.step(2, 0.4)
    assert sg.info()["steps"] == 2


def test_dt_history_range_after_set_clock(mm):
    """mm_get_dt_history after the documented resume path (mm_set_state + mm_set_clock(t, N)): steps
    before N were never taken by this solver and must be refused, not returned as zeros."""
    prob = wl.random_smooth14(40, 12, Kn=0.2, zsym=True)
    s = mm.Solver.from_problem(prob)
    s.step(7, 0.4)
    h = s.dt_history(0, 7)
    assert np.all(h > 0)
    U, inf = s.get_state(), s.info()
    r = mm.Solver.from_problem(prob, load_state=False)
    r.set_state(U); r.set_clock(inf["t"], inf["steps"])
    r.step(3, 0.4)
    assert r.info()["steps"] == 10
    assert np.all(r.dt_history(7, 3) > 0)
    for first, n in ((0, 7), (6, 2), (0, 10)):
        with pytest.raises(mm.MMError) as e:
            r.dt_history(first, n)
        assert e.value.status == mm.EINVAL
    s.step(3, 0.4)
    assert np.array_equal(s.dt_history(7, 3), r.dt_history(7, 3))       # bit-exact resume


def test_grid_taller_than_65535_rows(mm, mmo):
    """k_pack / k_unpack sweep rows with a grid-stride loop: ny > 65535 (CUDA's gridDim.y limit) works."""
    nx, ny = 3, 70001
    rng = np.random.default_rng(3)
    W = np.empty((14, ny, nx))
    W[:] = np.array([1.0, 0.1, -0.1, 0, 1.0, 0.05, 0, 0.9, 0, 1.1, 0.02, -0.03, 0, 16.0])[:, None, None]
    W[0] *= 1.0 + 0.01 * rng.uniform(-1, 1, size=(ny, nx))
    s = mm.Solver(14, nx, ny, extent=(0.0, 3.0 / ny, 0.0, 1.0), collision=dict(model=wl.TAU_NONE))
    s.set_state_prim(W)
    np.testing.assert_allclose(s.get_state_prim(), W, rtol=1e-12, atol=1e-14)
    U = s.get_state()
    s.set_state(U)
    assert np.array_equal(s.get_state(), U)
    # a few rows of it against the oracle after 3 steps (y-periodic window is not available: compare far
    # from the cut edges of a 64-row window)
    dt = 0.5 * s.cfl_dt(0.4)
    s.step_fixed_dt(3, dt)
    Ug = s.get_state()
    j0 = 66000
    so = mmo.Solver(14, nx, 64, extent=(0.0, 3.0 / ny, j0 / ny, (j0 + 64) / ny), collision=dict(model=wl.TAU_NONE))
    so.set_state_prim(W[:, j0:j0 + 64])
    so.step_fixed_dt(3, dt)
    Uo = so.get_state()
    assert moment_errors(Ug[:, j0 + 8:j0 + 56], Uo[:, 8:56]).max() <= TOL


# ------------------------------------------- memory safety and determinism without compute-sanitizer
# (compute-sanitizer is closed on this GPU pool, profiles/r2_sanitizer.md; these are its stand-ins)
@pytest.mark.parametrize("case", ["smooth14_midpoint", "smooth14_point_implicit", "jets", "zsym_periodic", "sod5"])
def test_no_write_outside_the_workspace(mm, case):
    """Every kernel of the path (pack, ghost fill, rate, the step kernel in all four instantiations, unpack)
    writes inside [workspace, workspace + mm_workspace_bytes): the solver runs in the middle of a buffer whose
    guard zones of 4 MB on either side carry a pattern that must survive bit for bit."""
    import torch
    if case == "smooth14_midpoint":
        prob = wl.random_smooth14(70, 37, Kn=0.05, time_scheme=wl.TIME_MIDPOINT)
    elif case == "smooth14_point_implicit":
        prob = wl.random_smooth14(61, 40, Kn=0.05, source_scheme=wl.SRC_POINT_IMPLICIT)
    elif case == "jets":
        prob = wl.crossed_jets(96, Kn=1.0)
    elif case == "zsym_periodic":
        prob = wl.random_smooth14(31, 9, Kn=0.2, zsym=True)
    else:
        prob = wl.sod5(333, Kn=0.01)
    nbytes = mm.mm_workspace_bytes(prob["system"], prob["nx"], prob["ny"], prob["extent"])
    guard = 4 << 20
    buf = torch.full((2 * guard + nbytes + 512,), 0xA5, dtype=torch.uint8, device="cuda")
    off = guard + (-(buf.data_ptr() + guard)) % 256
    s = mm.Solver.from_problem(prob, workspace=buf[off:off + nbytes + 255])
    assert s._ws_ptr == buf.data_ptr() + off
    s.step(25, 0.4)
    s.step_fixed_dt(5, 0.25 * s.cfl_dt(0.4))
    U = s.get_state()
    W = s.get_state_prim()
    s.set_state(U)
    s.step(3, 0.4)
    assert np.all(np.isfinite(U)) and np.all(np.isfinite(W))
    torch.cuda.synchronize()
    assert bool((buf[:off] == 0xA5).all()), "write below the workspace"
    assert bool((buf[off + nbytes:] == 0xA5).all()), "write above the workspace"


def test_runs_are_bitwise_reproducible(mm):
    """Two runs of the same problem give the same bits (state, time, dt sequence): the warp-local exchange through
    shared memory, cp.async and tensor memory in the step kernel has no race whose outcome varies from run to
    run, at a small ragged size and at the bench size in the bench launch configuration."""
    for prob, n in ((wl.random_smooth14(70, 37, Kn=0.05, zsym=True, shared_limiter=1), 40),
                    (wl.random_smooth14(70, 37, Kn=0.05), 40),
                    (wl.crossed_jets(2048, Kn=0.1, perturb=0.01), 12)):
        out = []
        for _ in range(2):
            s = mm.Solver.from_problem(prob)
            s.step(n, 0.4)
            out.append((s.get_state(), s.info()["t"], s.dt_history(0, n)))
            del s
        assert np.array_equal(out[0][0], out[1][0]) and out[0][1] == out[1][1] and np.array_equal(out[0][2], out[1][2])
