"""Pins of the CPU oracle's time step (oracle/mmo_scheme.c) against what the paper and the
mathematics fix -- invariants, closed forms and the exact Euler Riemann solution; none of them
re-types the oracle's update loop.

  * a uniform state stays uniform (bitwise), also next to Dirichlet ghosts holding that state;
  * on a periodic box all moments are conserved to round-off without collisions, and
    rho, rho u_i, tr U_ij with collisions (Eqs 17-18: C_1 = C_i = C_ii = 0);
  * x <-> y transpose symmetry of a full 2-D run (one routine, indices swapped);
  * a y-uniform 2-D run has identical rows;
  * uniform non-equilibrium gas, constant tau: forward Euler gives
    U_eq + (U_0 - U_eq)(1 - dt/tau)^n exactly (BGK is linear in U at fixed rho, u, P);
  * one first-order step equals the textbook finite-volume update assembled from the
    (separately pinned) pointwise flux / wave-speed / interface-flux functions;
  * the small-Kn Sod solution approaches the exact Euler Riemann solution (gamma = 3 for the
    1D1V gas, gamma = 5/3 for the 14-moment gas; values from SURVEY.md section 8(c));
  * point-implicit BGK source (L348): backward-Euler closed form for any dt/tau, second-order
    agreement with the explicit source, stable Sod solution at Kn = 1e-5;
  * midpoint scheme (L250): RK2 amplification factor of the uniform relaxation, second order in
    time against a fine-dt run.
"""
import math

import numpy as np
import pytest

import mm_workloads as wl


def oracle_solver(mmo, prob, nthreads=0, **override):
    opt = dict(prob["options"]); opt.update(override)
    s = mmo.Solver(prob["system"], prob["nx"], prob["ny"], extent=prob["extent"],
                   collision=prob["collision"], bcs=prob["bcs"], nthreads=nthreads, **opt)
    s.set_state_prim(prob["W0"])
    return s


# ----------------------------------------------------------------------------- uniform
@pytest.mark.parametrize("bc", ["periodic", "transmissive", "dirichlet"])
def test_uniform_state_stays_uniform_14(mmo, bc):
    W = np.array([0.7, 0.4, -0.3, 0.2, 0.8, 0.05, -0.02, 0.6, 0.03, 0.7, 0.05, -0.04, 0.02, 1.9])
    nx, ny = 9, 7
    W0 = np.broadcast_to(W[:, None, None], (14, ny, nx)).copy()
    t = {"periodic": wl.BC_PERIODIC, "transmissive": wl.BC_TRANSMISSIVE}.get(bc)
    bcs = [dict(type=t)] * 4 if t is not None else [dict(type=wl.BC_DIRICHLET, bands=[], default=W)] * 4
    s = mmo.Solver(14, nx, ny, extent=(0, 1, 0, 1), bcs=bcs,
                   collision=dict(model=wl.TAU_NONE))
    s.set_state_prim(W0)
    U0 = s.get_state()
    s.step(5, 0.4)
    U = s.get_state()
    for m in range(14):
        assert np.all(U[m] == U[m, 0, 0])
        # collisionless + uniform => nothing changes at all
        assert np.all(U[m] == U0[m])


def test_uniform_state_stays_uniform_5(mmo):
    W = np.array([0.7, 0.4, 0.8, 0.1, 3.2])
    W0 = np.broadcast_to(W[:, None, None], (5, 1, 11)).copy()
    s = mmo.Solver(5, 11, 1, bcs=[dict(type=wl.BC_TRANSMISSIVE)] * 4)
    s.set_state_prim(W0)
    U0 = s.get_state()
    s.step(5, 0.5)
    assert np.array_equal(s.get_state(), U0)


# ------------------------------------------------------------------------ conservation
@pytest.mark.parametrize("limiter,shared,flux", [(wl.LIM_MINMOD, 0, wl.FLUX_HLL),
                                                 (wl.LIM_VANALBADA, 1, wl.FLUX_RUSANOV)])
def test_periodic_conservation_14(mmo, limiter, shared, flux):
    prob = wl.random_smooth14(24, 16, limiter=limiter, shared_limiter=shared, flux=flux)
    s = oracle_solver(mmo, prob)
    U0 = s.get_state()
    s.step(10, 0.4)
    U1 = s.get_state()
    assert not np.allclose(U0, U1, rtol=1e-3, atol=0)           # something happened
    for m in range(14):
        scale = np.abs(U0[m]).sum()
        assert abs(U1[m].sum() - U0[m].sum()) <= 2e-14 * scale, m
    # with collisions: mass, momentum, energy (trace of U_ij)
    prob = wl.random_smooth14(24, 16, Kn=0.05, limiter=limiter, shared_limiter=shared, flux=flux)
    s = oracle_solver(mmo, prob)
    U0 = s.get_state()
    s.step(10, 0.4)
    U1 = s.get_state()
    E0 = U0[4] + U0[7] + U0[9]; E1 = U1[4] + U1[7] + U1[9]
    for a, b in [(U0[0], U1[0]), (U0[1], U1[1]), (U0[2], U1[2]), (U0[3], U1[3]), (E0, E1)]:
        assert abs(b.sum() - a.sum()) <= 2e-14 * np.abs(a).sum()
    # ... and the non-conserved ones do change through the source
    assert abs(U1[13].sum() - U0[13].sum()) > 1e-8 * np.abs(U0[13]).sum()


def test_periodic_conservation_5(mmo):
    prob = wl.random_smooth5(64)
    s = oracle_solver(mmo, prob)
    U0 = s.get_state(); s.step(20, 0.5); U1 = s.get_state()
    for m in range(5):
        assert abs(U1[m].sum() - U0[m].sum()) <= 2e-14 * np.abs(U0[m]).sum()
    prob = wl.random_smooth5(64, Kn=0.05)
    s = oracle_solver(mmo, prob)
    U0 = s.get_state(); s.step(20, 0.5); U1 = s.get_state()
    for m in range(3):
        assert abs(U1[m].sum() - U0[m].sum()) <= 2e-14 * np.abs(U0[m]).sum()
    assert abs(U1[4].sum() - U0[4].sum()) > 1e-8 * np.abs(U0[4]).sum()


# ---------------------------------------------------------------------------- symmetry
# x <-> y swap of the 14 primitives / conserved moments (u, P, q components)
SWAP_XY = [0, 2, 1, 3, 7, 5, 8, 4, 6, 9, 11, 10, 12, 13]


def test_transpose_symmetry(mmo):
    prob = wl.random_smooth14(12, 12, Kn=0.1)
    sA = oracle_solver(mmo, prob)
    WT = prob["W0"][SWAP_XY].transpose(0, 2, 1).copy()
    probT = dict(prob, W0=WT)
    sB = oracle_solver(mmo, probT)
    sA.step_fixed_dt(6, 2e-3); sB.step_fixed_dt(6, 2e-3)
    UA = sA.get_state(); UB = sB.get_state()[SWAP_XY].transpose(0, 2, 1)
    scale = np.abs(UA).max(axis=(1, 2), keepdims=True)
    assert np.max(np.abs(UA - UB) / scale) < 1e-13


def test_y_uniform_rows_identical(mmo):
    prob = wl.sod14(64, 4, Kn=0.01)
    s = oracle_solver(mmo, prob)
    s.step(20, 0.5)
    U = s.get_state()
    for j in range(1, 4):
        assert np.array_equal(U[:, j], U[:, 0])
    # z-odd and y-odd moments stay exactly zero
    for m in (2, 3, 5, 6, 8, 11, 12):
        assert np.all(U[m] == 0.0)


# -------------------------------------------------------------------------- relaxation
def test_uniform_relaxation_is_geometric(mmo):
    W = np.array([0.7, 0.4, -0.3, 0.2, 0.8, 0.05, -0.02, 0.6, 0.03, 0.7, 0.05, -0.04, 0.02, 1.9])
    nx, ny = 5, 4
    W0 = np.broadcast_to(W[:, None, None], (14, ny, nx)).copy()
    tau, dt, n = 0.05, 0.004, 25
    s = mmo.Solver(14, nx, ny, bcs=[dict(type=wl.BC_PERIODIC)] * 4,
                   collision=dict(model=wl.TAU_CONST, tau=tau))
    s.set_state_prim(W0)
    U0 = s.get_state()[:, 0, 0]
    s.step_fixed_dt(n, dt)
    Un = s.get_state()[:, 0, 0]
    # equilibrium: same rho, u, hydrostatic P; Maxwellian moments (L73)
    P = (W[4] + W[7] + W[9]) / 3
    Weq = wl.maxwellian(14, W[0], W[1:4], P / W[0])
    se = mmo.Solver(14, 1, 1, bcs=[dict(type=wl.BC_PERIODIC)] * 4)
    se.set_state_prim(Weq.reshape(14, 1, 1))
    Ueq = se.get_state()[:, 0, 0]
    expect = Ueq + (U0 - Ueq) * (1 - dt / tau) ** n
    assert np.allclose(Un, expect, rtol=1e-12, atol=1e-13)
    assert np.abs(U0 - Ueq).max() > 0.05

    W5 = np.array([0.7, 0.4, 0.8, 0.1, 3.2])
    s = mmo.Solver(5, 4, 1, bcs=[dict(type=wl.BC_PERIODIC)] * 4,
                   collision=dict(model=wl.TAU_CONST, tau=tau))
    s.set_state_prim(np.broadcast_to(W5[:, None, None], (5, 1, 4)).copy())
    U0 = s.get_state()[:, 0, 0]
    s.step_fixed_dt(n, dt)
    Un = s.get_state()[:, 0, 0]
    Ueq = mmo.prim2cons(wl.maxwellian(5, W5[0], W5[1], W5[2] / W5[0]))
    assert np.allclose(Un, Ueq + (U0 - Ueq) * (1 - dt / tau) ** n, rtol=1e-12, atol=1e-13)


# ------------------------------------------------- one first-order step, textbook assembly
def test_first_order_step_is_textbook_fv_update(mmo):
    """LIM_NONE => piecewise-constant states, so every interface flux is the (pinned) pointwise
    numerical flux of the two adjacent cell states; the step is U - dt/dx dF - dt/dy dG + dt C
    (PAPER.md L250).  Assembled here in numpy with periodic wrap-around by np.roll."""
    prob = wl.random_smooth14(6, 5, Kn=0.2, limiter=wl.LIM_NONE)
    s = oracle_solver(mmo, prob)
    nx, ny = 6, 5
    dx, dy = 1.0 / nx, (ny / nx) / ny
    W0 = prob["W0"]
    U0 = s.get_state()
    dt = 1.3e-3
    s.step_fixed_dt(1, dt)
    U1 = s.get_state()

    def hat(WL, WR, d):
        FL, FR = mmo.flux14(WL, d, 1e-4), mmo.flux14(WR, d, 1e-4)
        a, b = mmo.wavespeed14(WL, d, 1e-4), mmo.wavespeed14(WR, d, 1e-4)
        return mmo.numflux(wl.FLUX_HLL, FL, FR, mmo.prim2cons(WL), mmo.prim2cons(WR), a[0], a[1], b[0], b[1])

    exp = np.empty_like(U0)
    for j in range(ny):
        for i in range(nx):
            Wc = W0[:, j, i]
            Fe = hat(Wc, W0[:, j, (i + 1) % nx], 0); Fw = hat(W0[:, j, (i - 1) % nx], Wc, 0)
            Gn = hat(Wc, W0[:, (j + 1) % ny, i], 1); Gs = hat(W0[:, (j - 1) % ny, i], Wc, 1)
            Ph = (Wc[4] + Wc[7] + Wc[9]) / 3
            tau = mmo.tau(wl.TAU_KN, 0.0, 0.2, 1.0, 1.0, Wc[0], Ph)
            exp[:, j, i] = U0[:, j, i] - dt / dx * (Fe - Fw) - dt / dy * (Gn - Gs) + dt * mmo.source14(Wc, tau)
    scale = np.abs(U0).max(axis=(1, 2), keepdims=True)
    assert np.max(np.abs(U1 - exp) / scale) < 1e-14


def test_second_order_reproduces_linear_data_and_bands(mmo):
    """MUSCL with either limiter reconstructs linear data exactly (psi = 1), so for a state
    that is linear in x the interface states are W_i +- slope/2 on both sides, i.e. continuous:
    the interface flux is then the physical flux of that state (HLL consistency) and the
    update is a pure central difference of F.  Checked on the density flux: d rho/dt = -d(rho u)/dx."""
    nx, ny = 16, 3
    x = (np.arange(nx) + 0.5) / nx
    W0 = wl.maxwellian(14, np.broadcast_to(1.0 + 0.2 * x, (ny, nx)), (0.5, 0.0, 0.0), 1.0)
    for lim in (wl.LIM_MINMOD, wl.LIM_VANALBADA):
        s = mmo.Solver(14, nx, ny, extent=(0, 1, 0, ny / nx), limiter=lim,
                       bcs=[dict(type=wl.BC_TRANSMISSIVE)] * 2 + [dict(type=wl.BC_PERIODIC)] * 2)
        s.set_state_prim(W0)
        U0 = s.get_state(); dt = 1e-3
        s.step_fixed_dt(1, dt)
        U1 = s.get_state()
        drho = (U1[0] - U0[0])[:, 2:-2] / dt
        assert np.allclose(drho, -0.5 * 0.2, rtol=0, atol=1e-11)


def test_dirichlet_bands_select_by_cell_centre(mmo):
    """Inflow bands (L426): after one step only the first interior column next to a band feels
    the jet state; rows outside the bands next to the background-valued ghost stay untouched."""
    prob = wl.crossed_jets(20, Kn=None)
    s = oracle_solver(mmo, prob)
    U0 = s.get_state()
    s.step(1, 0.4)
    U1 = s.get_state()
    yc = (np.arange(20) + 0.5) / 20
    in_band = ((yc >= 0.3) & (yc <= 0.4)) | ((yc >= 0.6) & (yc <= 0.7))
    changed = np.any(U1[:, :, 0] != U0[:, :, 0], axis=0)
    assert np.array_equal(changed, in_band)
    assert np.all(U1[:, :, 2:] == U0[:, :, 2:])
    # lower jet carries +y momentum, upper jet -y momentum
    lo = np.where((yc >= 0.3) & (yc <= 0.4))[0]; hi = np.where((yc >= 0.6) & (yc <= 0.7))[0]
    assert np.all(U1[2, lo, 0] > 0) and np.all(U1[2, hi, 0] < 0)


def test_advance_to_and_info(mmo):
    prob = wl.sod5(100, Kn=0.01)
    s = oracle_solver(mmo, prob)
    dt0 = s.cfl_dt(0.5)
    # equilibrium 5-moment wave speed sqrt(5+sqrt(10)) c at sigma_lim -> dt = cfl dx / that (L434)
    assert dt0 == pytest.approx(0.5 * 0.01 / 2.856970013872806, rel=5e-3)
    s.advance_to(0.05, 0.5)
    inf = s.info()
    assert inf["t"] == 0.05 and inf["steps"] > 10 and 0 < inf["last_dt"] <= dt0 * 1.0001


# ------------------------------------------------------------- Sod -> exact Euler (physics)
EULER = {  # p*, u*, rho*_L, rho*_R, shock speed, fan head, fan tail
    3.0: (0.272909467286, 0.60856697289, 0.648643694382, 0.170703638658, 2.27300494425,
          -1.73205080757, -0.514916861788),
    5.0 / 3.0: (0.293945187666, 0.841194852169, 0.479689058721, 0.229805749312, 1.84447336705,
                -1.29099444874, -0.169401312511),
}


def exact_sod_density(x, t, gamma):
    ps, us, rL, rR, ss, head, tail = EULER[gamma]
    xi = (x - 0.5) / t
    aL = math.sqrt(gamma * 1.0 / 1.0)
    rho = np.where(xi < head, 1.0, 0.0)
    fan = (xi >= head) & (xi < tail)
    # left rarefaction: u - a = xi, u + 2a/(g-1) = 2aL/(g-1)
    a = (2 * aL / (gamma - 1) - xi) * (gamma - 1) / (gamma + 1)
    rho = np.where(fan, (a / aL) ** (2 / (gamma - 1)), rho)
    rho = np.where((xi >= tail) & (xi < us), rL, rho)
    rho = np.where((xi >= us) & (xi < ss), rR, rho)
    rho = np.where(xi >= ss, 0.125, rho)
    return rho


def test_exact_riemann_table_is_self_consistent():
    """The tabulated star states satisfy the Rankine-Hugoniot and isentropic relations."""
    for g, (ps, us, rL, rR, ss, head, tail) in EULER.items():
        assert rL == pytest.approx(ps ** (1 / g), rel=1e-9)
        assert 0.125 * ss == pytest.approx(rR * (ss - us), rel=1e-9)            # mass across shock
        assert ps - 0.1 == pytest.approx(0.125 * ss * us, rel=1e-9)             # momentum
        assert head == pytest.approx(-math.sqrt(g), rel=1e-9)
        assert tail == pytest.approx(us - math.sqrt(g * ps / rL), rel=1e-9)


def test_sod5_approaches_euler_gamma3(mmo):
    nx = 400
    x = (np.arange(nx) + 0.5) / nx
    ref = exact_sod_density(x, 0.2, 3.0)
    errs = []
    for Kn in (0.1, 0.01, 0.001):
        s = oracle_solver(mmo, wl.sod5(nx, Kn=Kn))
        s.advance_to(0.2, 0.5)
        errs.append(np.abs(s.get_state()[0, 0] - ref).mean())
    assert errs[0] > errs[1] > errs[2]
    assert errs[2] < 0.02 and errs[0] > 2.0 * errs[2]


def test_sod14_approaches_euler_gamma53(mmo):
    nx = 200
    x = (np.arange(nx) + 0.5) / nx
    ref = exact_sod_density(x, 0.2, 5.0 / 3.0)
    errs = []
    for Kn in (0.1, 0.01, 0.001):
        s = oracle_solver(mmo, wl.sod14(nx, 2, Kn=Kn))
        s.advance_to(0.2, 0.5)
        U = s.get_state()
        errs.append(np.abs(U[0, 0] - ref).mean())
    assert errs[0] > errs[1] > errs[2]
    assert errs[2] < 0.02 and errs[0] > 2.0 * errs[2]


def test_C1_roundoff_sensitivity(mmo):
    """BASELINE config 1 (5-moment Sod, Kn = 0.01, minmod + HLL, CFL 0.5) amplifies round-off:
    two ORACLE runs whose initial densities differ by a few 1e-15 relative drift apart by many
    orders of magnitude within 300 CFL steps, while the density profile stays close.  This is a
    property of the scheme at sigma -> sigma_lim (closure terms ~ 1/sigma_bar^2, L157-163), not of
    any implementation; it is why the GPU parity test for the whole run to t = 0.2 compares the
    density profile and the step count rather than every moment (R24)."""
    prob = wl.sod5(1000, Kn=0.01)
    a = oracle_solver(mmo, prob)
    W1 = prob["W0"].copy()
    W1[0, 0, 400:600] *= 1.0 + 1e-15 * (np.arange(200) % 3)
    b = oracle_solver(mmo, dict(prob, W0=W1))
    a.step(100, 0.5); b.step(100, 0.5)
    e100 = np.abs(a.get_state() - b.get_state()).max()
    assert e100 < 1e-8                       # still a round-off sized difference
    a.step(200, 0.5); b.step(200, 0.5)
    Ua, Ub = a.get_state(), b.get_state()
    rel = np.abs(Ua - Ub).max(axis=(1, 2)) / np.abs(Ua).max(axis=(1, 2))
    assert rel.max() > 1e-4                  # grown by > 1e10 from the 1e-15 seed
    assert np.abs(Ua[0] - Ub[0]).mean() < 1e-3 * np.abs(Ua[0]).mean()


# ------------------------- point-implicit source (L348), midpoint scheme (L250)
def _uniform_noneq(mmo, **opt):
    W = np.array([0.7, 0.4, -0.3, 0.2, 0.8, 0.05, -0.02, 0.6, 0.03, 0.7, 0.05, -0.04, 0.02, 1.9])
    W0 = np.broadcast_to(W[:, None, None], (14, 4, 5)).copy()
    tau = 0.05
    s = mmo.Solver(14, 5, 4, bcs=[dict(type=wl.BC_PERIODIC)] * 4,
                   collision=dict(model=wl.TAU_CONST, tau=tau), **opt)
    s.set_state_prim(W0)
    P = (W[4] + W[7] + W[9]) / 3
    Ueq = mmo.prim2cons(wl.maxwellian(14, W[0], W[1:4], P / W[0]))
    return s, s.get_state()[:, 0, 0].copy(), Ueq, tau


def test_point_implicit_source_is_backward_euler(mmo):
    """Uniform non-equilibrium gas, constant tau (no fluxes act): backward Euler on the linear BGK
    relaxation gives U_eq + (U_0 - U_eq)/(1 + dt/tau)^n exactly, for ANY dt/tau; an enormous dt/tau
    lands on the Maxwellian; rho, rho u and tr U_ij never change."""
    for dt, n in ((0.004, 25), (0.5, 3), (5e4, 1)):
        s, U0, Ueq, tau = _uniform_noneq(mmo, source_scheme=wl.SRC_POINT_IMPLICIT)
        s.step_fixed_dt(n, dt)
        Un = s.get_state()
        assert np.allclose(Un[:, 0, 0], Ueq + (U0 - Ueq) / (1 + dt / tau) ** n, rtol=1e-12, atol=1e-13)
        assert np.all(Un == Un[:, :1, :1])                                   # still uniform
        for m in (0, 1, 2, 3):
            assert Un[m, 0, 0] == pytest.approx(U0[m], rel=1e-14)
        assert Un[4, 0, 0] + Un[7, 0, 0] + Un[9, 0, 0] == pytest.approx(U0[4] + U0[7] + U0[9], rel=1e-14)
    assert np.allclose(Un[:, 0, 0], Ueq, rtol=1e-5)                          # dt/tau = 1e6: equilibrium


def test_point_implicit_agrees_with_explicit_to_second_order_in_dt_over_tau(mmo):
    diffs = []
    for dt in (0.004, 0.002, 0.001):
        a, *_ = _uniform_noneq(mmo)
        b, *_ = _uniform_noneq(mmo, source_scheme=wl.SRC_POINT_IMPLICIT)
        a.step_fixed_dt(1, dt); b.step_fixed_dt(1, dt)
        diffs.append(np.abs(a.get_state() - b.get_state()).max())
    assert 3.5 < diffs[0] / diffs[1] < 4.5 and 3.5 < diffs[1] / diffs[2] < 4.5


def test_point_implicit_sod_is_stable_where_explicit_is_not(mmo):
    """near Kn = 1e-4 the explicit BGK source sets the time-step limit and "a simple
    point-implicit treatment of the source terms is sufficient".  At Kn = 1e-5 the CFL time step is
    ~30 tau: the explicit scheme blows up, the point-implicit one gives the Euler (gamma = 3) solution."""
    nx = 400
    x = (np.arange(nx) + 0.5) / nx
    ref = exact_sod_density(x, 0.2, 3.0)
    prob = wl.sod5(nx, Kn=1e-5)
    s = oracle_solver(mmo, prob, source_scheme=wl.SRC_POINT_IMPLICIT)
    s.advance_to(0.2, 0.5)
    rho = s.get_state()[0, 0]
    assert np.all(np.isfinite(rho)) and rho.min() > 0
    err_implicit = np.abs(rho - ref).mean()
    assert err_implicit < 0.01
    e = oracle_solver(mmo, prob)
    try:
        e.advance_to(0.2, 0.5)
        Ue = e.get_state()
        # the explicit source oscillates (limiter and sigma clamps keep it bounded) or blows up
        assert (not np.all(np.isfinite(Ue))) or np.abs(Ue[0, 0] - ref).mean() > 3.0 * err_implicit
    except RuntimeError:
        pass                                                                 # non-finite CFL rate


def test_midpoint_uniform_relaxation_has_the_rk2_amplification_factor(mmo):
    """No fluxes act on a uniform state, U_eq is invariant: midpoint (L250) multiplies U - U_eq by
    1 - x + x^2/2 per step (x = dt/tau), forward Euler by 1 - x."""
    dt, n = 0.004, 25
    s, U0, Ueq, tau = _uniform_noneq(mmo, time_scheme=wl.TIME_MIDPOINT)
    s.step_fixed_dt(n, dt)
    x = dt / tau
    assert np.allclose(s.get_state()[:, 0, 0], Ueq + (U0 - Ueq) * (1 - x + 0.5 * x * x) ** n, rtol=1e-12, atol=1e-13)
    with pytest.raises(ValueError):                                         # midpoint needs the explicit source
        mmo.Solver(14, 4, 4, time_scheme=wl.TIME_MIDPOINT, source_scheme=wl.SRC_POINT_IMPLICIT)


def test_midpoint_is_second_order_in_time(mmo):
    """Smooth periodic problem on a fixed grid: against a run with dt/16 the error of the midpoint
    scheme falls 4x per halving of dt, that of forward Euler 2x; conserved totals stay conserved."""
    # first order in space (no limiter): the spatial operator is then smooth in the state and the
    # asymptotic temporal orders show cleanly
    prob = wl.random_smooth14(24, 12, Kn=0.1, amp=0.1, limiter=wl.LIM_NONE)
    T, dt0 = 0.01, 0.0005
    def run(scheme, dt):
        s = oracle_solver(mmo, prob, time_scheme=scheme)
        s.step_fixed_dt(int(round(T / dt)), dt)
        return s.get_state()
    ref = run(wl.TIME_MIDPOINT, dt0 / 16)
    em = [np.abs(run(wl.TIME_MIDPOINT, dt) - ref).max() for dt in (dt0, dt0 / 2, dt0 / 4)]
    ee = [np.abs(run(wl.TIME_EULER, dt) - ref).max() for dt in (dt0, dt0 / 2, dt0 / 4)]
    assert 3.3 < em[0] / em[1] < 4.8 and 3.3 < em[1] / em[2] < 4.8
    assert 1.7 < ee[0] / ee[1] < 2.3 and 1.7 < ee[1] / ee[2] < 2.3
    assert em[0] < 0.1 * ee[0]
    U0 = oracle_solver(mmo, prob).get_state()
    for m in (0, 1, 2, 3):
        assert ref[m].sum() == pytest.approx(U0[m].sum(), rel=1e-12, abs=1e-12)


# ------------------------------------------------- MUSCL face states, shared limiter (L262-266)
# Hand-computed three-cell examples.  Every expected face value below is typed from the paper's
# definition (L262: slope = psi (dm + dp)/2 with the symmetric limiter function; L266: "the same,
# most stringent value of the limiter" for all primitive variables), not from the oracle.
#   variable      Wm     W0     Wp      dm      dp     psi_minmod = 2 min/(|dm|+|dp|)   psi_vanAlbada = 2 dm dp/(dm^2+dp^2)
#   a            1.0    2.0    4.0     1.0     2.0     2/3                               4/5
#   b (flat)     0.0    0.0    0.0     0       0       imposes nothing (reading R14)
#   c            2.0    2.5    2.625   0.5     0.125   2*0.125/0.625 = 2/5               0.125/0.265625 = 8/17
#   d            0.4    0.5    0.6     0.1     0.1     1                                 1
#   e            1.0    2.0    3.0     1.0     1.0     1                                 1
FS_WM = [1.0, 0.0, 2.0, 0.4, 1.0]
FS_W0 = [2.0, 0.0, 2.5, 0.5, 2.0]
FS_WP = [4.0, 0.0, 2.625, 0.6, 3.0]
FS_CENTRAL = [1.5, 0.0, 0.3125, 0.1, 1.0]          # (dm + dp)/2


def test_face_states_shared_limiter_named_variable_sets_psi(mmo):
    """Variable c is the most stringent one: psi = 2/5 (minmod) resp. 8/17 (van Albada) multiplies
    the central slope of EVERY variable; the exactly flat variable b is skipped -- without the
    skip rule its psi(0, 0) = 0 would flatten everything."""
    for lim, psi in ((1, 2.0 / 5.0), (2, 8.0 / 17.0)):
        lo, hi = mmo.face_states(lim, True, FS_WM, FS_W0, FS_WP)
        for k in range(5):
            half = 0.5 * psi * FS_CENTRAL[k]
            assert lo[k] == pytest.approx(FS_W0[k] - half, rel=1e-15, abs=1e-16)
            assert hi[k] == pytest.approx(FS_W0[k] + half, rel=1e-15, abs=1e-16)
    # spelled out for minmod: psi = 0.4 -> half slopes 0.3, 0, 0.0625, 0.02, 0.2
    lo, hi = mmo.face_states(1, True, FS_WM, FS_W0, FS_WP)
    np.testing.assert_allclose(lo, [1.7, 0.0, 2.4375, 0.48, 1.8], rtol=1e-15, atol=0)
    np.testing.assert_allclose(hi, [2.3, 0.0, 2.5625, 0.52, 2.2], rtol=1e-15, atol=0)


def test_face_states_per_variable_limiter_differs(mmo):
    """Per-variable mode on the same cells: each variable takes its own psi (minmod: the smaller
    difference), so a = 2 -/+ 0.5, c = 2.5 -/+ 0.0625, d and e keep their full central slope."""
    lo, hi = mmo.face_states(1, False, FS_WM, FS_W0, FS_WP)
    np.testing.assert_allclose(lo, [1.5, 0.0, 2.4375, 0.45, 1.5], rtol=1e-15, atol=0)
    np.testing.assert_allclose(hi, [2.5, 0.0, 2.5625, 0.55, 2.5], rtol=1e-15, atol=0)
    lo, hi = mmo.face_states(2, False, FS_WM, FS_W0, FS_WP)           # van Albada: psi_k * central
    np.testing.assert_allclose(hi - np.array(FS_W0), 0.5 * np.array([0.8, 0, 8 / 17, 1, 1]) * np.array(FS_CENTRAL),
                               rtol=1e-14, atol=0)


def test_face_states_shared_limiter_extremum_and_one_sided_flat(mmo):
    """An extremum in ONE variable (dm dp < 0) gives psi = 0 for all of them (first order in that
    cell); so does a variable that is flat on one side only (dm = 0, dp != 0: dm dp = 0 is not
    > 0) -- only dm = dp = 0 exactly is exempt."""
    for lim in (1, 2):
        Wp = list(FS_WP); Wp[4] = 1.5                  # e: 1, 2, 1.5 -> local maximum
        lo, hi = mmo.face_states(lim, True, FS_WM, FS_W0, Wp)
        assert np.array_equal(lo, np.array(FS_W0)) and np.array_equal(hi, np.array(FS_W0))
        Wm = list(FS_WM); Wm[3] = 0.5                  # d: 0.5, 0.5, 0.6 -> dm = 0, dp = 0.1
        lo, hi = mmo.face_states(lim, True, Wm, FS_W0, FS_WP)
        assert np.array_equal(lo, np.array(FS_W0)) and np.array_equal(hi, np.array(FS_W0))
    # limiter off: zero slopes whatever the flag
    lo, hi = mmo.face_states(0, True, FS_WM, FS_W0, FS_WP)
    assert np.array_equal(lo, np.array(FS_W0)) and np.array_equal(hi, np.array(FS_W0))


def test_face_states_shared_limiter_is_what_the_step_uses(mmo):
    """The exported routine is the one inside the time step: one first-order-in-time step of a 1-D
    5-moment problem with the shared limiter equals the update assembled here from face_states +
    the pointwise flux / wave-speed / HLL functions (each pinned on its own)."""
    rng = np.random.default_rng(11)
    nx = 12
    x = (np.arange(nx) + 0.5) / nx
    W = np.stack([1 + 0.3 * np.sin(2 * np.pi * x), 0.2 * np.cos(2 * np.pi * x), 0.8 + 0.2 * np.sin(4 * np.pi * x),
                  0.05 * np.sin(2 * np.pi * x + 1), 2.2 + 0.3 * np.cos(2 * np.pi * x)])
    s = mmo.Solver(5, nx, 1, bcs=[dict(type=wl.BC_PERIODIC)] * 4, collision=dict(model=wl.TAU_NONE),
                   limiter=wl.LIM_MINMOD, shared_limiter=1, flux=wl.FLUX_HLL)
    s.set_state_prim(W[:, None, :])
    U0 = s.get_state()[:, 0, :]
    dt = 1e-3
    s.step_fixed_dt(1, dt)
    U1 = s.get_state()[:, 0, :]
    lo = np.empty((5, nx)); hi = np.empty((5, nx))
    for i in range(nx):
        lo[:, i], hi[:, i] = mmo.face_states(wl.LIM_MINMOD, True, W[:, i - 1], W[:, i], W[:, (i + 1) % nx])
    F = np.empty((5, nx))                               # F[:, i]: interface between cells i-1 and i
    for i in range(nx):
        WL, WR = hi[:, i - 1], lo[:, i]
        a = mmo.wavespeed5(WL, 1e-4); b = mmo.wavespeed5(WR, 1e-4)
        F[:, i] = mmo.numflux(wl.FLUX_HLL, mmo.flux5(WL, 1e-4), mmo.flux5(WR, 1e-4),
                              mmo.prim2cons(WL), mmo.prim2cons(WR), a[0], a[1], b[0], b[1])
    expect = U0 - dt * nx * (np.roll(F, -1, axis=1) - F)
    np.testing.assert_allclose(U1, expect, rtol=1e-13, atol=1e-15)


# ------------------------------------------------- 2-D CFL rate (section 6.1, Fig 14; reading R13)
LAMBDA_EQ = 2.18259874765634      # Eq 29 at equilibrium, sigma_bar = 1e-4 (mpmath; SURVEY.md section 8(c), row "wave speeds")


@pytest.mark.parametrize("u, winner", [((0.3, 0.1), "y"), ((6.0, 0.1), "x"), ((-6.0, 0.1), "x"), ((0.3, -2.0), "y")])
def test_cfl_dt_2d_anisotropic_cells(mmo, u, winner):
    """dt = cfl / max over cells of max(s_x/dx, s_y/dy) with s_d = |u_d| + lambda* c for a uniform Maxwellian
    (q = 0: the two speeds of Eq 29 are u_d +- lambda* c), on cells with dx = 2 dy: a scheme that divides both
    directions by dx, takes the minimum, or forgets a direction gives another number in one of the cases."""
    rho, T = 0.7, 1.3
    c = math.sqrt(T)
    nx, ny = 8, 6
    W = wl.maxwellian(wl.SYS14, np.full((ny, nx), rho), (u[0], u[1], 0.0), T)
    dx, dy = 2.0 / nx, 0.75 / ny
    assert dx == 2.0 * dy
    s = mmo.Solver(14, nx, ny, extent=(0.0, 2.0, 0.0, 0.75), collision=dict(model=wl.TAU_NONE),
                   bcs=[dict(type=wl.BC_PERIODIC)] * 4, sigma_lim=1e-4)
    s.set_state_prim(W)
    rx, ry = (abs(u[0]) + LAMBDA_EQ * c) / dx, (abs(u[1]) + LAMBDA_EQ * c) / dy
    assert (rx > ry) == (winner == "x") and abs(rx - ry) > 0.1 * max(rx, ry)
    for cfl in (0.5, 0.4):
        assert s.cfl_dt(cfl) == pytest.approx(cfl / max(rx, ry), rel=1e-12)
    # the step taken by step(1, cfl) is that dt (L434: "imposing a Courant number of 0.5")
    s.step(1, 0.5)
    assert s.info()["last_dt"] == pytest.approx(0.5 / max(rx, ry), rel=1e-12)


def test_cfl_dt_is_set_by_a_dirichlet_ghost_state(mmo):
    """Reading R13: ghost cells take part in the CFL maximum.  Gas at rest (rho = T = 1) on 20 x 20 unit-square cells,
    dx = dy = 0.05; one Dirichlet band on the left side holds a Maxwellian moving at u_x = 5.  Interior cells alone
    would give dt = 0.4 * 0.05 / 2.18259874765634 = 9.1634e-3; with the ghost state the fastest cell has
    s_x = 5 + 2.18259874765634, so dt = 0.4 * 0.05 / 7.18259874765634 = 2.7845075e-3."""
    n = 20
    rest = wl.maxwellian(wl.SYS14, 1.0, (0.0, 0.0, 0.0), 1.0)
    fast = wl.maxwellian(wl.SYS14, 1.0, (5.0, 0.0, 0.0), 1.0)
    bcs = [dict(type=wl.BC_DIRICHLET, bands=[(0.3, 0.4, fast)], default=rest),
           dict(type=wl.BC_TRANSMISSIVE), dict(type=wl.BC_TRANSMISSIVE), dict(type=wl.BC_TRANSMISSIVE)]
    s = mmo.Solver(14, n, n, extent=(0.0, 1.0, 0.0, 1.0), collision=dict(model=wl.TAU_NONE), bcs=bcs, sigma_lim=1e-4)
    s.set_state_prim(wl.maxwellian(wl.SYS14, np.ones((n, n)), (0.0, 0.0, 0.0), 1.0))
    assert s.cfl_dt(0.4) == pytest.approx(2.784507488536227e-3, rel=1e-12)
    # without a band in reach of any cell centre the interior value is back
    bcs[0] = dict(type=wl.BC_DIRICHLET, bands=[(0.33, 0.37, fast)], default=rest)     # cell centres 0.325, 0.375: none inside
    s2 = mmo.Solver(14, n, n, extent=(0.0, 1.0, 0.0, 1.0), collision=dict(model=wl.TAU_NONE), bcs=bcs, sigma_lim=1e-4)
    s2.set_state_prim(wl.maxwellian(wl.SYS14, np.ones((n, n)), (0.0, 0.0, 0.0), 1.0))
    assert s2.cfl_dt(0.4) == pytest.approx(9.163388378865272e-3, rel=1e-12)
