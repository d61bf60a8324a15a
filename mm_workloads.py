"""Seeded synthetic inputs for the moment-method time step (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic: it only describes problems (grid, collision
model, boundary tables, options) and fills arrays of *primitive* states
W = (rho | u_x u_y u_z | P_xx P_xy P_xz P_yy P_yz P_zz | q_x q_y q_z | R)   (14-moment)
W = (rho, u, P, q, r)                                                       (5-moment)
with Maxwellian values (P_ij = rho T delta_ij, q = 0, R = 15 P^2/rho resp. r = 3 P^2/rho,
PAPER.md L73, L127).  Each implementation (oracle/, the CUDA library) converts primitives to
conserved moments with its own code.

The workloads stand in for the paper's Sod tube and crossing-jet cases
(L426, L474); they are the synthetic variants BASELINE.json asks for.
Plain-int constants mirror the enums of include/mm.h and oracle/mmo.h (same numbering).
"""
from __future__ import annotations

import math

import numpy as np

SYS5, SYS14 = 5, 14
TAU_NONE, TAU_CONST, TAU_KN = 0, 1, 2
BC_TRANSMISSIVE, BC_PERIODIC, BC_DIRICHLET = 0, 1, 2
LIM_NONE, LIM_MINMOD, LIM_VANALBADA = 0, 1, 2
FLUX_HLL, FLUX_RUSANOV = 0, 1
SRC_EXPLICIT, SRC_POINT_IMPLICIT = 0, 1      # BGK source: forward Euler | point-implicit
TIME_EULER, TIME_MIDPOINT = 0, 1             # forward Euler | midpoint (2nd-order RK)

SEED = 240115233
_MASK = (1 << 64) - 1


def splitmix64(x: np.ndarray) -> np.ndarray:
    """Counter-based generator: the splitmix64 output function applied to uint64 counters."""
    x = x.astype(np.uint64)
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(n: int, seed: int = SEED, offset: int = 0) -> np.ndarray:
    """n doubles in [0,1): top 53 bits of splitmix64(counter XOR seed)."""
    ctr = np.arange(offset, offset + n, dtype=np.uint64) ^ np.uint64(seed & _MASK)
    return (splitmix64(ctr) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))


def maxwellian(system: int, rho, u=(0.0, 0.0, 0.0), T=1.0) -> np.ndarray:
    """Primitive Maxwellian state(s); rho may be an array (result [nm, ...])."""
    rho = np.asarray(rho, dtype=np.float64)
    P = rho * T
    z = np.zeros_like(rho)
    if system == SYS5:
        ux = u if np.isscalar(u) else u[0]
        return np.stack([rho, z + ux, P, z, 3.0 * P * P / rho])
    return np.stack([rho, z + u[0], z + u[1], z + u[2], P, z, z, P, z, P, z, z, z,
                     15.0 * P * P / rho])


def _problem(system, nx, ny, extent, collision, bcs, W0, **options):
    opt = dict(sigma_lim=1e-4, ws_scale=1.0, limiter=LIM_MINMOD, shared_limiter=0, flux=FLUX_HLL,
               source_scheme=SRC_EXPLICIT, time_scheme=TIME_EULER)
    opt.update(options)
    return dict(system=system, nx=nx, ny=ny, extent=extent, collision=collision, bcs=bcs,
                options=opt, W0=np.ascontiguousarray(W0, dtype=np.float64))


def sod5(nx: int = 1000, Kn: float = 0.01, **options):
    """C1: 5-moment Sod tube, (rho,u,p) = (1,0,1) | (0.125,0,0.1), diaphragm at 0.5."""
    xc = (np.arange(nx) + 0.5) / nx
    left = xc < 0.5
    rho = np.where(left, 1.0, 0.125)
    T = np.where(left, 1.0, 0.8)
    W0 = maxwellian(SYS5, rho, 0.0, T).reshape(5, 1, nx)
    col = dict(model=TAU_KN, Kn=Kn, L_ref=1.0, rho_ref=1.0) if Kn is not None else dict(model=TAU_NONE)
    bcs = [dict(type=BC_TRANSMISSIVE)] * 4
    return _problem(SYS5, nx, 1, (0.0, 1.0, 0.0, 1.0), col, bcs, W0, **options)


def sod14(nx: int = 4096, ny: int = 4, Kn: float = 0.01, **options):
    """C2: 14-moment Sod tube on nx x ny square cells, periodic in y."""
    xc = (np.arange(nx) + 0.5) / nx
    left = xc < 0.5
    rho = np.broadcast_to(np.where(left, 1.0, 0.125), (ny, nx))
    T = np.broadcast_to(np.where(left, 1.0, 0.8), (ny, nx))
    W0 = maxwellian(SYS14, rho, (0.0, 0.0, 0.0), T)
    col = dict(model=TAU_KN, Kn=Kn, L_ref=1.0, rho_ref=1.0) if Kn is not None else dict(model=TAU_NONE)
    bcs = [dict(type=BC_TRANSMISSIVE), dict(type=BC_TRANSMISSIVE),
           dict(type=BC_PERIODIC), dict(type=BC_PERIODIC)]
    return _problem(SYS14, nx, ny, (0.0, 1.0, 0.0, ny / nx), col, bcs, W0, **options)


def crossed_jets(n: int = 512, Kn: float = 1.0, perturb: float = 0.0, mach: float = 3.0,
                 angle_deg: float = 20.0, rho_bg: float = 1e-3, seed: int = SEED, **options):
    """C3-C5: two Mach-`mach` jets (rho = T = 1) entering through the left side in the bands
    y in [0.3,0.4] (+angle) and [0.6,0.7] (-angle) into a background rho_bg, T = 1; the rest of
    the left side is held at the background, the other sides are transmissive.  Speed uses
    a = sqrt(gamma R T) with gamma = 5/3.  `perturb` = relative amplitude of
    the uniform random density perturbation of the initial background (T = 1 kept, so P = rho).
    The limiter value is shared by all primitives unless overridden: with
    per-variable limiting this problem loses positivity within a few steps (R14)."""
    options.setdefault("shared_limiter", 1)
    speed = mach * math.sqrt(5.0 / 3.0)
    th = math.radians(angle_deg)
    jet_lo = maxwellian(SYS14, 1.0, (speed * math.cos(th), speed * math.sin(th), 0.0), 1.0)
    jet_hi = maxwellian(SYS14, 1.0, (speed * math.cos(th), -speed * math.sin(th), 0.0), 1.0)
    bg = maxwellian(SYS14, rho_bg, (0.0, 0.0, 0.0), 1.0)
    rho = np.full((n, n), rho_bg)
    if perturb:
        xi = 2.0 * uniform01(n * n, seed).reshape(n, n) - 1.0
        rho = rho * (1.0 + perturb * xi)
    W0 = maxwellian(SYS14, rho, (0.0, 0.0, 0.0), 1.0)
    col = dict(model=TAU_KN, Kn=Kn, L_ref=0.1, rho_ref=1.0) if Kn is not None else dict(model=TAU_NONE)
    bcs = [dict(type=BC_DIRICHLET, bands=[(0.3, 0.4, jet_lo), (0.6, 0.7, jet_hi)], default=bg),
           dict(type=BC_TRANSMISSIVE), dict(type=BC_TRANSMISSIVE), dict(type=BC_TRANSMISSIVE)]
    return _problem(SYS14, n, n, (0.0, 1.0, 0.0, 1.0), col, bcs, W0, **options)


def paper_jets(n: int = 1200, two: bool = True, Kn=None, mach: float = 5.0, rho_bg: float = 1e-5, **options):
    """The paper's own jet cases in its recommended robust configuration (
    SURVEY section 8(f) item 1), non-dimensional: unit square, jets of width L/7 centred on the
    left side (directed +x) and, if `two`, on the bottom side (directed +y, crossing at a right
    angle), rho_jet = T = 1, Mach `mach` with a = sqrt(5/3 R T), background rho_bg = 1e-5 held on
    the rest of those sides, the other sides transmissive; collisionless unless Kn is given
    (Kn based on the jet width, L474).  Rusanov flux (L258), van Albada limiter with one shared
    psi (L262-266), sigma_lim = 1e-4 (L442); the paper's Courant number is 0.5 (L434)."""
    options.setdefault("shared_limiter", 1)
    options.setdefault("limiter", LIM_VANALBADA)
    options.setdefault("flux", FLUX_RUSANOV)
    speed = mach * math.sqrt(5.0 / 3.0)
    lo, hi = 0.5 - 1.0 / 14.0, 0.5 + 1.0 / 14.0
    jet_x = maxwellian(SYS14, 1.0, (speed, 0.0, 0.0), 1.0)
    jet_y = maxwellian(SYS14, 1.0, (0.0, speed, 0.0), 1.0)
    bg = maxwellian(SYS14, rho_bg, (0.0, 0.0, 0.0), 1.0)
    W0 = maxwellian(SYS14, np.full((n, n), rho_bg), (0.0, 0.0, 0.0), 1.0)
    col = dict(model=TAU_KN, Kn=Kn, L_ref=1.0 / 7.0, rho_ref=1.0) if Kn is not None else dict(model=TAU_NONE)
    ylo = dict(type=BC_DIRICHLET, bands=[(lo, hi, jet_y)], default=bg) if two else dict(type=BC_TRANSMISSIVE)
    bcs = [dict(type=BC_DIRICHLET, bands=[(lo, hi, jet_x)], default=bg), dict(type=BC_TRANSMISSIVE),
           ylo, dict(type=BC_TRANSMISSIVE)]
    return _problem(SYS14, n, n, (0.0, 1.0, 0.0, 1.0), col, bcs, W0, **options)


def random_smooth14(nx: int, ny: int, seed: int = SEED, amp: float = 0.2, periodic: bool = True,
                    Kn=None, zsym: bool = False, **options):
    """Generic smooth, fully 3-D non-equilibrium test state on a periodic box: every one of the
    14 primitives varies (including the z-odd ones) so no component of the scheme is idle.
    zsym=True sets the z-odd primitives u_z, P_xz, P_yz, q_z to exactly zero (the symmetry every
    BASELINE config has) and leaves the other ten as they are."""
    x = (np.arange(nx) + 0.5) / nx
    y = (np.arange(ny) + 0.5) / ny
    X, Y = np.meshgrid(x, y)
    r = uniform01(64, seed)
    def wave(k):
        return (np.sin(2 * math.pi * (X + r[k])) * np.cos(2 * math.pi * (Y + r[k + 1]))
                + 0.5 * np.sin(4 * math.pi * (X - Y + r[k + 2])))
    rho = 1.0 + amp * wave(0)
    u = [0.5 * amp * wave(3 + 3 * i) + (0.3, -0.2, 0.1)[i] for i in range(3)]
    T = 1.0 + 0.5 * amp * wave(12)
    P = rho * T
    W0 = np.zeros((14, ny, nx))
    W0[0] = rho
    W0[1], W0[2], W0[3] = u
    W0[4] = P * (1.0 + 0.3 * amp * wave(15)); W0[7] = P * (1.0 + 0.3 * amp * wave(18))
    W0[9] = P * (1.0 + 0.3 * amp * wave(21))
    W0[5] = 0.2 * amp * P * wave(24); W0[6] = 0.2 * amp * P * wave(27); W0[8] = 0.2 * amp * P * wave(30)
    Ph = (W0[4] + W0[7] + W0[9]) / 3.0
    c3 = rho * (Ph / rho) ** 1.5
    W0[10] = 0.3 * amp * c3 * wave(33); W0[11] = 0.3 * amp * c3 * wave(36); W0[12] = 0.3 * amp * c3 * wave(39)
    W0[13] = 15.0 * Ph * Ph / rho * (1.0 + 0.3 * amp * wave(42))
    if zsym:
        W0[3] = 0.0; W0[6] = 0.0; W0[8] = 0.0; W0[12] = 0.0
    t = BC_PERIODIC if periodic else BC_TRANSMISSIVE
    bcs = [dict(type=t)] * 4
    col = dict(model=TAU_KN, Kn=Kn, L_ref=1.0, rho_ref=1.0) if Kn is not None else dict(model=TAU_NONE)
    return _problem(SYS14, nx, ny, (0.0, 1.0, 0.0, ny / nx), col, bcs, W0, **options)


def anisotropic14(nx: int, ny: int, axis: int = 0, ratio: float = 0.025, seed: int = SEED, amp: float = 0.1,
                  zsym: bool = False, Kn=None, **options):
    """Smooth periodic state whose pressure tensor is strongly anisotropic: the normal pressure along `axis`
    (0: P_xx, 1: P_yy) is `ratio` x the hydrostatic pressure, the other two share the rest, so that
    P_dd* = P_dd / P < 1/32 everywhere along that direction -- below the range a tabulated a(P*), b(P*) of
    Eq 29c-d would normally cover.  R_iijj is 1.3 x the fourth moment of the Gaussian with this pressure tensor,
    ((tr P)^2 + 2 P_ij P_ij) / rho, which keeps the state inside the realizability bound of Eq 19; everything
    else as random_smooth14."""
    prob = random_smooth14(nx, ny, seed=seed, amp=amp, zsym=zsym, Kn=Kn, **options)
    W0 = prob["W0"]
    rho = W0[0]
    Ph = (W0[4] + W0[7] + W0[9]) / 3.0
    diag = (4, 7, 9)
    small = diag[axis]
    shape = W0[small] / Ph                              # 1 + a few percent, smooth
    for m in diag:
        W0[m] = Ph * (ratio * shape if m == small else 0.5 * (3.0 - ratio * shape))
    W0[5] *= 0.2; W0[6] *= 0.2; W0[8] *= 0.2            # keep P positive definite next to the small eigenvalue
    W0[10] *= 0.3; W0[11] *= 0.3; W0[12] *= 0.3
    trP = W0[4] + W0[7] + W0[9]
    PP = W0[4] ** 2 + W0[7] ** 2 + W0[9] ** 2 + 2.0 * (W0[5] ** 2 + W0[6] ** 2 + W0[8] ** 2)
    W0[13] = 1.3 * (trP * trP + 2.0 * PP) / rho
    return prob


def random_smooth5(nx: int, seed: int = SEED, amp: float = 0.2, periodic: bool = True, Kn=None,
                   **options):
    """Smooth non-equilibrium 5-moment state on a periodic interval."""
    x = (np.arange(nx) + 0.5) / nx
    r = uniform01(16, seed ^ 0x5)
    def wave(k):
        return np.sin(2 * math.pi * (x + r[k])) + 0.5 * np.sin(4 * math.pi * (x + r[k + 1]))
    rho = 1.0 + amp * wave(0)
    u = 0.3 + 0.5 * amp * wave(2)
    P = rho * (1.0 + 0.5 * amp * wave(4))
    c = np.sqrt(P / rho)
    q = 0.3 * amp * rho * c ** 3 * wave(6)
    rr = 3.0 * P * P / rho * (1.0 + 0.3 * amp * wave(8))
    W0 = np.stack([rho, u, P, q, rr]).reshape(5, 1, nx)
    t = BC_PERIODIC if periodic else BC_TRANSMISSIVE
    col = dict(model=TAU_KN, Kn=Kn, L_ref=1.0, rho_ref=1.0) if Kn is not None else dict(model=TAU_NONE)
    return _problem(SYS5, nx, 1, (0.0, 1.0, 0.0, 1.0), col, [dict(type=t)] * 4, W0, **options)
