/*
 * mmo_scheme.c -- CPU ORACLE (test infrastructure, not the product; see mmo.h).
 * The explicit finite-volume time step of PAPER.md section 3 (L248-266), step by step:
 *   1. ghost cells (L426)            2. conserved -> primitive (L264)
 *   3. dt from the CFL number (L434) 4. MUSCL slopes on primitives + limiter (L262-266)
 *   5. closure fluxes + approximate wave speeds at both sides of every interface,
 *      HLL / Rusanov interface flux (L256-258, Eqs 21-25, 28-31)
 *   6. forward-Euler update with the BGK source (L250, Eqs 12, 17-18)
 * Cell (i,j), i in [-2,nx+2), j in [-2,ny+2), is stored array-of-structures with two ghost
 * layers.  No blocking, no fusion: every stage sweeps the whole grid into its own array.
 * OpenMP only splits the row loops (rows are independent inside a stage).
 */
#include "mmo.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NG 2 /* ghost layers: a limited slope at the first ghost cell needs the second */

/* ------------------------------------------------------------------ limiter (L262-266) */

/* psi multiplies the central slope (dm + dp)/2.
 *   minmod:       psi = 2 min(|dm|,|dp|) / (|dm| + |dp|)   if dm dp > 0, else 0
 *   van Albada:   psi = 2 dm dp / (dm^2 + dp^2)            if dm dp > 0, else 0
 * (the symmetric van Albada limiter (r^2 + r)/(r^2 + 1) of L262 written for the central
 * slope: (r^2+r)/(r^2+1) dp = psi (dm+dp)/2 with r = dm/dp). */
double mmo_limiter_psi(int limiter, double dm, double dp)
{
    if (limiter == MMO_LIM_NONE) return 0.0;
    if (!(dm * dp > 0.0)) return 0.0;
    if (limiter == MMO_LIM_MINMOD) {
        double am = fabs(dm), ap = fabs(dp);
        return 2.0 * (am < ap ? am : ap) / (am + ap);
    }
    return 2.0 * dm * dp / (dm * dm + dp * dp);
}

/* Per-variable mode: the limited slope itself.
 *   minmod:     sign * min(|dm|,|dp|)                     if dm dp > 0, else 0
 *   van Albada: dm dp (dm + dp) / (dm^2 + dp^2)           if dm dp > 0, else 0 */
double mmo_limited_slope(int limiter, double dm, double dp)
{
    if (limiter == MMO_LIM_NONE) return 0.0;
    if (!(dm * dp > 0.0)) return 0.0;
    if (limiter == MMO_LIM_MINMOD) return fabs(dm) < fabs(dp) ? dm : dp;
    return dm * dp * (dm + dp) / (dm * dm + dp * dp);
}

/* ------------------------------------------------------- interface flux (L256-258, R12) */

/* HLL: S_L = min(lmin_L, lmin_R, 0), S_R = max(lmax_L, lmax_R, 0),
 *   Fhat = (S_R F_L - S_L F_R + S_L S_R (U_R - U_L)) / (S_R - S_L).
 * Rusanov: S = max |lambda| over both states, Fhat = (F_L + F_R)/2 - S (U_R - U_L)/2. */
void mmo_numflux(int flux, int n, const double *FL, const double *FR, const double *UL,
                 const double *UR, double lminL, double lmaxL, double lminR, double lmaxR,
                 double *Fhat)
{
    if (flux == MMO_FLUX_RUSANOV) {
        double S = fabs(lminL);
        if (fabs(lmaxL) > S) S = fabs(lmaxL);
        if (fabs(lminR) > S) S = fabs(lminR);
        if (fabs(lmaxR) > S) S = fabs(lmaxR);
        for (int m = 0; m < n; ++m)
            Fhat[m] = 0.5 * (FL[m] + FR[m]) - 0.5 * S * (UR[m] - UL[m]);
        return;
    }
    double SL = lminL < lminR ? lminL : lminR;
    if (SL > 0.0) SL = 0.0;
    double SR = lmaxL > lmaxR ? lmaxL : lmaxR;
    if (SR < 0.0) SR = 0.0;
    for (int m = 0; m < n; ++m)
        Fhat[m] = (SR * FL[m] - SL * FR[m] + SL * SR * (UR[m] - UL[m])) / (SR - SL);
}

/* ------------------------------------------------------------------------------- solver */

struct mmo_solver {
    mmo_grid g;
    mmo_collision col;
    mmo_options opt;
    mmo_bc bc[4];
    double *bc_store[4];      /* owned copies of the band tables */
    int nm, ndim, sx, sy;     /* moments per cell, space dimensions, padded sizes */
    double dx, dy;
    double *U, *W, *Un;       /* [sy][sx][nm] with ghosts */
    double *U0;               /* midpoint scheme: U^n kept while the half step is in U */
    double *Fx, *Fy;          /* [ny][nx+1][nm], [ny+1][nx][nm] */
    double t, last_dt;
    long long steps;
    int nthreads;
};

static inline size_t cidx(const mmo_solver *s, int i, int j)
{
    return ((size_t)(j + NG) * s->sx + (size_t)(i + NG)) * s->nm;
}

static void c2p(const mmo_solver *s, const double *U, double *W)
{
    if (s->nm == 5) mmo_cons2prim5(U, W); else mmo_cons2prim14(U, W);
}
static void p2c(const mmo_solver *s, const double *W, double *U)
{
    if (s->nm == 5) mmo_prim2cons5(W, U); else mmo_prim2cons14(W, U);
}
static void physflux(const mmo_solver *s, const double *W, int d, double *F)
{
    if (s->nm == 5) mmo_flux5(W, s->opt.sigma_lim, F);
    else mmo_flux14(W, d, s->opt.sigma_lim, F);
}
static void wavespeed(const mmo_solver *s, const double *W, int d, double *lmin, double *lmax)
{
    if (s->nm == 5) mmo_wavespeed5(W, s->opt.sigma_lim, s->opt.ws_scale, lmin, lmax);
    else mmo_wavespeed14(W, d, s->opt.sigma_lim, s->opt.ws_scale, lmin, lmax);
}
static double hydrostatic(const mmo_solver *s, const double *W)
{
    return s->nm == 5 ? W[2] : (W[4] + W[7] + W[9]) / 3.0;
}

int mmo_create(mmo_solver **out, const mmo_grid *g, const mmo_collision *c,
               const mmo_bc bcs[4], const mmo_options *o)
{
    if (!out || !g || !c || !bcs || !o) return MMO_EINVAL;
    if (g->system != MMO_SYS5_1D && g->system != MMO_SYS14_2D) return MMO_EINVAL;
    if (g->nx < 1 || g->ny < 1 || !(g->x1 > g->x0)) return MMO_EINVAL;
    if (g->system == MMO_SYS5_1D && g->ny != 1) return MMO_EINVAL;
    if (g->system == MMO_SYS14_2D && !(g->y1 > g->y0)) return MMO_EINVAL;
    if (!(o->sigma_lim > 0.0) || !(o->ws_scale > 0.0)) return MMO_EINVAL;
    if (o->source_scheme < 0 || o->source_scheme > 1 || o->time_scheme < 0 || o->time_scheme > 1) return MMO_EINVAL;
    if (o->time_scheme == MMO_TIME_MIDPOINT && o->source_scheme != MMO_SRC_EXPLICIT) return MMO_EINVAL;
    mmo_solver *s = (mmo_solver *)calloc(1, sizeof *s);
    if (!s) return MMO_EINVAL;
    s->g = *g; s->col = *c; s->opt = *o;
    s->nm = g->system;
    s->ndim = g->system == MMO_SYS5_1D ? 1 : 2;
    s->sx = g->nx + 2 * NG; s->sy = g->ny + 2 * NG;
    s->dx = (g->x1 - g->x0) / g->nx;
    s->dy = s->ndim == 2 ? (g->y1 - g->y0) / g->ny : 1.0;
    for (int b = 0; b < 2 * s->ndim; ++b) {
        s->bc[b] = bcs[b];
        int nb = bcs[b].type == MMO_BC_DIRICHLET ? bcs[b].nbands : 0;
        if (nb < 0) { mmo_destroy(s); return MMO_EINVAL; }
        /* store: lo[nb], hi[nb], W[nb][nm], default[nm] */
        s->bc_store[b] = (double *)calloc((size_t)nb * (2 + s->nm) + s->nm + 1, sizeof(double));
        double *lo = s->bc_store[b], *hi = lo + nb, *bw = hi + nb, *dw = bw + (size_t)nb * s->nm;
        if (nb > 0) {
            memcpy(lo, bcs[b].band_lo, nb * sizeof(double));
            memcpy(hi, bcs[b].band_hi, nb * sizeof(double));
            memcpy(bw, bcs[b].band_W, (size_t)nb * s->nm * sizeof(double));
        }
        s->bc[b].nbands = nb;
        s->bc[b].band_lo = lo; s->bc[b].band_hi = hi; s->bc[b].band_W = bw;
        if (bcs[b].type == MMO_BC_DIRICHLET && bcs[b].default_W) {
            memcpy(dw, bcs[b].default_W, s->nm * sizeof(double));
            s->bc[b].default_W = dw;
        } else s->bc[b].default_W = 0;
    }
    /* a periodic side needs its partner */
    for (int d = 0; d < s->ndim; ++d)
        if ((s->bc[2 * d].type == MMO_BC_PERIODIC) != (s->bc[2 * d + 1].type == MMO_BC_PERIODIC)) {
            mmo_destroy(s); return MMO_EINVAL;
        }
    size_t ncell = (size_t)s->sx * s->sy;
    s->U = (double *)calloc(ncell * s->nm, sizeof(double));
    s->W = (double *)calloc(ncell * s->nm, sizeof(double));
    s->Un = (double *)calloc(ncell * s->nm, sizeof(double));
    s->U0 = (double *)calloc(ncell * s->nm, sizeof(double));
    s->Fx = (double *)calloc((size_t)g->ny * (g->nx + 1) * s->nm, sizeof(double));
    s->Fy = (double *)calloc((size_t)(g->ny + 1) * g->nx * s->nm, sizeof(double));
    if (!s->U || !s->W || !s->Un || !s->U0 || !s->Fx || !s->Fy) { mmo_destroy(s); return MMO_EINVAL; }
    int nt = o->nthreads;
#ifdef _OPENMP
    if (nt <= 0) nt = omp_get_max_threads();
#else
    nt = 1;
#endif
    s->nthreads = nt;
    *out = s;
    return MMO_OK;
}

void mmo_destroy(mmo_solver *s)
{
    if (!s) return;
    for (int b = 0; b < 4; ++b) free(s->bc_store[b]);
    free(s->U); free(s->W); free(s->Un); free(s->U0); free(s->Fx); free(s->Fy);
    free(s);
}

int mmo_threads_used(mmo_solver *s) { return s ? s->nthreads : 0; }

int mmo_set_state(mmo_solver *s, const double *Uin)
{
    if (!s || !Uin) return MMO_EINVAL;
    int nx = s->g.nx, ny = s->g.ny;
    for (int m = 0; m < s->nm; ++m)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                s->U[cidx(s, i, j) + m] = Uin[((size_t)m * ny + j) * nx + i];
    s->t = 0.0; s->steps = 0; s->last_dt = 0.0;
    return MMO_OK;
}

int mmo_set_state_prim(mmo_solver *s, const double *Win)
{
    if (!s || !Win) return MMO_EINVAL;
    int nx = s->g.nx, ny = s->g.ny;
    double w[14], u[14];
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            for (int m = 0; m < s->nm; ++m) w[m] = Win[((size_t)m * ny + j) * nx + i];
            p2c(s, w, u);
            for (int m = 0; m < s->nm; ++m) s->U[cidx(s, i, j) + m] = u[m];
        }
    s->t = 0.0; s->steps = 0; s->last_dt = 0.0;
    return MMO_OK;
}

int mmo_get_state(mmo_solver *s, double *Uout)
{
    if (!s || !Uout) return MMO_EINVAL;
    int nx = s->g.nx, ny = s->g.ny;
    for (int m = 0; m < s->nm; ++m)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i)
                Uout[((size_t)m * ny + j) * nx + i] = s->U[cidx(s, i, j) + m];
    return MMO_OK;
}

int mmo_get_state_prim(mmo_solver *s, double *Wout)
{
    if (!s || !Wout) return MMO_EINVAL;
    int nx = s->g.nx, ny = s->g.ny;
    double w[14];
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            c2p(s, s->U + cidx(s, i, j), w);
            for (int m = 0; m < s->nm; ++m) Wout[((size_t)m * ny + j) * nx + i] = w[m];
        }
    return MMO_OK;
}

/* ---- step 1: ghost cells (L426: "imposing the said values into the ghost cells ...
 * remaining boundaries set to the background ... zero-gradient").  Corner ghosts are
 * never read (stencils are face-only). */
static void ghost_value(const mmo_solver *s, int side, double coord, const double *Uinner,
                        const double *Uperiodic, double *Ug)
{
    const mmo_bc *b = &s->bc[side];
    const double *src = Uinner;                       /* zero-gradient copy */
    if (b->type == MMO_BC_PERIODIC) src = Uperiodic;
    else if (b->type == MMO_BC_DIRICHLET) {
        const double *Wd = b->default_W;
        for (int k = 0; k < b->nbands; ++k)          /* cell-centre test, reading R20 */
            if (coord >= b->band_lo[k] && coord <= b->band_hi[k]) { Wd = b->band_W + (size_t)k * s->nm; break; }
        if (Wd) { p2c(s, Wd, Ug); return; }
    }
    memcpy(Ug, src, s->nm * sizeof(double));
}

static void fill_ghosts(mmo_solver *s)
{
    int nx = s->g.nx, ny = s->g.ny;
    for (int j = 0; j < ny; ++j) {
        double yc = s->g.y0 + (j + 0.5) * s->dy;
        for (int g = 1; g <= NG; ++g) {
            /* periodic image of ghost -g is cell nx-g; of ghost nx-1+g is cell g-1 */
            int ipl = ((nx - g) % nx + nx) % nx, iph = (g - 1) % nx;
            ghost_value(s, 0, yc, s->U + cidx(s, 0, j), s->U + cidx(s, ipl, j), s->U + cidx(s, -g, j));
            ghost_value(s, 1, yc, s->U + cidx(s, nx - 1, j), s->U + cidx(s, iph, j), s->U + cidx(s, nx - 1 + g, j));
        }
    }
    if (s->ndim == 2)
        for (int i = 0; i < nx; ++i) {
            double xc = s->g.x0 + (i + 0.5) * s->dx;
            for (int g = 1; g <= NG; ++g) {
                int jpl = ((ny - g) % ny + ny) % ny, jph = (g - 1) % ny;
                ghost_value(s, 2, xc, s->U + cidx(s, i, 0), s->U + cidx(s, i, jpl), s->U + cidx(s, i, -g));
                ghost_value(s, 3, xc, s->U + cidx(s, i, ny - 1), s->U + cidx(s, i, jph), s->U + cidx(s, i, ny - 1 + g));
            }
        }
}

/* is (i,j) a cell that is ever read: interior, or a face ghost (not a corner) */
static int cell_in_use(const mmo_solver *s, int i, int j)
{
    int nx = s->g.nx, ny = s->g.ny;
    int in_x = i >= 0 && i < nx, in_y = j >= 0 && j < ny;
    if (s->ndim == 1) return in_y;
    return in_x || in_y;
}

/* ---- step 2: W = cons -> prim in every cell that is read (L264) */
static void all_cons2prim(mmo_solver *s)
{
    int nx = s->g.nx, ny = s->g.ny;
    int jlo = s->ndim == 2 ? -NG : 0, jhi = s->ndim == 2 ? ny + NG : ny;
#pragma omp parallel for num_threads(s->nthreads) schedule(static)
    for (int j = jlo; j < jhi; ++j)
        for (int i = -NG; i < nx + NG; ++i)
            if (cell_in_use(s, i, j)) c2p(s, s->U + cidx(s, i, j), s->W + cidx(s, i, j));
}

/* ---- step 3: max over interior and ghost cells of max(s_x/dx, s_y/dy), s_d =
 * max(|lmin_d|,|lmax_d|) from cell-centre primitives (L434; reading R13).
 * Returns NaN when a cell has rho <= 0, P <= 0 or a non-finite speed. */
static double max_rate(mmo_solver *s, double *max_speed)
{
    int nx = s->g.nx, ny = s->g.ny;
    int jlo = s->ndim == 2 ? -NG : 0, jhi = s->ndim == 2 ? ny + NG : ny;
    double rate = 0.0, speed = 0.0;
    int bad = 0;
#pragma omp parallel for num_threads(s->nthreads) schedule(static) reduction(max : rate, speed) reduction(| : bad)
    for (int j = jlo; j < jhi; ++j)
        for (int i = -NG; i < nx + NG; ++i) {
            if (!cell_in_use(s, i, j)) continue;
            const double *W = s->W + cidx(s, i, j);
            if (!(W[0] > 0.0) || !(hydrostatic(s, W) > 0.0)) { bad = 1; continue; }
            for (int d = 0; d < s->ndim; ++d) {
                double lmin, lmax;
                wavespeed(s, W, d, &lmin, &lmax);
                double sd = fabs(lmin) > fabs(lmax) ? fabs(lmin) : fabs(lmax);
                if (!isfinite(sd)) { bad = 1; continue; }
                double r = sd / (d == 0 ? s->dx : s->dy);
                if (r > rate) rate = r;
                if (sd > speed) speed = sd;
            }
        }
    if (max_speed) *max_speed = bad ? NAN : speed;
    return bad ? NAN : rate;
}

/* ---- step 4: limited slopes and face states of cell c along one direction (L262-266).
 * Wm, W0, Wp: primitives of the low neighbour, the cell, the high neighbour.
 * Wlo = W0 - slope/2 (low face), Whi = W0 + slope/2 (high face).
 * Exported so that tests/test_oracle_scheme.py can pin it against hand-computed face values. */
void mmo_face_states(int nm, int lim, int shared_limiter, const double *Wm, const double *W0,
                     const double *Wp, double *Wlo, double *Whi)
{
    double slope[14];
    if (shared_limiter && lim != MMO_LIM_NONE) {
        /* L266: the same, most stringent limiter value for all primitive variables.
         * A variable with dm = dp = 0 imposes no constraint (reading R14). */
        double psi = 1.0;
        for (int k = 0; k < nm; ++k) {
            double dm = W0[k] - Wm[k], dp = Wp[k] - W0[k];
            if (dm == 0.0 && dp == 0.0) continue;
            double pk = mmo_limiter_psi(lim, dm, dp);
            if (pk < psi) psi = pk;
        }
        for (int k = 0; k < nm; ++k) {
            double dm = W0[k] - Wm[k], dp = Wp[k] - W0[k];
            slope[k] = psi * (0.5 * (dm + dp));
        }
    } else {
        for (int k = 0; k < nm; ++k)
            slope[k] = mmo_limited_slope(lim, W0[k] - Wm[k], Wp[k] - W0[k]);
    }
    for (int k = 0; k < nm; ++k) {
        Wlo[k] = W0[k] - 0.5 * slope[k];
        Whi[k] = W0[k] + 0.5 * slope[k];
    }
}

static void face_states(const mmo_solver *s, const double *Wm, const double *W0,
                        const double *Wp, double *Wlo, double *Whi)
{
    mmo_face_states(s->nm, s->opt.limiter, s->opt.shared_limiter, Wm, W0, Wp, Wlo, Whi);
}

/* ---- step 5: interface flux between cell a (low side) and cell b (high side) along d.
 * am/bp are the outer neighbours needed for the slopes. */
static void interface_flux(const mmo_solver *s, int d, const double *Wam, const double *Wa,
                           const double *Wb, const double *Wbp, double *Fhat)
{
    double lo[14], hi[14], WL[14], WR[14];
    face_states(s, Wam, Wa, Wb, lo, WL);     /* high face of the low cell  */
    face_states(s, Wa, Wb, Wbp, WR, hi);     /* low face of the high cell  */
    double FL[14], FR[14], UL[14], UR[14], lminL, lmaxL, lminR, lmaxR;
    physflux(s, WL, d, FL);
    physflux(s, WR, d, FR);
    p2c(s, WL, UL);
    p2c(s, WR, UR);
    wavespeed(s, WL, d, &lminL, &lmaxL);
    wavespeed(s, WR, d, &lminR, &lmaxR);
    mmo_numflux(s->opt.flux, s->nm, FL, FR, UL, UR, lminL, lmaxL, lminR, lmaxR, Fhat);
}

static void all_fluxes(mmo_solver *s)
{
    int nx = s->g.nx, ny = s->g.ny, nm = s->nm;
    /* x interfaces: Fx[j][f], f = 0..nx, between cells (f-1, j) and (f, j) */
#pragma omp parallel for num_threads(s->nthreads) schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int f = 0; f <= nx; ++f)
            interface_flux(s, 0, s->W + cidx(s, f - 2, j), s->W + cidx(s, f - 1, j),
                           s->W + cidx(s, f, j), s->W + cidx(s, f + 1, j),
                           s->Fx + ((size_t)j * (nx + 1) + f) * nm);
    if (s->ndim == 2) {
        /* y interfaces: Fy[f][i], f = 0..ny, between cells (i, f-1) and (i, f) */
#pragma omp parallel for num_threads(s->nthreads) schedule(static)
        for (int f = 0; f <= ny; ++f)
            for (int i = 0; i < nx; ++i)
                interface_flux(s, 1, s->W + cidx(s, i, f - 2), s->W + cidx(s, i, f - 1),
                               s->W + cidx(s, i, f), s->W + cidx(s, i, f + 1),
                               s->Fy + ((size_t)f * nx + i) * nm);
    }
}

/* Moments of the Maxwellian with the density, velocity and hydrostatic pressure of W (L73, L127):
 * the equilibrium the BGK operator relaxes to (Eqs 17-18; Eq 12d-e). */
static void equilibrium_of(const mmo_solver *s, const double *W, double *Ueq)
{
    double Weq[14];
    double P = hydrostatic(s, W);
    if (s->nm == 5) {
        Weq[0] = W[0]; Weq[1] = W[1]; Weq[2] = P; Weq[3] = 0.0; Weq[4] = 3.0 * P * P / W[0];
    } else {
        for (int m = 0; m < 14; ++m) Weq[m] = 0.0;
        Weq[0] = W[0]; Weq[1] = W[1]; Weq[2] = W[2]; Weq[3] = W[3];
        Weq[4] = P; Weq[7] = P; Weq[9] = P;
        Weq[13] = 15.0 * P * P / W[0];
    }
    p2c(s, Weq, Ueq);
}

/* ---- step 6: U^{new} = B - dt/dx (Fx_{i+1/2} - Fx_{i-1/2}) - dt/dy (Fy_{j+1/2} - Fy_{j-1/2}) + source,
 * with the fluxes and primitives W of the state currently in s->U, and B = `base` (U^n itself for
 * forward Euler; U^n while s->U holds the half step of the midpoint scheme, L250).
 * Source, explicit:        + dt C(W), tau from the cell's own W (L250; Eqs 12, 17-18).
 * Source, point-implicit (L348): with U* the flux-updated state, the BGK relaxation is integrated by
 *   backward Euler, U^{new} = (U* + (dt/tau) U_eq) / (1 + dt/tau); U_eq and tau depend only on rho, u
 *   and the hydrostatic pressure, which the source does not change, so they are those of U*. */
static void update(mmo_solver *s, double dt, const double *base)
{
    int nx = s->g.nx, ny = s->g.ny, nm = s->nm;
#pragma omp parallel for num_threads(s->nthreads) schedule(static)
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            const double *U = base + cidx(s, i, j), *W = s->W + cidx(s, i, j);
            double *Un = s->Un + cidx(s, i, j);
            const double *Fw = s->Fx + ((size_t)j * (nx + 1) + i) * nm, *Fe = Fw + nm;
            double v[14];
            for (int m = 0; m < nm; ++m) {
                v[m] = U[m] - dt / s->dx * (Fe[m] - Fw[m]);
                if (s->ndim == 2) {
                    const double *Fs = s->Fy + ((size_t)j * nx + i) * nm;
                    const double *Fn = s->Fy + ((size_t)(j + 1) * nx + i) * nm;
                    v[m] -= dt / s->dy * (Fn[m] - Fs[m]);
                }
            }
            if (s->col.model == MMO_TAU_NONE) {
                for (int m = 0; m < nm; ++m) Un[m] = v[m];
            } else if (s->opt.source_scheme == MMO_SRC_POINT_IMPLICIT) {
                double Ws[14], Ueq[14];
                c2p(s, v, Ws);
                double tau = mmo_tau(s->col.model, s->col.tau, s->col.Kn, s->col.L_ref,
                                     s->col.rho_ref, Ws[0], hydrostatic(s, Ws));
                equilibrium_of(s, Ws, Ueq);
                double x = dt / tau;
                for (int m = 0; m < nm; ++m) Un[m] = (v[m] + x * Ueq[m]) / (1.0 + x);
            } else {
                double C[14];
                double tau = mmo_tau(s->col.model, s->col.tau, s->col.Kn, s->col.L_ref,
                                     s->col.rho_ref, W[0], hydrostatic(s, W));
                if (nm == 5) mmo_source5(W, tau, C);
                else mmo_source14(W, tau, C);
                for (int m = 0; m < nm; ++m) Un[m] = v[m] + dt * C[m];
            }
        }
    double *tmp = s->U; s->U = s->Un; s->Un = tmp;
}

/* one step; dt <= 0 means "from the CFL number" */
static int one_step(mmo_solver *s, double dt_fixed, double cfl, double t_end)
{
    fill_ghosts(s);
    all_cons2prim(s);
    double dt = dt_fixed;
    if (!(dt > 0.0)) {
        double rate = max_rate(s, 0);
        if (!isfinite(rate) || !(rate > 0.0)) return MMO_ENONFINITE;
        dt = cfl / rate;
    }
    int last = t_end > s->t && s->t + dt >= t_end;               /* land on t_end */
    if (last) dt = t_end - s->t;
    if (s->opt.time_scheme == MMO_TIME_MIDPOINT) {
        /* L250 "midpoint Euler (2nd order Runge-Kutta)": U' = U^n + dt/2 L(U^n); U^{n+1} = U^n + dt L(U') */
        size_t nbytes = (size_t)s->sx * s->sy * s->nm * sizeof(double);
        memcpy(s->U0, s->U, nbytes);
        all_fluxes(s);
        update(s, 0.5 * dt, s->U0);
        fill_ghosts(s);
        all_cons2prim(s);
        all_fluxes(s);
        update(s, dt, s->U0);
    } else {
        all_fluxes(s);
        update(s, dt, s->U);
    }
    if (last) s->t = t_end; else s->t += dt;
    s->last_dt = dt;
    s->steps += 1;
    return MMO_OK;
}

double mmo_cfl_dt(mmo_solver *s, double cfl)
{
    if (!s) return NAN;
    fill_ghosts(s);
    all_cons2prim(s);
    return cfl / max_rate(s, 0);
}

int mmo_step(mmo_solver *s, int n, double cfl)
{
    if (!s || n < 0 || !(cfl > 0.0)) return MMO_EINVAL;
    for (int k = 0; k < n; ++k) {
        int rc = one_step(s, 0.0, cfl, -1.0);
        if (rc) return rc;
    }
    return MMO_OK;
}

int mmo_step_fixed_dt(mmo_solver *s, int n, double dt)
{
    if (!s || n < 0 || !(dt > 0.0)) return MMO_EINVAL;
    for (int k = 0; k < n; ++k) {
        int rc = one_step(s, dt, 0.0, -1.0);
        if (rc) return rc;
    }
    return MMO_OK;
}

int mmo_advance_to(mmo_solver *s, double t_end, double cfl, int max_steps)
{
    if (!s || !(cfl > 0.0)) return MMO_EINVAL;
    int k = 0;
    while (s->t < t_end && (max_steps <= 0 || k < max_steps)) {
        int rc = one_step(s, 0.0, cfl, t_end);
        if (rc) return rc;
        ++k;
    }
    return MMO_OK;
}

int mmo_get_info(mmo_solver *s, double *t, long long *steps, double *last_dt, double *max_speed)
{
    if (!s) return MMO_EINVAL;
    if (t) *t = s->t;
    if (steps) *steps = s->steps;
    if (last_dt) *last_dt = s->last_dt;
    if (max_speed) {
        fill_ghosts(s);
        all_cons2prim(s);
        max_rate(s, max_speed);
        if (!isfinite(*max_speed)) return MMO_ENONFINITE;
    }
    return MMO_OK;
}
