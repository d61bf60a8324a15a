/*
 * mmo.h -- CPU ORACLE for the explicit finite-volume time step of the 5-moment (1-D) and
 * 14-moment (2-D) maximum-entropy systems with the interpolative closure
 * (Boccelli, Kaufmann, Magin, McDonald, JCP 2024, arXiv 2401.15233; "PAPER.md").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  It is a plain, slow, scalar fp64
 * restatement of the paper's equations in the paper's order and notation.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no code, header, table or helper with the CUDA library (include/mm.h,
 * paper_2401_15233_b200/csrc/); neither includes the other.
 *
 * Every function cites the PAPER.md line (L...) and equation it follows.  Readings of
 * silent / garbled passages are the ones listed in DESIGN.md section 3 ("Readings").
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): see the header of each function and
 * DESIGN.md section 4.  Functions whose behaviour is the builder's own definition and has no
 * pin outside this file say "parity unpinned".
 *
 * Index conventions
 *   5-moment primitive  W5  = (rho, u, P, q, r)                              Eq 11  L117-125
 *   5-moment conserved  U5  = (rho, rho u, rho u^2+P, rho u^3+3uP+q,
 *                              rho u^4+6u^2P+4uq+r)                          Eq 12  L129-137
 *   14-moment primitive W14 = (rho | u_x u_y u_z | P_xx P_xy P_xz P_yy P_yz P_zz |
 *                              q_x q_y q_z | R),  q_i = Q_ijj (L183), R = R_iijj    L264
 *   14-moment conserved U14 = (rho | rho u_i | U_xx U_xy U_xz U_yy U_yz U_zz |
 *                              U_xjj U_yjj U_zjj | U_iijj)                   Eq 16  L169-181
 *   Field arrays passed through the solver API are [moment][ny][nx] (interior cells only).
 */
#ifndef MMO_H
#define MMO_H

#ifdef __cplusplus
extern "C" {
#endif

enum { MMO_SYS5_1D = 5, MMO_SYS14_2D = 14 };
enum { MMO_TAU_NONE = 0, MMO_TAU_CONST = 1, MMO_TAU_KN = 2 };
enum { MMO_BC_TRANSMISSIVE = 0, MMO_BC_PERIODIC = 1, MMO_BC_DIRICHLET = 2 };
enum { MMO_LIM_NONE = 0, MMO_LIM_MINMOD = 1, MMO_LIM_VANALBADA = 2 };
enum { MMO_FLUX_HLL = 0, MMO_FLUX_RUSANOV = 1 };
enum { MMO_SRC_EXPLICIT = 0, MMO_SRC_POINT_IMPLICIT = 1 };   /* BGK source: forward Euler | point-implicit (L348) */
enum { MMO_TIME_EULER = 0, MMO_TIME_MIDPOINT = 1 };          /* L250: forward Euler | midpoint (2nd-order RK) */
enum { MMO_OK = 0, MMO_EINVAL = -1, MMO_ENONFINITE = -4 };

/* ------------------------------------------------------------------ 5-moment, pointwise */

/* Inverse / forward of the conserved forms of Eq 12 (L129-137). */
void mmo_cons2prim5(const double U[5], double W[5]);
void mmo_prim2cons5(const double W[5], double U[5]);

/* Eq 14 (L151): sigma(q*, r*), unlimited.  Branch of DESIGN.md reading R4. */
double mmo_sigma5(double qstar, double rstar);

/* Eq 15 (L155): s* = q*^3/sigma^2 + (10 - 8 sigma^(1/2)) q*  (dimensionless, reading R1). */
double mmo_sstar5(double qstar, double sigma_bar);

/* Closing moment s (dimensional) of state W with sigma_bar = min(max(sigma,sigma_lim),1)
 * (L163, L512; reading R5).  Also returns sigma and sigma_bar when the pointers are non-NULL. */
double mmo_closure5(const double W[5], double sigma_lim, double *sigma, double *sigma_bar);

/* Flux vector of Eq 12 for a given closing moment s, and with the closure. */
void mmo_flux5_given_s(const double W[5], double s, double F[5]);
void mmo_flux5(const double W[5], double sigma_lim, double F[5]);

/* Eq 34-35 (L543-551), lambda_min by q* -> -q* (Eq 30 / 44), times k, redimensionalised
 * with sqrt(P/rho) and shifted by u (Eq 31). */
void mmo_wavespeed5(const double W[5], double sigma_lim, double k, double *lmin, double *lmax);

/* BGK source of Eq 12d-e (L135-137).  tau = +inf gives C = 0. */
void mmo_source5(const double W[5], double tau, double C[5]);

/* ----------------------------------------------------------------- 14-moment, pointwise */

/* Inverse / forward of the conserved forms of Eq 16 (L169-181). */
void mmo_cons2prim14(const double U[14], double W[14]);
void mmo_prim2cons14(const double W[14], double U[14]);

/* Eq 21 (L210), unlimited, evaluated dimensionless (Eq 6; L272). */
double mmo_sigma14(const double W[14]);

/* Eqs 22-25 (L214-230): dimensional closing moments
 *   Q[i][j][k] = Q_ijk, R2[i][j] = R_ijkk, S[i] = S_ijjkk
 * evaluated dimensionless with sigma_bar = min(max(sigma,sigma_lim),1) and
 * re-dimensionalised (L272).  sigma / sigma_bar returned when non-NULL. */
void mmo_closure14(const double W[14], double sigma_lim, double *sigma, double *sigma_bar,
                   double Q[3][3][3], double R2[3][3], double S[3]);

/* Flux of Eq 16 in direction k (0=x,1=y,2=z) for GIVEN closing moments. */
void mmo_flux14_given_closure(const double W[14], const double Q[3][3][3],
                              const double R2[3][3], const double S[3], int k, double F[14]);
/* Same with the interpolative closure. */
void mmo_flux14(const double W[14], int k, double sigma_lim, double F[14]);

/* Eq 29 / 43 (L393-403, L632-643) in dimensionless variables:
 * lambda*_max(Pdd*, q_d*, qtilde*, sigma). */
double mmo_wavespeed14_star(double Pdd, double qd, double qtilde, double sigma_bar);

/* Eqs 28-31 for direction d (L388-414): lambda_min, lambda_max in the laboratory frame. */
void mmo_wavespeed14(const double W[14], int d, double sigma_lim, double k,
                     double *lmin, double *lmax);

/* BGK source, Eqs 17-18 (L185-194). */
void mmo_source14(const double W[14], double tau, double C[14]);

/* ---------------------------------------------------------------- scheme building blocks */

/* tau model (L284, L474; reading R17).  P is the hydrostatic pressure. */
double mmo_tau(int model, double tau_const, double Kn, double L_ref, double rho_ref,
               double rho, double P);

/* Limiter function psi in [0,1] multiplying the central slope (dm+dp)/2 (L262; reading R14):
 * minmod: 2 min(|dm|,|dp|)/(|dm|+|dp|) if dm*dp>0 else 0;  van Albada (symmetric):
 * 2 dm dp/(dm^2+dp^2) if dm*dp>0 else 0;  none: 0. */
double mmo_limiter_psi(int limiter, double dm, double dp);
/* Limited slope used in per-variable mode: minmod(dm,dp) resp. dm dp (dm+dp)/(dm^2+dp^2). */
double mmo_limited_slope(int limiter, double dm, double dp);

/* MUSCL face states of one cell along one direction from the primitives of the low neighbour Wm,
 * the cell W0 and the high neighbour Wp (L262-266): Wlo = W0 - slope/2, Whi = W0 + slope/2 with
 * slope_k = psi_k (dm_k + dp_k)/2 per variable, or -- shared_limiter (L266) -- one psi = min_k psi_k
 * for all nm variables, a variable with dm = dp = 0 exactly imposing no constraint (reading R14).
 * Pinned by hand-computed three-cell examples (tests/test_oracle_scheme.py). */
void mmo_face_states(int nm, int limiter, int shared_limiter, const double *Wm, const double *W0,
                     const double *Wp, double *Wlo, double *Whi);

/* HLL (L256-258; reading R12) or Rusanov (L258) interface flux for n components. */
void mmo_numflux(int flux, int n, const double *FL, const double *FR, const double *UL,
                 const double *UR, double lminL, double lmaxL, double lminR, double lmaxR,
                 double *Fhat);

/* ------------------------------------------------------------------------------- solver */

typedef struct { int system; int nx, ny; double x0, x1, y0, y1; } mmo_grid;
typedef struct { int model; double tau, Kn, L_ref, rho_ref; } mmo_collision;
/* One side of the domain (order: xlo, xhi, ylo, yhi).  DIRICHLET: piecewise-constant
 * primitive states along the side, chosen by cell-centre coordinate (reading R20);
 * outside every band default_W is used, or zero-gradient when default_W == NULL (L426). */
typedef struct { int type; int nbands; const double *band_lo, *band_hi, *band_W;
                 const double *default_W; } mmo_bc;
typedef struct { double sigma_lim, ws_scale; int limiter, shared_limiter, flux;
                 int source_scheme, time_scheme;   /* MMO_SRC_*, MMO_TIME_* (midpoint needs the explicit source) */
                 int nthreads; /* OpenMP threads over rows; <=0: all available */ } mmo_options;
typedef struct mmo_solver mmo_solver;

int  mmo_create(mmo_solver **out, const mmo_grid *g, const mmo_collision *c,
                const mmo_bc bcs[4], const mmo_options *o);
int  mmo_set_state(mmo_solver *s, const double *U);        /* conserved [nmom][ny][nx] */
int  mmo_set_state_prim(mmo_solver *s, const double *W);   /* primitive [nmom][ny][nx] */
int  mmo_get_state(mmo_solver *s, double *U);
int  mmo_get_state_prim(mmo_solver *s, double *W);
/* dt = cfl / max over interior and ghost cells of max(s_x/dx, s_y/dy)  (L434; reading R13) */
double mmo_cfl_dt(mmo_solver *s, double cfl);
int  mmo_step(mmo_solver *s, int n, double cfl);
int  mmo_step_fixed_dt(mmo_solver *s, int n, double dt);
int  mmo_advance_to(mmo_solver *s, double t_end, double cfl, int max_steps);
int  mmo_get_info(mmo_solver *s, double *t, long long *steps, double *last_dt,
                  double *max_speed);
int  mmo_threads_used(mmo_solver *s);
void mmo_destroy(mmo_solver *s);

#ifdef __cplusplus
}
#endif
#endif /* MMO_H */
