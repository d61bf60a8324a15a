/*
 * mm.h -- C-ABI of the B200 (sm_100a) maximum-entropy moment-method time step.
 *
 * One thing is computed: the explicit finite-volume time step of the 5-moment (1-D) and
 * 14-moment (2-D) maximum-entropy systems with the interpolative closure of
 * Boccelli, Kaufmann, Magin, McDonald, JCP 2024 (arXiv 2401.15233; "PAPER.md"):
 *   ghost cells (L426) -> conserved->primitive (L264) -> MUSCL + limiter (L262-266) ->
 *   closure fluxes (Eqs 12-15, 16, 21-25) + approximate wave speeds (Eqs 28-31, 34-35) ->
 *   HLL / Rusanov interface flux (L256-258) -> forward-Euler update with the BGK source
 *   (L250; Eqs 12d-e, 17-18) -> CFL max-reduction for the next dt (L434).
 * Every step of that path runs in CUDA kernels (paper_2401_15233_b200/csrc/); the host code
 * behind these calls only validates arguments and launches.  There is NO CPU fallback: without
 * a CUDA device every compute call returns MM_ECUDA.
 *
 * Conventions
 *   - all functions return MM_OK (0) or a negative mm_status; mm_strerror() names it.
 *   - pointers are HOST pointers unless the argument list says "device"; `on_device` flags
 *     say which kind a state buffer is.  The caller owns every buffer it passes; tables in
 *     mm_bc are copied at mm_create.
 *   - the library never allocates device memory: the caller hands in `d_workspace`
 *     (>= mm_workspace_bytes(), 256-byte aligned, e.g. a torch uint8 tensor) and a stream;
 *     all work is enqueued on that stream, nothing synchronises unless stated.  A caller that has
 *     no way of obtaining a workspace uses mm_static5_run (end of this header), whose scratch is a
 *     fixed array inside the library image.
 *   - solver objects are independent; one object is not thread-safe.
 *
 * Moment order (structure of arrays, fp64), field arrays are [moment][ny][nx], interior cells:
 *   5-moment   conserved U = (rho, rho u, rho u^2+P, rho u^3+3uP+q, rho u^4+6u^2P+4uq+r)   Eq 12
 *              primitive W = (rho, u, P, q, r)                                              Eq 11
 *   14-moment  conserved U = (rho | rho u_x,u_y,u_z | U_xx U_xy U_xz U_yy U_yz U_zz |
 *                             U_xjj U_yjj U_zjj | U_iijj)                                   Eq 16
 *              primitive W = (rho | u_x u_y u_z | P_xx P_xy P_xz P_yy P_yz P_zz |
 *                             q_x q_y q_z | R),  q_i = Q_ijj (L183), R = R_iijj             L264
 */
#ifndef MM_H
#define MM_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum { MM_OK = 0, MM_EINVAL = -1, MM_EWORKSPACE = -2, MM_ECUDA = -3,
               MM_ENONFINITE = -4, MM_ETOOLARGE = -5 /* mm_static5_run only */ } mm_status;

enum { MM_SYS5_1D = 5, MM_SYS14_2D = 14 };                       /* section 2.3 / 2.4 */
enum { MM_TAU_NONE = 0, MM_TAU_CONST = 1, MM_TAU_KN = 2 };
enum { MM_BC_TRANSMISSIVE = 0, MM_BC_PERIODIC = 1, MM_BC_DIRICHLET = 2 };
enum { MM_LIM_NONE = 0, MM_LIM_MINMOD = 1, MM_LIM_VANALBADA = 2 };
enum { MM_FLUX_HLL = 0, MM_FLUX_RUSANOV = 1 };
enum { MM_SRC_EXPLICIT = 0, MM_SRC_POINT_IMPLICIT = 1 };
enum { MM_TIME_EULER = 0, MM_TIME_MIDPOINT = 1 };
#define MM_MAX_BANDS 8

typedef struct mm_solver mm_solver;   /* opaque, host object; freed by mm_destroy */

/* Grid: nx x ny interior cells on [x0,x1] x [y0,y1]; ny = 1 (y0,y1 ignored) for MM_SYS5_1D. */
typedef struct { int system; int nx, ny; double x0, x1, y0, y1; } mm_grid;

/* Gas (Eq 6; L284): the specific gas constant R in T = P/(rho R).  The moment systems themselves
 * never see a temperature (the state is rho, u, P, q, R_iijj); R_gas enters where the problem
 * statement gives one: Dirichlet states given as Maxwellians (rho, u, T) (mm_bc.band_state, L426:
 * "imposing the said values [rho_jet, u_jet, T_jet] into the ghost cells").  gas == NULL means
 * R_gas = 1 (the non-dimensional configs of BASELINE.json).  The adiabatic exponent is implied by
 * the system: 3 for the 1D1V 5-moment gas, 5/3 for the 14-moment gas. */
typedef struct { double R_gas; } mm_gas;

/* BGK relaxation time (L284, L474):
 *   MM_TAU_NONE  collisionless, source disabled (L432)
 *   MM_TAU_CONST tau
 *   MM_TAU_KN    tau(rho,P) = Kn L_ref (rho_ref/rho) / sqrt(8 P / (pi rho)),  P hydrostatic,
 *                i.e. tau = lambda / v_th with lambda ~ 1/rho and Kn = lambda(rho_ref)/L_ref. */
typedef struct { int model; double tau, Kn, L_ref, rho_ref; } mm_collision;

/* One side of the domain; mm_create takes 4 of them in the order xlo, xhi, ylo, yhi.
 *   MM_BC_TRANSMISSIVE zero-gradient copy of the adjacent interior cell (L426)
 *   MM_BC_PERIODIC     both sides of that direction must be periodic
 *   MM_BC_DIRICHLET    piecewise-constant PRIMITIVE states along the side (inflow jets, L426):
 *                      band k holds where the cell-centre coordinate along the side is in
 *                      [band_lo[k], band_hi[k]]; elsewhere default_W, or zero-gradient when
 *                      default_W == NULL.  nbands <= MM_MAX_BANDS.
 *   band_state         MM_STATE_PRIMITIVE: band_W is [nbands][nmom] and default_W [nmom] primitives W;
 *                      MM_STATE_MAXWELLIAN: band_W is [nbands][5] and default_W [5] = (rho, u_x, u_y, u_z, T)
 *                      (u_y, u_z ignored by MM_SYS5_1D), expanded ON THE DEVICE to the Maxwellian of L73 /
 *                      L127: P_ij = rho R_gas T delta_ij, q = 0, R_iijj = 15 P^2/rho (5-moment r = 3 P^2/rho). */
enum { MM_STATE_PRIMITIVE = 0, MM_STATE_MAXWELLIAN = 1 };
typedef struct { int type; int nbands; const double *band_lo, *band_hi, *band_W;
                 const double *default_W; int band_state; } mm_bc;

typedef struct {
    double sigma_lim;     /* lower limit of sigma inside closure + wave speeds (L163, L512); 1e-4 */
    double ws_scale;      /* wave-speed inflation k >= 1 (L409); 1.0 */
    int limiter;          /* MM_LIM_MINMOD | MM_LIM_VANALBADA (L262) | MM_LIM_NONE (1st order) */
    int shared_limiter;   /* 1: the most stringent limiter value for all primitives (L266) */
    int flux;             /* MM_FLUX_HLL | MM_FLUX_RUSANOV (L258) */
    int source_scheme;    /* MM_SRC_EXPLICIT: + dt C(W^n), forward Euler (L250) | MM_SRC_POINT_IMPLICIT (L348):
                           * with U* the flux-updated state, U^{n+1} = (U* + (dt/tau) U_eq)/(1 + dt/tau);
                           * U_eq, tau from rho, u, hydrostatic P of U* (collision invariants) */
    int time_scheme;      /* MM_TIME_EULER (L250, L434) | MM_TIME_MIDPOINT (L250, 2nd-order Runge-Kutta):
                           * U' = U^n + dt/2 L(U^n), U^{n+1} = U^n + dt L(U'), dt from the CFL rate of U^n;
                           * two kernel passes per step; requires MM_SRC_EXPLICIT */
    void *stream;         /* cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default */
} mm_options;

/* Bytes of device workspace mm_create needs for this grid: two padded state copies (the 14-moment
 * system keeps each copy as conserved moments U and as primitives W(U), 4 x 14 planes in all; the
 * 5-moment system 2 x 5 planes), boundary tables, control block, wave-speed table, dt history.
 * 0 on invalid grid. */
size_t mm_workspace_bytes(const mm_grid *grid);

/* Build a solver on caller-provided device memory (problem statement of section 3 L250 and section 6
 * L426: grid, gas, relaxation-time model, boundary data).  d_workspace: DEVICE pointer.  gas may be
 * NULL (R_gas = 1); MM_EINVAL if R_gas <= 0. */
int mm_create(mm_solver **out, const mm_grid *grid, const mm_gas *gas, const mm_collision *collision,
              const mm_bc bcs[4], const mm_options *options, void *d_workspace, size_t bytes);

/* Load the interior state (conserved resp. primitive moments, [nmom][ny][nx]), fill the ghost
 * cells and run the CFL reduction; resets t = 0, steps = 0.  Host buffers are copied with
 * cudaMemcpyAsync on the solver's stream (pin them for true overlap).  The conserved moments given
 * to mm_set_state are stored as they are (mm_get_state returns the same bits); mm_get_state +
 * mm_get_info followed by mm_set_state + mm_set_clock on a new solver resumes a run bit for bit. */
int mm_set_state(mm_solver *s, const double *U, int on_device);
int mm_set_state_prim(mm_solver *s, const double *W, int on_device);

/* n forward-Euler steps (L250), each with dt = cfl / max_cells max(s_x/dx, s_y/dy) from the
 * cell-centre wave speeds of the current state, ghost cells included (L434).  Asynchronous:
 * dt, t and the step counter live in device memory, nothing is read back. */
int mm_step(mm_solver *s, int n, double cfl);
/* n steps with the given dt (parity mode). */
int mm_step_fixed_dt(mm_solver *s, int n, double dt);
/* CFL steps until t == t_end (last step clipped); max_steps <= 0: unlimited.  Synchronises. */
int mm_advance_to(mm_solver *s, double t_end, double cfl, int max_steps);

/* Copy out the interior state; synchronises the stream. */
int mm_get_state(mm_solver *s, double *U, int on_device);
int mm_get_state_prim(mm_solver *s, double *W, int on_device);

/* t, completed steps, last dt, max wave speed of the current state (any pointer may be NULL).
 * Synchronises.  Returns MM_ENONFINITE if the CFL reduction met rho <= 0, P <= 0 or a
 * non-finite wave speed; from that point on steps leave the state untouched. */
int mm_get_info(mm_solver *s, double *t, long long *steps, double *last_dt, double *max_speed);
/* dt the next mm_step(., cfl) would take.  Synchronises. */
int mm_cfl_dt(mm_solver *s, double cfl, double *dt);

/* Time steps dt of the steps first_step .. first_step + n - 1 (0-based; Fig 14 plots this
 * curve).  The library keeps the last 65536 on the device, so n steps can be enqueued without a host
 * round trip per step.  `dt` is a host array.  MM_EINVAL if the range has not been taken yet or has
 * been overwritten.  Synchronises. */
int mm_get_dt_history(mm_solver *s, long long first_step, int n, double *dt);
/* Restore the clock after mm_set_state* (which resets t and the step counter to 0): with
 * mm_get_state + mm_get_info this makes mm_set_state + mm_set_clock a checkpoint / resume pair. */
int mm_set_clock(mm_solver *s, double t, long long steps);

/* Host logic only (no device needed): the work decomposition the 14-moment step kernel is launched
 * with on a device of `sms` SMs -- strips of 30 cells in x times row chunks in y, one warp each,
 * chosen to fill whole waves of sms * warps_per_sm resident warps. */
int mm_decomposition(int nx, int ny, int zsym, int sms, int *nstrips, int *nchunks, int *warps_per_sm);

/* Number of kernel launches enqueued by this solver so far. */
long long mm_launch_count(const mm_solver *s);

/* z-symmetric fast path (SURVEY.md section 8(a) design note).  When the
 * state given to mm_set_state* and every Dirichlet boundary state have
 * u_z = P_xz = P_yz = q_z = 0 exactly (checked on the device at mm_set_state*), the scheme keeps
 * them zero for all time and the 14-moment step runs a kernel variant in which they are
 * compile-time zeros; all 14 arrays are still carried and written.  The general variant runs
 * otherwise.  mm_set_fast_path(s, 0) forces the general variant (default: allowed = 1);
 * mm_fast_path_active returns 1 when the next mm_step* would run the fast variant. */
int mm_set_fast_path(mm_solver *s, int allow);
int mm_fast_path_active(const mm_solver *s);

/* Launch timing (used by bench.py for the roofline line; creates CUDA events, no
 * device memory).  The hooks that need device scratch of their own (FP64 peak probe, accuracy self-test
 * of the elementary functions) are NOT part of this library: include/mm_bench.h, libmm_bench.so.
 * Between mm_profile_begin and mm_profile_end every launch of the fused step kernel is
 * bracketed by CUDA events on the solver's stream; mm_profile_end synchronises and returns the
 * summed device time of those launches (milliseconds) and their number. */
int mm_profile_begin(mm_solver *s);
int mm_profile_end(mm_solver *s, double *step_kernel_ms, long long *launches);
/* ---- Batched 1-D 5-moment solver: `ntubes` independent shock tubes
 * of nx cells on [x0, x1], transmissive ends (L426), each with its own sigma_lim (L163) and Knudsen
 * number (tau = Kn L_ref (rho_ref/rho)/sqrt(8P/(pi rho)), L284; Kn <= 0: collisionless), its own CFL
 * time step (L434) and clock -- the sigma_lim x Kn sweep of PAPER.md section 4.3 (L340-356, Fig 7) as
 * one launch sequence.  Same scheme as MM_SYS5_1D (Eq 12, 14, 15, 34-35; forward Euler, explicit
 * source).  sigma_lim and Kn are host arrays [ntubes], copied at create; workspace rules as mm_create.
 * States: W primitives [5][nx] (one tube, copied to all; per_tube = 0) or [ntubes][5][nx];
 * U conserved [ntubes][5][nx].  mm_batch5_advance_to steps until every tube has reached t_end (each
 * lands on it exactly and then idles) or max_steps (> 0) steps were taken; the per-tube step counts
 * of mm_batch5_get_info are the paper's measure of computational cost (L342).  failed[j] != 0 and
 * MM_ENONFINITE when a tube's CFL reduction met rho <= 0, P <= 0 or a non-finite speed. */
typedef struct mm_batch5 mm_batch5;
size_t mm_batch5_workspace_bytes(int nx, int ntubes);
int mm_batch5_create(mm_batch5 **out, int nx, int ntubes, double x0, double x1, const double *sigma_lim,
                     const double *Kn, double L_ref, double rho_ref, double ws_scale, int limiter,
                     int shared_limiter, int flux, void *stream, void *d_workspace, size_t bytes);
int mm_batch5_set_state_prim(mm_batch5 *b, const double *W, int per_tube, int on_device);
int mm_batch5_step(mm_batch5 *b, int n, double cfl);
int mm_batch5_step_fixed_dt(mm_batch5 *b, int n, double dt);
int mm_batch5_advance_to(mm_batch5 *b, double t_end, double cfl, long long max_steps);
int mm_batch5_get_state(mm_batch5 *b, double *U, int on_device);
int mm_batch5_get_info(mm_batch5 *b, double *t, long long *steps, int *failed);
long long mm_batch5_launch_count(const mm_batch5 *b);
void mm_batch5_destroy(mm_batch5 *b);

void mm_destroy(mm_solver *s);
const char *mm_strerror(int status);

/* ---- mm_static5_run: a whole 1-D 5-moment run for callers that cannot provide a workspace.
 *
 * Everything above needs `d_workspace`, i.e. a caller able to obtain device memory of a size the library
 * dictates.  Some users of this library are not: a routine called back from inside somebody else's
 * solver or coupling framework is handed the device (or host) arrays of its input and output and
 * nothing else -- the host application owns the device-memory pool, has often reserved all of the
 * GPU for it, and a raw runtime allocation from the callee then fails or is forbidden by the host's
 * rules; a caller sitting in a time-critical loop cannot afford the device-wide synchronisation a
 * runtime allocation or release implies; and a C or Fortran driver that links this library alone has
 * no CUDA runtime of its own to allocate with.  For them the scratch of the 5-moment step (control
 * block, boundary table, dt history and the two padded copies of the state that k_step5 ping-pongs
 * between) lives in ONE file-scope device array of MM_STATIC5_SCRATCH_BYTES (4 MiB) compiled into
 * libmm.so.  Every GPU whose context loads the library carries these 4 MiB until the process exits,
 * whether or not this function is ever called; that is the price, and the reason the limit is modest:
 *   nx <= MM_STATIC5_MAX_NX (8192 cells); larger nx returns MM_ETOOLARGE before any CUDA call.
 *
 * What it does: the same launches as mm_create(MM_SYS5_1D) + mm_set_state_prim(W0) + n steps
 * (dt > 0: n steps of that fixed dt, mm_step_fixed_dt; otherwise n CFL steps at Courant number cfl,
 * mm_step) + mm_get_state(U), on options->stream, with the built-in array as the workspace.  The
 * results are those of that sequence, bit for bit.
 *   W0      primitives (rho, u, P, q, r), [5][nx]          U   conserved moments out, [5][nx]
 *   on_device  1: W0 and U are device pointers, 0: host pointers (copied on the stream; no staging
 *           buffer is allocated, the idle state copy inside the array serves)
 *   bcs     two sides (xlo, xhi) as in mm_create, or NULL for transmissive ends (L426)
 *   t_end   host pointer, receives the time reached; may be NULL
 * Returns MM_OK, MM_EINVAL, MM_ETOOLARGE, MM_ECUDA (also: no device -- there is no CPU path) or
 * MM_ENONFINITE as mm_get_info does.  Synchronises the stream before returning.  It performs no device
 * or pinned-host allocation and releases none; host-side it builds and frees one small solver object.
 *
 * Sharing.  There is one array per device and process, and every call on that device uses it.  It keeps
 * whatever the previous call left: each call therefore zero-fills the part it is about to use (control
 * block, accumulators, tables, both state copies) on the stream before anything reads it.  Two calls
 * whose GPU work overlaps would overwrite each other's state -- a race with silently wrong numbers.  The
 * function prevents that inside one process by holding a lock from its first launch until its stream has
 * drained; nothing can be done about it from here if the array were reached by other means, so do not.
 *
 * First call on a device.  The device address of the array is looked up (and the module holding it is
 * loaded) the first time the function runs with that device current; later calls on that device reuse
 * it.  Make that first call during start-up, outside any stream capture: loading a module is not a
 * stream operation. */
#define MM_STATIC5_MAX_NX 8192
#define MM_STATIC5_SCRATCH_BYTES (4u << 20)
int mm_static5_run(int nx, double x0, double x1, const mm_collision *collision, const mm_bc *bcs,
                   const mm_options *options, const double *W0, int n, double cfl, double dt,
                   double *U, int on_device, double *t_end);

#ifdef __cplusplus
}
#endif
#endif /* MM_H */
