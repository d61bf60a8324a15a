// mm_physics.cuh -- pointwise device functions of the 5-/14-moment maximum-entropy systems
// (PAPER.md = arXiv 2401.15233).  Everything is fp64 and evaluated in the paper's
// dimensionless variables (Eq 6; L272).  Written for registers: symmetric tensors are
// kept as 6 scalars, the closure is only evaluated for the components the x-flux needs, and
// powers of the pressure tensor use the Cayley-Hamilton identity instead of matrix products.
// The y direction reuses the x routines on index-swapped states (L414).
//
// The 14-moment routines are templates over the type Z of the z-odd quantities
// (u_z, P_xz, P_yz, q_z and everything derived from them): Z = double is the general path;
// Z = zero_t is the z-symmetric fast path, in which those quantities are exact compile-time
// zeros and every product with them disappears from the instruction stream.  It is selected
// only when the state and the boundary data have u_z = P_xz = P_yz = q_z = 0 exactly
// (checked on the device at mm_set_state); such a state keeps them zero for all time.
#pragma once
#ifndef MM_OPCOUNT_HOST          // csrc/opcount_host.cpp compiles this header on the host instead
#include <cuda_runtime.h>
#include <math.h>
#endif
#include <type_traits>

namespace mm {

// ------------------------------------------------------------------ exact compile-time zero
struct zero_t {};
template <class T> __host__ __device__ __forceinline__ zero_t operator*(zero_t, const T&) { return {}; }
template <class T> __host__ __device__ __forceinline__ zero_t operator*(const T&, zero_t) { return {}; }
__host__ __device__ __forceinline__ zero_t operator*(zero_t, zero_t) { return {}; }
template <class T> __host__ __device__ __forceinline__ T operator+(zero_t, const T& b) { return b; }
template <class T> __host__ __device__ __forceinline__ T operator+(const T& a, zero_t) { return a; }
__host__ __device__ __forceinline__ zero_t operator+(zero_t, zero_t) { return {}; }
template <class T> __host__ __device__ __forceinline__ T operator-(zero_t, const T& b) { return -b; }
template <class T> __host__ __device__ __forceinline__ T operator-(const T& a, zero_t) { return a; }
__host__ __device__ __forceinline__ zero_t operator-(zero_t, zero_t) { return {}; }
__host__ __device__ __forceinline__ zero_t operator-(zero_t) { return {}; }

// read / write a z-odd slot of a 14-array: nothing is touched on the zero path
template <class Z> __host__ __device__ __forceinline__ Z zget(const double& x)
{
    if constexpr (std::is_same<Z, zero_t>::value) return zero_t{}; else return x;
}
__host__ __device__ __forceinline__ void zput(double& dst, const double& v) { dst = v; }
__host__ __device__ __forceinline__ void zput(double&, zero_t) {}
__host__ __device__ __forceinline__ void zadd(double& dst, const double& v) { dst = dst + v; }
__host__ __device__ __forceinline__ void zadd(double&, zero_t) {}

// a * b + c as ONE explicitly fused operation, with the exact-zero type folded away.  Routines written with
// it produce the same bits in every kernel and instantiation they are inlined into (the compiler's own
// contraction of a * b + c depends on the surrounding code): cons2prim14 needs that, because the primitives
// mm_set_state derives from a checkpointed U must equal the ones the step kernel's tail derived from it.
template <class T> struct is_zero_t : std::false_type {};
template <> struct is_zero_t<zero_t> : std::true_type {};
template <class A, class B, class C>
__device__ __forceinline__ auto ffma(const A& a, const B& b, const C& c)
{
    if constexpr (is_zero_t<A>::value || is_zero_t<B>::value) return c;
#ifdef MM_OPCOUNT_HOST
    else if constexpr (is_zero_t<C>::value) return a * b;
    else return a * b + c;
#else
    else if constexpr (is_zero_t<C>::value) return __dmul_rn(a, b);
    else return fma(a, b, c);
#endif
}

// ------------------------------------------------------------------ reciprocal / square root
// rcp(x) ~ 1/x and fsqrt(x) ~ sqrt(x) to ~1 ulp for normal x: hardware seed (MUFU.RCP64H /
// MUFU.RSQ64H, ~20 bits) + one higher-order Newton step, branch-free (no slow-path call).
// fsqrt(x) = 0 for |x| < 1e-290; negative or NaN arguments give NaN.  rcp is only applied to
// well-scaled arguments (densities, pressures, O(1) determinants, wave-speed differences).
// -DMM_EXACT_MATH restores IEEE div/sqrt.
// dmin / dmax: one compare and one select (fmin / fmax cost six instructions for their NaN rules);
// like fmin / fmax they return the second argument when the first is NaN.
#ifdef MM_OPCOUNT_HOST
__forceinline__ double rcp(double x) { return 1.0 / x; }
__forceinline__ double fsqrt(double x) { return sqrt(x); }
__forceinline__ double fsqrt_pos(double x) { return sqrt(x); }
__forceinline__ double rsqrt_nr(double x) { return 1.0 / sqrt(x); }
__forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
#elif defined(MM_EXACT_MATH)
__device__ __forceinline__ double rcp(double x) { return 1.0 / x; }
__device__ __forceinline__ double fsqrt(double x) { return sqrt(x); }
__device__ __forceinline__ double fsqrt_pos(double x) { return sqrt(x); }
__device__ __forceinline__ double rsqrt_nr(double x) { return 1.0 / sqrt(x); }
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
#else
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
// 1/sqrt(x) for normal x > 0
__device__ __forceinline__ double rsqrt_nr(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-(x * y), y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
}
__device__ __forceinline__ double rcp(double x)
{
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double e = fma(-x, r, 1.0);          // |e| <~ 2^-20 (the seed sees the high word of x only)
    const double e2 = fma(e, e, e);            // e + e^2
    return fma(r, e2, r);                      // r (1 + e + e^2): error e^3 ~ 2^-60
}
// sqrt(x) for x known to be positive and normal (P/rho, B >= 1): no zero / subnormal guard
__device__ __forceinline__ double fsqrt_pos(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double s0 = x * y;
    const double e = fma(-s0, y, 1.0);
    return fma(s0 * e, fma(0.375, e, 0.5), s0);
}
__device__ __forceinline__ double fsqrt(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double s0 = x * y;
    const double e = fma(-s0, y, 1.0);         // 1 - x y^2, |e| <~ 2^-19
    const double pe = fma(0.375, e, 0.5);
    const double s = fma(s0 * e, pe, s0);      // x y (1 + e/2 + 3e^2/8): error ~ e^3
    // the hardware seed flushes subnormal arguments to zero (-> inf): everything below 1e-290
    // is returned as 0 (absolute error < 1e-145); negative or NaN arguments still give NaN
    return fabs(x) < 1e-290 ? 0.0 : s;
}
#endif

// Added to (or used as the floor of) square-root arguments that may be exactly zero or subnormal, so
// that the guard-free fsqrt_pos applies: sqrt(1.5e-300) = 1.2e-150 instead of 0 is far below round-off of
// the O(1) dimensionless quantities involved; negative / NaN arguments still give NaN.
// 2^-996 ~ 1.5e-300: a power of two has a zero low word, so it is an instruction immediate
#ifdef MM_OPCOUNT_HOST
static const double kTiny = 0x1p-996;
#else
constexpr double kTiny = 0x1p-996;
#endif
// max(x, kTiny) for the floored radicands (R6), decided on the high word with integer instructions: for x >= kTiny
// the signed high word is >= that of kTiny; negative, zero and subnormal x have a smaller one.  A NaN passes through
// only with its sign bit clear; the canonical NaN of CUDA arithmetic (0xFFF8000000000000, sign bit set) has a negative
// high word and comes out as kTiny -- exactly what dmax(x, kTiny) = (x > kTiny ? x : kTiny) returns for a NaN too, so
// the values are those of dmax without an FP64-pipe compare.  A failed state is therefore not detected through a
// floored radicand: the CFL reduction flags it through rho <= 0, P <= 0 or a non-finite speed from the other terms
// (C, E and the prefactor of Eq 29 carry the NaN).
#ifdef MM_OPCOUNT_HOST
__forceinline__ double floor_tiny(double x) { return dmax(x, kTiny); }
#else
__device__ __forceinline__ double floor_tiny(double x)
{
    const int hi = __double2hiint(x);
    const bool ok = hi >= 0x01b00000;                      // high word of 2^-996
    return __hiloint2double(ok ? hi : 0x01b00000, ok ? __double2loint(x) : 0);
}
#endif

// x <-> y swap of the 14 moments (primitive or conserved); an involution.
__host__ __device__ constexpr int swap_xy(int m)
{
    const int t[14] = {0, 2, 1, 3, 7, 5, 8, 4, 6, 9, 11, 10, 12, 13};
    return t[m];
}
// z-odd moments: u_z, P_xz, P_yz, q_z (a set closed under swap_xy)
__host__ __device__ constexpr bool z_odd(int m) { return m == 3 || m == 6 || m == 8 || m == 12; }

struct Params {               // per-solver constants, passed by value to the kernels
    double sigma_lim;         // L163, L512
    double ws_scale;          // k of L409
    double dx, dy, x0, y0;
    double inv_dx, inv_dy;    // 1/dx, 1/dy (CFL rate of a cell without a division)
    double inv_tau_coef;      // MM_TAU_KN: 1/tau = inv_tau_coef * rho * sqrt(8 P /(pi rho))
    double inv_tau_const;     // MM_TAU_CONST: 1/tau
    double R_gas;             // T = P/(rho R_gas): Maxwellian Dirichlet states (k_bc_table)
    int tau_model, limiter, shared_limiter, flux;
    int source_scheme;        // 0 explicit, 1 point-implicit (L348)
    int nx, ny, pitch, rows;  // padded array: rows x pitch doubles per moment, interior at (+2,+2)
    const double* ab;         // table of the functions a(P*), b(P*) of Eq 29c-d (AbTable below)
    // Literals whose low word is not zero (0.8, 0.1, ... of Eq 29, 1/3) cost two register moves per use
    // as immediates; as kernel parameters they are constant-bank operands of the FP64 instructions.
    double k08, k01, k06, k038, k035, k13;
    __host__ void set_constants() { k08 = 0.8; k01 = 0.1; k06 = 0.6; k038 = 0.38; k035 = 0.35; k13 = 1.0 / 3.0; }
};

__device__ __forceinline__ double clamp_sigma(double s, double lim)
{
    // sigma_bar = min(max(sigma, sigma_lim), 1)  (L163, L512; upper clamp: DESIGN.md R5).  Written so that
    // a NaN sigma (indefinite pressure tensor: negative radicand in Eq 21) stays NaN -- both comparisons
    // are false -- and reaches the CFL reduction's failure flag.
    const double t = s < lim ? lim : s;
    return t > 1.0 ? 1.0 : t;
}

// ------------------------------------------------------------------ limiter (L262-266)
// the limited slope itself: minmod(dm,dp) resp. symmetric van Albada dm dp (dm+dp)/(dm^2+dp^2)
__device__ __forceinline__ double limited_slope(int lim, double dm, double dp)
{
    if (!(dm * dp > 0.0)) return 0.0;
    if (lim == 1) return fabs(dm) < fabs(dp) ? dm : dp;
    return dm * dp * (dm + dp) / (dm * dm + dp * dp);     // IEEE: differences may be subnormal
}

// Shared, most stringent limiter value (L266) over a set of variables, without a division or a
// sign test per variable.  For dm dp > 0 both limiter functions are one minus a ratio,
//   minmod      2 min(|dm|,|dp|)/(|dm|+|dp|) = 1 - |dm - dp| / |dm + dp|,
//   van Albada  2 dm dp / (dm^2 + dp^2)       = 1 - (dm - dp)^2 / (dm^2 + dp^2),
// and for dm dp <= 0 that ratio is >= 1, so psi = max(0, 1 - max_k N_k / D_k) covers every case;
// a variable with dm = dp = 0 has N = D = 0 and never wins the comparison, i.e. imposes nothing
// (R14).  The running maximum is kept as a fraction and compared by cross-multiplication;
// one reciprocal per slope forms psi.  `s` = dm + dp is shared with the slope itself.
// LIM (1 minmod, 2 van Albada) is a template parameter: a run-time test inside the unrolled loop over the
// variables is if-converted by the compiler into BOTH formulas plus a select per variable.
template <int LIM>
struct PsiShared {
    double n = 0.0, d = 1.0;
    __device__ __forceinline__ void add(double dm, double dp, double s)
    {
        double nk, dk;
        if (LIM == 1) { nk = fabs(dm - dp); dk = fabs(s); }
        else { const double t = dm - dp; nk = t * t; dk = dm * dm + dp * dp; }
        if (nk * d > n * dk) { n = nk; d = dk; }
    }
    __device__ __forceinline__ double psi() const
    {
        // d = 0 or subnormal (dm = -dp, or differences below 1e-300) makes rcp NaN -> psi = 0
        const double r = n * rcp(d);
        return r < 1.0 ? 1.0 - r : 0.0;
    }
};

template <int LIM, int NV>
__device__ __forceinline__ void shared_half_slopes(const double (&Wm)[NV], const double (&Wc)[NV],
                                                   const double (&Wp)[NV], double (&h)[NV])
{
    PsiShared<LIM> pm;
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        const double dm = Wc[k] - Wm[k], dp = Wp[k] - Wc[k];
        h[k] = dm + dp;
        pm.add(dm, dp, h[k]);
    }
    const double q = 0.25 * pm.psi();
#pragma unroll
    for (int k = 0; k < NV; ++k) h[k] = q * h[k];
}

// a3: limited HALF slopes h_k of one cell along one direction from the primitives of its two neighbours
// (L262-266): h = psi (dm + dp)/4 with one shared psi (L266), or h_k = limited_slope_k / 2 per variable.
template <int NV>
__device__ __forceinline__ void half_slopes(const Params& p, const double (&Wm)[NV], const double (&Wc)[NV],
                                            const double (&Wp)[NV], double (&h)[NV])
{
    if (p.limiter == 0) {
#pragma unroll
        for (int k = 0; k < NV; ++k) h[k] = 0.0;
    } else if (p.shared_limiter) {
        if (p.limiter == 1) shared_half_slopes<1, NV>(Wm, Wc, Wp, h);
        else shared_half_slopes<2, NV>(Wm, Wc, Wp, h);
    } else {
#pragma unroll
        for (int k = 0; k < NV; ++k) h[k] = 0.5 * limited_slope(p.limiter, Wc[k] - Wm[k], Wp[k] - Wc[k]);
    }
}

// ============================================================================ 5-moment
// Eq 12 (L129-137).
__device__ __forceinline__ void cons2prim5(const double (&U)[5], double (&W)[5])
{
    double rho = U[0], u = U[1] * rcp(rho);
    double P = U[2] - rho * u * u;
    double q = U[3] - rho * u * u * u - 3.0 * u * P;
    double r = U[4] - rho * u * u * u * u - 6.0 * u * u * P - 4.0 * u * q;
    W[0] = rho; W[1] = u; W[2] = P; W[3] = q; W[4] = r;
}
__device__ __forceinline__ void prim2cons5(const double (&W)[5], double (&U)[5])
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    U[0] = rho;
    U[1] = rho * u;
    U[2] = rho * u * u + P;
    U[3] = rho * u * u * u + 3.0 * u * P + q;
    U[4] = rho * u * u * u * u + 6.0 * u * u * P + 4.0 * u * q + r;
}

// Eq 14 (L151), cancellation-free branch for b < 0 (R4).
__device__ __forceinline__ double sigma5(double qs, double rs)
{
    double b = 3.0 - rs, X = qs * qs;
    double D = fsqrt_pos(b * b + 8.0 * X + kTiny);
    return b >= 0.0 ? 0.25 * (b + D) : 2.0 * X * rcp(D - b);
}

// Eq 34-35 (L543-551): lambda*_max(q*, sigma_bar); radicand floored at 0 (R6).
struct WS5 { double E, C, Y4, inv2s; };
__device__ __forceinline__ WS5 ws5_common(double sb)
{
    WS5 w;
    double ss = fsqrt_pos(sb);
    w.C = fsqrt_pos(3.0 - 3.0 * sb + kTiny);
    w.E = 0.8 * w.C;
    double B = 5.0 - 4.0 * ss + fsqrt_pos(floor_tiny(10.0 - 16.0 * ss + 6.0 * sb));
    double Y = B + w.E * w.E - 2.0 * w.E * fsqrt_pos(B);
    w.Y4 = 4.0 * sb * sb * Y;
    w.inv2s = 0.5 * rcp(sb);
    return w;
}
__device__ __forceinline__ double ws5_lambda(const WS5& w, double sb, double qs)
{
    double rad = floor_tiny(qs * qs - 0.8 * qs * sb * w.C + w.Y4);
    return (qs + fsqrt_pos(rad)) * w.inv2s + w.E;
}

// min / max wave speed of a 5-moment state (Eqs 30, 31, 34).  ok = rho > 0 && P > 0.
__device__ __forceinline__ void wavespeed5(const Params& p, const double (&W)[5], double& lmin,
                                           double& lmax)
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    // one reciprocal square root: y = (P rho)^-1/2, c = P y, 1/P = rho y^2, 1/(rho c^4) = rho / P^2
    double y = rsqrt_nr(P * rho), c = P * y, iP = (rho * y) * y;
    double irc4 = (rho * iP) * iP;                        // 1/(rho c^4); 1/(rho c^3) = c/(rho c^4)
    double qs = q * (c * irc4), rs = r * irc4;
    double sb = clamp_sigma(sigma5(qs, rs), p.sigma_lim);
    WS5 w = ws5_common(sb);
    lmax = u + p.ws_scale * ws5_lambda(w, sb, qs) * c;
    lmin = u - p.ws_scale * ws5_lambda(w, sb, -qs) * c;
}

// Face evaluation: flux F (Eq 12 with s from Eq 15), conserved U, wave speeds.
__device__ __forceinline__ void eval_face5(const Params& p, const double (&W)[5], double (&F)[5],
                                           double (&U)[5], double& lmin, double& lmax)
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    double y = rsqrt_nr(P * rho), c = P * y, iP = (rho * y) * y;     // as in wavespeed5
    double c2 = c * c, rc3 = P * c;                                  // rho c^2 = P
    double irc4 = (rho * iP) * iP;
    double qs = q * (c * irc4), rs = r * irc4;
    double sb = clamp_sigma(sigma5(qs, rs), p.sigma_lim);
    // Eq 15 (L155): s* = q*^3/sigma^2 + (10 - 8 sqrt(sigma)) q*;  s = rho c^5 s*
    double s = rc3 * c2 * (qs * qs * qs * rcp(sb * sb) + (10.0 - 8.0 * fsqrt_pos(sb)) * qs);
    prim2cons5(W, U);
    F[0] = U[1];
    F[1] = U[2];
    F[2] = U[3];
    F[3] = U[4];
    F[4] = rho * u * u * u * u * u + 10.0 * u * u * u * P + 10.0 * u * u * q + 5.0 * u * r + s;
    WS5 w = ws5_common(sb);
    lmax = u + p.ws_scale * ws5_lambda(w, sb, qs) * c;
    lmin = u - p.ws_scale * ws5_lambda(w, sb, -qs) * c;
}

// BGK source Eq 12d-e (L135-137) times dt: adds dt*C to Un.
__device__ __forceinline__ void add_source5(const double (&W)[5], double dt_over_tau,
                                            double (&Un)[5])
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    Un[3] += dt_over_tau * (-q);
    Un[4] += dt_over_tau * (-(4.0 * u * q + r - 3.0 * P * P * rcp(rho)));
}
__device__ __forceinline__ bool cell_speed5(const Params& p, const double (&W)[5], double& sx)
{
    if (!(W[0] > 0.0) || !(W[2] > 0.0)) { sx = 0.0; return false; }
    double a, b;
    wavespeed5(p, W, a, b);
    sx = dmax(fabs(a), fabs(b));
    return true;
}

// 1/tau (L284, L474): tau = Kn L_ref (rho_ref/rho)/sqrt(8P/(pi rho)); 0 when collisionless.
__device__ __forceinline__ double inv_tau(const Params& p, double rho, double Ph)
{
    if (p.tau_model == 1) return p.inv_tau_const;
    if (p.tau_model == 2) return p.inv_tau_coef * rho * fsqrt_pos(8.0 * Ph * rcp(3.14159265358979323846 * rho));
    return 0.0;
}

// HLL (L256-258; speeds combined as in DESIGN.md R12) or Rusanov (L258) interface flux.
// cL = SR inv, cR = -SL inv, cU = SL SR inv with inv = 1/(SR - SL)
__device__ __forceinline__ double hll1(double cL, double cR, double cU, double FL, double FR,
                                       double UL, double UR)
{
    return cL * FL + (cR * FR + cU * (UR - UL));
}
template <int NM>
__device__ __forceinline__ void numflux(int flux, const double (&FL)[NM], const double (&FR)[NM],
                                        const double (&UL)[NM], const double (&UR)[NM],
                                        double lminL, double lmaxL, double lminR, double lmaxR,
                                        double (&Fh)[NM])
{
    if (flux == 1) {
        double S = fmax(fmax(fabs(lminL), fabs(lmaxL)), fmax(fabs(lminR), fabs(lmaxR)));
#pragma unroll
        for (int m = 0; m < NM; ++m) Fh[m] = 0.5 * (FL[m] + FR[m]) - 0.5 * S * (UR[m] - UL[m]);
        return;
    }
    double SL = fmin(fmin(lminL, lminR), 0.0), SR = fmax(fmax(lmaxL, lmaxR), 0.0);
    const double inv = rcp(SR - SL), cL = SR * inv, cR = -SL * inv, cU = SL * cL;
#pragma unroll
    for (int m = 0; m < NM; ++m) Fh[m] = hll1(cL, cR, cU, FL[m], FR[m], UL[m], UR[m]);
}

// =========================================================================== 14-moment
// Inverse of the conserved forms of Eq 16 (L169-181).  z-odd slots of U are not read and
// z-odd slots of W are not written when Z = zero_t.
template <class Z>
__device__ __forceinline__ void cons2prim14(const double (&U)[14], double (&W)[14])
{
    // written with the momenta m_i = rho u_i and the trace U_jj = rho u^2 + P_jj of the conserved state itself:
    //   P_ij = U_ij - m_i u_j,   q_i = U_ijj - u_i U_jj - 2 P_ij u_j,
    //   R = U_iijj - u^2 (U_jj + P_jj) - 4 u_i (P_ij u_j + q_i)
    // every multiply-add is an explicit ffma (bit-reproducible across kernels, see ffma)
    const double rho = U[0], ir = rcp(rho);
    const double mx = U[1], my = U[2];
    const Z mz = zget<Z>(U[3]);
    const double ux = mx * ir, uy = my * ir;
    const Z uz = mz * ir;
    const double Pxx = ffma(-mx, ux, U[4]), Pxy = ffma(-mx, uy, U[5]);
    const Z Pxz = ffma(-mx, uz, zget<Z>(U[6]));
    const double Pyy = ffma(-my, uy, U[7]);
    const Z Pyz = ffma(-my, uz, zget<Z>(U[8]));
    const double Pzz = ffma(-mz, uz, U[9]);
    const double e = (U[4] + U[7]) + U[9], trP = (Pxx + Pyy) + Pzz;
    const double Pux = ffma(Pxz, uz, ffma(Pxy, uy, Pxx * ux));
    const double Puy = ffma(Pyz, uz, ffma(Pyy, uy, Pxy * ux));
    const Z Puz = ffma(Pzz, uz, ffma(Pyz, uy, Pxz * ux));
    const double qx = ffma(-2.0, Pux, ffma(-ux, e, U[10]));
    const double qy = ffma(-2.0, Puy, ffma(-uy, e, U[11]));
    const Z qz = ffma(-2.0, Puz, ffma(-uz, e, zget<Z>(U[12])));
    const double u2 = ffma(uz, uz, ffma(uy, uy, ux * ux));
    const double uPq = ffma(uz, Puz + qz, ffma(uy, Puy + qy, ux * (Pux + qx)));
    const double R = ffma(-4.0, uPq, ffma(-u2, e + trP, U[13]));
    W[0] = rho; W[1] = ux; W[2] = uy; zput(W[3], uz);
    W[4] = Pxx; W[5] = Pxy; zput(W[6], Pxz); W[7] = Pyy; zput(W[8], Pyz); W[9] = Pzz;
    W[10] = qx; W[11] = qy; zput(W[12], qz); W[13] = R;
}

template <class Z>
__device__ __forceinline__ void prim2cons14(const double (&W)[14], double (&U)[14])
{
    const double rho = W[0], ux = W[1], uy = W[2];
    const Z uz = zget<Z>(W[3]);
    const double Pxx = W[4], Pxy = W[5], Pyy = W[7], Pzz = W[9];
    const Z Pxz = zget<Z>(W[6]), Pyz = zget<Z>(W[8]), qz = zget<Z>(W[12]);
    const double u2 = ux * ux + uy * uy + uz * uz, trP = Pxx + Pyy + Pzz;
    const double Pux = Pxx * ux + Pxy * uy + Pxz * uz;
    const double Puy = Pxy * ux + Pyy * uy + Pyz * uz;
    const Z Puz = Pxz * ux + Pyz * uy + Pzz * uz;
    const double e = rho * u2 + trP;
    const double rux = rho * ux, ruy = rho * uy;
    const Z ruz = rho * uz;
    U[0] = rho; U[1] = rux; U[2] = ruy; zput(U[3], ruz);
    U[4] = rux * ux + Pxx; U[5] = rux * uy + Pxy; zput(U[6], rux * uz + Pxz);
    U[7] = ruy * uy + Pyy; zput(U[8], ruy * uz + Pyz); U[9] = ruz * uz + Pzz;
    const double qx = W[10], qy = W[11];
    U[10] = ux * e + (2.0 * Pux + qx);
    U[11] = uy * e + (2.0 * Puy + qy);
    zput(U[12], uz * e + (2.0 * Puz + qz));
    // rho u^4 + 2 u^2 P_jj + 4 u_i u_j P_ij + 4 u_i q_i + R, factored
    const double uPq = ux * (Pux + qx) + uy * (Puy + qy) + uz * (Puz + qz);
    U[13] = u2 * (rho * u2 + 2.0 * trP) + (4.0 * uPq + W[13]);
}

// Dimensionless state (Eq 6, rho* = 1): c = sqrt(P/rho), P = P_ii/3, p = P_ij/P (tr p = 3),
// h = q/(rho c^3), Rs = R/(rho c^4); plus p^2, adj(p), det p, w = p^-1 h, and sigma (Eq 21).
template <class Z>
struct Star14 {
    double c, Ph;
    double pxx, pxy, pyy, pzz;               // p
    Z pxz, pyz;
    double sxx, sxy, syy, szz;               // p^2
    Z sxz, syz;
    double t2, I3;                           // tr p^2, det p
    double hx, hy, wx, wy;                   // h, w = p^-1 h
    Z hz, wz;
    double sigma;                            // Eq 21, unlimited
};

template <class Z>
__device__ __forceinline__ void nondim_sigma14(const Params& p, const double (&W)[14], Star14<Z>& s)
{
    const double rho = W[0];
    const double Ph = (W[4] + W[7] + W[9]) * p.k13;
    // one reciprocal square root serves c, 1/P and 1/(rho c^3):  y = (P rho)^-1/2, c = P y, 1/P = rho y^2
    const double y = rsqrt_nr(Ph * rho), ry = rho * y, iP = ry * y;
    const double c = Ph * y;
    s.c = c; s.Ph = Ph;
    s.pxx = W[4] * iP; s.pxy = W[5] * iP; s.pxz = zget<Z>(W[6]) * iP;
    s.pyy = W[7] * iP; s.pyz = zget<Z>(W[8]) * iP; s.pzz = W[9] * iP;
    const double ih = iP * ry;                             // 1/(rho c^3) = 1/(P c) = rho y / P
    s.hx = W[10] * ih; s.hy = W[11] * ih; s.hz = zget<Z>(W[12]) * ih;
    const double Rs = W[13] * (rho * iP) * iP;             // R/(rho c^4) = R rho / P^2
    s.sxx = s.pxx * s.pxx + s.pxy * s.pxy + s.pxz * s.pxz;
    s.sxy = s.pxx * s.pxy + s.pxy * s.pyy + s.pxz * s.pyz;
    s.sxz = s.pxx * s.pxz + s.pxy * s.pyz + s.pxz * s.pzz;
    s.syy = s.pxy * s.pxy + s.pyy * s.pyy + s.pyz * s.pyz;
    s.syz = s.pxy * s.pxz + s.pyy * s.pyz + s.pyz * s.pzz;
    s.szz = s.pxz * s.pxz + s.pyz * s.pyz + s.pzz * s.pzz;
    s.t2 = s.sxx + s.syy + s.szz;
    double X;
    if constexpr (std::is_same<Z, zero_t>::value) {
        // p = (2x2 block) (+) p_zz: w = block^-1 h, det p = p_zz det(block)
        const double d2 = s.pxx * s.pyy - s.pxy * s.pxy;
        const double id = rcp(d2);
        s.I3 = s.pzz * d2;
        s.wx = (s.pyy * s.hx - s.pxy * s.hy) * id;
        s.wy = (s.pxx * s.hy - s.pxy * s.hx) * id;
        X = s.hx * s.wx + s.hy * s.wy;
    } else {
        // adjugate (cofactors) of p and det p
        const double axx = s.pyy * s.pzz - s.pyz * s.pyz, axy = s.pxz * s.pyz - s.pxy * s.pzz;
        const double axz = s.pxy * s.pyz - s.pxz * s.pyy, ayy = s.pxx * s.pzz - s.pxz * s.pxz;
        const double ayz = s.pxy * s.pxz - s.pxx * s.pyz, azz = s.pxx * s.pyy - s.pxy * s.pxy;
        s.I3 = s.pxx * axx + s.pxy * axy + s.pxz * axz;
        const double id = rcp(s.I3);
        s.wx = (axx * s.hx + axy * s.hy + axz * s.hz) * id;
        s.wy = (axy * s.hx + ayy * s.hy + ayz * s.hz) * id;
        s.wz = (axz * s.hx + ayz * s.hy + azz * s.hz) * id;
        X = s.hx * s.wx + s.hy * s.wy + s.hz * s.wz;
    }
    // Eq 21 with P_ii P_jj = 9: sigma = [b + sqrt(b^2 + 8 t2 X)]/(4 t2), b = 2 t2 + 9 - R*,
    // X = h.p^-1.h; conjugate form when b < 0 (R4)
    const double b = 2.0 * s.t2 + 9.0 - Rs;
    const double D = fsqrt_pos(b * b + 8.0 * s.t2 * X + kTiny);       // kTiny: no zero / subnormal argument
    const bool pos = b >= 0.0;
    s.sigma = (pos ? b + D : 2.0 * X) * rcp(pos ? 4.0 * s.t2 : D - b);
}

// Quantities of Eq 29 that depend on sigma_bar only (shared by all directions of a state).
struct SbTerms { double sb, ss, isb, B, sqB; };
__device__ __forceinline__ SbTerms sb_terms(double sb)
{
    SbTerms t;
    const double y = rsqrt_nr(sb);                     // sb >= sigma_lim > 0
    t.sb = sb; t.ss = sb * y; t.isb = y * y;
    t.B = 5.0 - 4.0 * t.ss + fsqrt_pos(floor_tiny(10.0 - 16.0 * t.ss + 6.0 * sb));   // Eq 29e
    t.sqB = fsqrt_pos(t.B);
    return t;
}
// sigma_bar = clamp(sigma) and its terms.  (A warp-uniform shortcut for sigma_bar = sigma_lim -- the terms are
// constants there -- was measured and dropped: the branch splits the face evaluation into two basic blocks,
// which costs 1.5 % on near-equilibrium and on developed jet states alike, more than the skipped square roots save.)
__device__ __forceinline__ SbTerms sb_terms_clamped(const Params& p, double sigma)
{
    return sb_terms(clamp_sigma(sigma, p.sigma_lim));
}

// ---- a(P*) = 1.4 P*^1.1 exp(-P*^2) and b(P*) = 0.9 P* exp(-P*^1.4 / 2) of Eq 29c-d (L397-399)
// They depend on the single variable P* = p_dd in (0, 3) and cost a pow and two exp per call,
// six calls per cell update.  They are tabulated once per solver (k_ab_table, on the device, from
// the formulas with libm pow / exp) as degree-8 Chebyshev interpolants re-expanded in powers of
// the local coordinate t in [-1, 1], on 224 intervals read off the bits of P*: 32 per octave on
// [2^-5, 4),  [2^e (1 + j/32), 2^e (1 + (j+1)/32)),  i.e. the exponent and the top five mantissa bits
// of P* are the interval index.  The branch point P* = 0 is at least 64 half-widths from every
// interval's centre, and exp(-P*^2) varies by less than e^(+-1/4) over a half-width; the interpolation
// error is below 2e-15 relative everywhere (what remains is the round-off of 8 FMAs).
// mm_selftest_fastmath (include/mm_bench.h) measures it against the direct formulas.  Outside
// [2^-5, 4) and for NaN the direct formulas are used.
#ifndef MM_AB_SUBBITS
#define MM_AB_SUBBITS 5
#endif
struct AbTable {
    static constexpr int kSubBits = MM_AB_SUBBITS, kSub = 1 << kSubBits;        // sub-intervals per octave
    static constexpr int kOctLo = -5, kOctaves = 7;                 // [2^-5, 2^2)
    static constexpr int kIntervals = kOctaves * kSub, kDeg = 8;
    static constexpr int kStride = 2 * (kDeg + 1);                  // (a_i, b_i) pairs, highest power first
    static constexpr int kDoubles = kIntervals * kStride;
    static constexpr int kHiMin = (1023 + kOctLo) << 20;            // hi word of 2^-5 and of 4
    static constexpr int kHiMax = (1023 + kOctLo + kOctaves) << 20;
    static constexpr int kShift = 20 - kSubBits;                    // hi >> kShift = (exponent, top mantissa bits)
    // interval i: lower edge and 1 / half-width
    __host__ __device__ static double lower(int i)
    {
        const int e = kOctLo + i / kSub, j = i % kSub;
        const double two_e = e >= 0 ? (double)(1 << e) : 1.0 / (double)(1 << -e);
        return two_e * (1.0 + (double)j / kSub);
    }
    __host__ __device__ static double inv_half(int i)
    {
        const int e = kOctLo + i / kSub;                            // half-width 2^e / (2 kSub)
        return e >= 0 ? (double)(2 * kSub) / (double)(1 << e) : (double)(2 * kSub) * (double)(1 << -e);
    }
};
#ifndef MM_OPCOUNT_HOST
__device__ __noinline__ void ab_direct(double P, double* a, double* b)
{
    *a = 1.4 * pow(P, 1.1) * exp(-(P * P));
    *b = 0.9 * P * exp(-0.5 * pow(P, 1.4));
}
__device__ __forceinline__ bool ab_in_table(double P)
{
    const int hi = __double2hiint(P);
    return hi >= AbTable::kHiMin && hi < AbTable::kHiMax;
}
// table value, no branch: for P outside [2^-5, 4) the interval index is clamped and the result is NOT a(P), b(P)
// -- the caller tests ab_in_table and redoes those (rare) states with the direct formulas
__device__ __forceinline__ void ab_table(const double* __restrict__ tab, double P, double& a, double& b)
{
    const int hi = __double2hiint(P);
    const int idx = min(max((hi - AbTable::kHiMin) >> AbTable::kShift, 0), AbTable::kIntervals - 1);
    const double lo = __hiloint2double(hi & ~((1 << AbTable::kShift) - 1), 0);
    // 1 / half-width = 2^(kSubBits + 1 - e): exponent field 1023 + kSubBits + 1 - (E - 1023)
    const double ih = __hiloint2double(((2046 + AbTable::kSubBits + 1) << 20) - (hi & 0x7FF00000), 0);
    const double t = fma(P - lo, ih, -1.0);
    const double2* c = reinterpret_cast<const double2*>(tab + idx * AbTable::kStride);
    double2 q = c[0];
#pragma unroll
    for (int i = 1; i <= AbTable::kDeg; ++i) {
        const double2 ci = c[i];
        q.x = fma(q.x, t, ci.x);
        q.y = fma(q.y, t, ci.y);
    }
    a = q.x; b = q.y;
}
__device__ __forceinline__ void ab_eval(const double* __restrict__ tab, double P, double& a, double& b)
{
    if (ab_in_table(P)) ab_table(tab, P, a, b);
    else ab_direct(P, &a, &b);
}
#else
// Counted at the METHOD's operation count (pow and exp are one operation each):
// a = 1.4 P^1.1 exp(-P^2) and b = 0.9 P exp(-P^1.4 / 2) are 5 + 5 operations, whatever the kernel's table
// evaluation executes (2 x kDeg FMAs + 2) -- the roofline fraction cannot rise by adding instructions.
// g_ab_executed_flops accumulates the executed count beside it.
static long long g_ab_executed_flops = 0;
__forceinline__ void ab_eval(const double* tab, double P, double& a, double& b)
{
    (void)tab;
    a = 1.4 * pow(P, 1.1) * exp(-(P * P));
    b = 0.9 * P * exp(-0.5 * pow(P, 1.4));
    g_ab_executed_flops += 2 * 2 * AbTable::kDeg + 2 - 10;      // what the table evaluation executes beyond the 10 counted
}
#endif

// Eq 29a-e (L393-403): lambda*_max and -lambda*_min along one direction given P* = p_dd, the
// heat flux along (hd) and across (qt2 = sum of squares of the other two), sigma_bar terms.
// a(P*), b(P*) come from the table (ab_eval); Y = B + E^2 - 2 E sqrt(B)
// is evaluated as (sqrt(B) - E)^2; the radicand is floored at 0 (R6).
template <bool TABLE_ONLY = false>
__device__ __forceinline__ void ws14_dir(const Params& p, double Pdd, double hd,
                                         double qt, double qt2, const SbTerms& t, double& lam_max,
                                         double& lam_min_neg)
{
    double a, b;
#ifndef MM_OPCOUNT_HOST
    if constexpr (TABLE_ONLY) ab_table(p.ab, Pdd, a, b); else
#endif
    ab_eval(p.ab, Pdd, a, b);
    const double C = fsqrt_pos((3.0 - 3.0 * t.sb) * Pdd + kTiny);
    const double E = p.k08 * C;
    const double sY = t.sqB - E;
    const double pref = (a * t.sb + b) * (0.5 * t.isb);
    const double sC = t.sb * E;
    const double cst = 4.0 * t.sb * t.sb * (sY * sY) + p.k01 * qt2;
    const double alpha = (p.k06 * Pdd - p.k038) * Pdd + p.k035;      // Eq 29b
    const double zp = hd + alpha * qt, zm = -hd + alpha * qt;        // Eq 30: q_d -> -q_d
    const double rp = floor_tiny(zp * (zp - sC) + cst), rm = floor_tiny(zm * (zm - sC) + cst);
    lam_max = pref * (zp + fsqrt_pos(rp)) + E;
    lam_min_neg = pref * (zm + fsqrt_pos(rm)) + E;
}

// lambda_min / lambda_max along x of an (index-swapped for y) state, Eqs 28-31 (L388-411).
template <class Z, bool TABLE_ONLY = false>
__device__ __forceinline__ void wavespeed14_x(const Params& p, const Star14<Z>& s,
                                              const SbTerms& t, double ux, double& lmin, double& lmax)
{
    double a, b, qt;                                                 // Eq 28: qtilde >= 0 (R7)
    const double qt2 = s.hy * s.hy + s.hz * s.hz;
    if constexpr (std::is_same<Z, zero_t>::value) qt = fabs(s.hy); else qt = fsqrt(qt2);
    ws14_dir<TABLE_ONLY>(p, s.pxx, s.hx, qt, qt2, t, a, b);
    const double kc = p.ws_scale * s.c;
    lmax = ux + kc * a; lmin = ux - kc * b;
}
// the same along y without swapping the state: P* = p_yy, q_d = h_y, qtilde from (h_x, h_z)
template <class Z>
__device__ __forceinline__ void wavespeed14_y(const Params& p, const Star14<Z>& s,
                                              const SbTerms& t, double uy, double& lmin, double& lmax)
{
    double a, b, qt;
    const double qt2 = s.hx * s.hx + s.hz * s.hz;
    if constexpr (std::is_same<Z, zero_t>::value) qt = fabs(s.hx); else qt = fsqrt(qt2);
    ws14_dir(p, s.pyy, s.hy, qt, qt2, t, a, b);
    const double kc = p.ws_scale * s.c;
    lmax = uy + kc * a; lmin = uy - kc * b;
}

// Face evaluation along x: F = x-flux of Eq 16 (L169-181) with the closing moments Q_ijx,
// R_ixjj, S_xiijj of Eqs 22-25 (L214-230) at sigma_bar; U = conserved moments of W; the
// approximate wave speeds (Eqs 28-31).  Only what the x-flux needs is evaluated:
//   B = 2 t2 p + 4 p^3 (Eq 25a), v = B^-1 h, a = p v,
//   Q*_ijx = 2 [a_i (p^2)_jx + a_x (p^2)_ij + a_j (p^2)_ix]                       (Eqs 22, 25b)
//   T_i = Q*_ixl w_l,  R*_ix = T_i/sb + 2(1-sb)(p^2)_ix + 3 p_ix                   (Eq 23)
//   S*_x = (w.T)/sb^2 + 6 sqrt(sb) h_x + (1 - sqrt(sb)) (M v)_x                    (Eq 24)
//   M = [2*27 p + 12 t3 p + 14 t2 p^2 + 60 p^3 + 20 p^4 - 6 t2 p - 54 p^2]         (Eq 25c, tr p = 3)
// with p^3 = 3p^2 - I2 p + I3, p^4 = (9-I2)p^2 + (I3-3I2)p + 3I3 (Cayley-Hamilton, I1 = 3,
// I2 = (9 - t2)/2, I3 = det p), so M = m2 p^2 + m1 p + m0.
// The flux polynomials are written as F = u_x U + (pressure / heat-flux / closure terms).
// z-odd slots of F and U are left untouched when Z = zero_t.
// The evaluation in two parts, so that the step kernel can run part B of one face next to part A of the
// other in one basic block (the latency-bound reciprocal / square-root chains of A against the
// multiply-add-rich B):
//   A: dimensionless state, sigma, sigma_bar terms, wave speeds (Eqs 6, 21, 28-31);
//   B: closing moments, flux, conserved state (Eqs 22-25, 16).
template <class Z>
struct FaceA { Star14<Z> s; SbTerms t; };

// TABLE_ONLY: a(P*), b(P*) from the table without the range test (no branch inside the block); the caller
// must check ab_in_table(a.s.pxx) afterwards and call face14_speeds_direct where it fails.
template <class Z, bool TABLE_ONLY = false>
__device__ __forceinline__ void eval_face14_A(const Params& p, const double (&W)[14], FaceA<Z>& a,
                                              double& lmin, double& lmax)
{
    nondim_sigma14<Z>(p, W, a.s);
    a.t = sb_terms_clamped(p, a.s.sigma);
    wavespeed14_x<Z, TABLE_ONLY>(p, a.s, a.t, W[1], lmin, lmax);
}
template <class Z>
__device__ __forceinline__ void face14_speeds_direct(const Params& p, const double (&W)[14], const FaceA<Z>& a,
                                                     double& lmin, double& lmax)
{
    wavespeed14_x<Z, false>(p, a.s, a.t, W[1], lmin, lmax);
}

template <class Z>
__device__ __forceinline__ void eval_face14_B(const Params& p, const double (&W)[14], const FaceA<Z>& fa,
                                              double (&F)[14], double (&U)[14])
{
    const Star14<Z>& s = fa.s;
    const SbTerms& t = fa.t;
    const double sb = t.sb, isb = t.isb, ss = t.ss;

    // Cayley-Hamilton coefficients with I1 = tr p = 3, I2 = (9 - t2)/2, t3 = 3 t2 - 3 I2 + 3 I3 substituted:
    //   B = 12 p^2 + (4 t2 - 18) p + 4 I3 I,   M = (24 t2 + 216) p^2 + (108 t2 - 648 + 56 I3) p + 120 I3 I
    const double I3 = s.I3;
    const double bp = 4.0 * s.t2 - 18.0, b0 = 4.0 * I3;
    const double Bxx = 12.0 * s.sxx + (bp * s.pxx + b0), Bxy = 12.0 * s.sxy + bp * s.pxy;
    const double Byy = 12.0 * s.syy + (bp * s.pyy + b0);
    double vx, vy;
    Z vz;
    if constexpr (std::is_same<Z, zero_t>::value) {
        const double idB = rcp(Bxx * Byy - Bxy * Bxy);           // 2x2 block; v_z = 0
        vx = (Byy * s.hx - Bxy * s.hy) * idB;
        vy = (Bxx * s.hy - Bxy * s.hx) * idB;
    } else {
        const double Bxz = 12.0 * s.sxz + bp * s.pxz, Byz = 12.0 * s.syz + bp * s.pyz;
        const double Bzz = 12.0 * s.szz + (bp * s.pzz + b0);
        const double cxx = Byy * Bzz - Byz * Byz, cxy = Bxz * Byz - Bxy * Bzz;
        const double cxz = Bxy * Byz - Bxz * Byy, cyy = Bxx * Bzz - Bxz * Bxz;
        const double cyz = Bxy * Bxz - Bxx * Byz, czz = Bxx * Byy - Bxy * Bxy;
        const double idB = rcp(Bxx * cxx + Bxy * cxy + Bxz * cxz);
        vx = (cxx * s.hx + cxy * s.hy + cxz * s.hz) * idB;
        vy = (cxy * s.hx + cyy * s.hy + cyz * s.hz) * idB;
        vz = (cxz * s.hx + cyz * s.hy + czz * s.hz) * idB;
    }
    const double ax = s.pxx * vx + s.pxy * vy + s.pxz * vz;
    const double ay = s.pxy * vx + s.pyy * vy + s.pyz * vz;
    const Z az = s.pxz * vx + s.pyz * vy + s.pzz * vz;
    // dimensional Q_ijx = rho c^3 Q*_ijx, the scale folded into a: A = 2 rho c^3 a  (rho c^2 = P)
    const double rc3 = s.Ph * s.c, rc4 = rc3 * s.c, rc5 = rc4 * s.c, k2 = 2.0 * rc3;
    const double Ax = k2 * ax, Ay = k2 * ay;
    const Z Az = k2 * az;
    const double Qxxx = 3.0 * (Ax * s.sxx);
    const double Qxyx = 2.0 * (Ax * s.sxy) + Ay * s.sxx;
    const Z Qxzx = 2.0 * (Ax * s.sxz) + Az * s.sxx;
    const double Qyyx = 2.0 * (Ay * s.sxy) + Ax * s.syy;
    const Z Qyzx = Ay * s.sxz + Ax * s.syz + Az * s.sxy;
    const double Qzzx = 2.0 * (Az * s.sxz) + Ax * s.szz;
    // T_i = Q_ixl w_l (dimensional: rho c^3 T*)
    const double Tx = Qxxx * s.wx + Qxyx * s.wy + Qxzx * s.wz;
    const double Ty = Qxyx * s.wx + Qyyx * s.wy + Qyzx * s.wz;
    const Z Tz = Qxzx * s.wx + Qyzx * s.wy + Qzzx * s.wz;
    // R_ix = rho c^4 R*_ix = (c / sb) T_i + rho c^4 [2 (1 - sb) (p^2)_ix + 3 p_ix]                    (Eq 23)
    const double g = 2.0 - 2.0 * sb, ci = s.c * isb;
    const double Rx = ci * Tx + rc4 * (g * s.sxx + 3.0 * s.pxx);
    const double Ry = ci * Ty + rc4 * (g * s.sxy + 3.0 * s.pxy);
    const Z Rz = ci * Tz + rc4 * (g * s.sxz + 3.0 * s.pxz);
    // S_x = rho c^5 S*_x = (c / sb)^2 (w . T) + rho c^5 [6 sqrt(sb) h_x + (1 - sqrt(sb)) (M v)_x]    (Eq 24)
    const double m2 = 24.0 * s.t2 + 216.0;
    const double m1 = 108.0 * s.t2 + (56.0 * I3 - 648.0);
    const double m0 = 120.0 * I3;
    const double pax = s.pxx * ax + s.pxy * ay + s.pxz * az;          // (p^2 v)_x
    const double Mvx = m2 * pax + (m1 * ax + m0 * vx);
    const double Sx = (ci * ci) * (s.wx * Tx + s.wy * Ty + s.wz * Tz)
                    + rc5 * ((6.0 * ss) * s.hx + (1.0 - ss) * Mvx);

    prim2cons14<Z>(W, U);
    const double ux = W[1], uy = W[2];
    const Z uz = zget<Z>(W[3]);
    const double Pxx = W[4], Pxy = W[5];
    const Z Pxz = zget<Z>(W[6]);
    const double qx = W[10];
    const double u2 = ux * ux + uy * uy + uz * uz;
    const double uPx = ux * Pxx + uy * Pxy + uz * Pxz;                 // u_j P_jx
    F[0] = U[1];                                                       // 16a
    F[1] = U[4];                                                       // 16b: rho u_i u_x + P_ix = U_ix
    F[2] = U[5];
    zput(F[3], zget<Z>(U[6]));
    F[4] = ux * (U[4] + 2.0 * Pxx) + Qxxx;                             // 16c
    F[5] = ux * (U[5] + Pxy) + (uy * Pxx + Qxyx);
    zput(F[6], ux * (zget<Z>(U[6]) + Pxz) + (uz * Pxx + Qxzx));
    F[7] = ux * U[7] + ((2.0 * uy) * Pxy + Qyyx);
    zput(F[8], ux * zget<Z>(U[8]) + (uy * Pxz + uz * Pxy + Qyzx));
    F[9] = ux * U[9] + ((2.0 * uz) * Pxz + Qzzx);
    const double k1 = 2.0 * uPx + qx;                                  // 16d
    const double uQx = ux * Qxxx + uy * Qxyx + uz * Qxzx;              // u_j Q_jix
    const double uQy = ux * Qxyx + uy * Qyyx + uz * Qyzx;
    const Z uQz = ux * Qxzx + uy * Qyzx + uz * Qzzx;
    F[10] = ux * (U[10] + k1) + (u2 * Pxx + (2.0 * uQx + Rx));
    F[11] = ux * U[11] + (uy * k1 + (u2 * Pxy + (2.0 * uQy + Ry)));
    zput(F[12], ux * zget<Z>(U[12]) + (uz * k1 + (u2 * Pxz + (2.0 * uQz + Rz))));
    // 16e: u_x U_iijj + 2 u^2 (2 u_j P_jx + q_x) + 4 u_i (u_j Q_ijx + R_ix) + S_x
    F[13] = ux * U[13] + ((2.0 * u2) * k1 + (4.0 * (ux * (uQx + Rx) + uy * (uQy + Ry) + uz * (uQz + Rz)) + Sx));
}

template <class Z>
__device__ __forceinline__ void eval_face14(const Params& p, const double (&W)[14],
                                            double (&F)[14], double (&U)[14], double& lmin,
                                            double& lmax)
{
    FaceA<Z> a;
#ifndef MM_OPCOUNT_HOST
    // a(P*), b(P*) straight from the table: no branch between the wave-speed chains of part A and the
    // multiply-add-rich part B, so the two interleave; the (rare) state outside the table's range redoes
    // its wave speeds with the direct formulas afterwards
    eval_face14_A<Z, true>(p, W, a, lmin, lmax);
    eval_face14_B<Z>(p, W, a, F, U);
    if (!ab_in_table(a.s.pxx)) face14_speeds_direct<Z>(p, W, a, lmin, lmax);
    // the fallback diverges per lane (and calls a function); the step kernel's warp-collective tensor-memory
    // instructions that follow need all 32 lanes back together
    __syncwarp();
#else
    eval_face14_A<Z>(p, W, a, lmin, lmax);
    eval_face14_B<Z>(p, W, a, F, U);
#endif
}

// max(|lmin|,|lmax|) along x and y of a cell-centre state, for the CFL reduction (L434).
// ok = false when rho <= 0 or P <= 0.
template <class Z>
__device__ __forceinline__ bool cell_speeds14(const Params& p, const double (&W)[14], double& sx,
                                              double& sy)
{
    double Ph = W[4] + W[7] + W[9];
    if (!(W[0] > 0.0) || !(Ph > 0.0)) { sx = sy = 0.0; return false; }
    Star14<Z> s;
    nondim_sigma14<Z>(p, W, s);
    const SbTerms t = sb_terms_clamped(p, s.sigma);
    double a, b;
    wavespeed14_x<Z>(p, s, t, W[1], a, b);
    sx = dmax(fabs(a), fabs(b));
    wavespeed14_y<Z>(p, s, t, W[2], a, b);
    sy = dmax(fabs(a), fabs(b));
    return true;
}

// BGK source Eqs 17-18 (L185-194), times dt: Un += dt * C(W).
template <class Z>
__device__ __forceinline__ void add_source14(const double (&W)[14], double dt_over_tau,
                                             double (&Un)[14])
{
    const double rho = W[0], ux = W[1], uy = W[2];
    const Z uz = zget<Z>(W[3]);
    const double Pxx = W[4], Pxy = W[5], Pyy = W[7], Pzz = W[9];
    const Z Pxz = zget<Z>(W[6]), Pyz = zget<Z>(W[8]), qz = zget<Z>(W[12]);
    const double Ph = (Pxx + Pyy + Pzz) * (1.0 / 3.0);
    const double k = -dt_over_tau;
    Un[4] += k * (Pxx - Ph); Un[5] += k * Pxy; zadd(Un[6], k * Pxz);
    Un[7] += k * (Pyy - Ph); zadd(Un[8], k * Pyz); Un[9] += k * (Pzz - Ph);
    const double Pux = Pxx * ux + Pxy * uy + Pxz * uz;
    const double Puy = Pxy * ux + Pyy * uy + Pyz * uz;
    const Z Puz = Pxz * ux + Pyz * uy + Pzz * uz;
    Un[10] += k * (2.0 * Pux + W[10] - 2.0 * ux * Ph);
    Un[11] += k * (2.0 * Puy + W[11] - 2.0 * uy * Ph);
    zadd(Un[12], k * (2.0 * Puz + qz - 2.0 * uz * Ph));
    const double u2 = ux * ux + uy * uy + uz * uz;
    const double uPu = ux * Pux + uy * Puy + uz * Puz;
    const double uq = ux * W[10] + uy * W[11] + uz * qz;
    Un[13] += k * ((4.0 * uPu + 4.0 * uq + W[13]) - (4.0 * u2 * Ph + 15.0 * Ph * Ph * rcp(rho)));
}

}  // namespace mm
