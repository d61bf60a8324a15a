// mm_physics.cuh -- pointwise device functions of the 5-/14-moment maximum-entropy systems
// (PAPER.md = arXiv 2401.15233).  Everything is fp64 and evaluated in the paper's
// dimensionless variables (Eq 6; L272).  Written for registers: symmetric tensors are
// kept as 6 scalars, the closure is only evaluated for the components the x-flux needs, and
// powers of the pressure tensor use the Cayley-Hamilton identity instead of matrix products.
// The y direction reuses the x routines on index-swapped states (L414).
#pragma once
#ifndef MM_OPCOUNT_HOST          // csrc/opcount_host.cpp compiles this header on the host instead
#include <cuda_runtime.h>
#include <math.h>
#endif

namespace mm {

// x <-> y swap of the 14 moments (primitive or conserved); an involution.
__host__ __device__ constexpr int swap_xy(int m)
{
    const int t[14] = {0, 2, 1, 3, 7, 5, 8, 4, 6, 9, 11, 10, 12, 13};
    return t[m];
}

struct Params {               // per-solver constants, passed by value to the kernels
    double sigma_lim;         // L163, L512
    double ws_scale;          // k of L409
    double dx, dy, x0, y0;
    double inv_tau_coef;      // MM_TAU_KN: 1/tau = inv_tau_coef * rho * sqrt(8 P /(pi rho))
    double inv_tau_const;     // MM_TAU_CONST: 1/tau
    int tau_model, limiter, shared_limiter, flux;
    int nx, ny, pitch, rows;  // padded array: rows x pitch doubles per moment, interior at (+2,+2)
};

__device__ __forceinline__ double clamp_sigma(double s, double lim)
{
    // sigma_bar = min(max(sigma, sigma_lim), 1)  (L163, L512; upper clamp: DESIGN.md R5)
    return fmin(fmax(s, lim), 1.0);
}

// ------------------------------------------------------------------ limiter (L262-266)
// psi in [0,1] multiplying the central slope (dm+dp)/2.
__device__ __forceinline__ double limiter_psi(int lim, double dm, double dp)
{
    if (!(dm * dp > 0.0)) return 0.0;
    if (lim == 1) {
        double am = fabs(dm), ap = fabs(dp);
        return 2.0 * fmin(am, ap) / (am + ap);
    }
    return 2.0 * dm * dp / (dm * dm + dp * dp);
}
// the limited slope itself: minmod(dm,dp) resp. symmetric van Albada dm dp (dm+dp)/(dm^2+dp^2)
__device__ __forceinline__ double limited_slope(int lim, double dm, double dp)
{
    if (!(dm * dp > 0.0)) return 0.0;
    if (lim == 1) return fabs(dm) < fabs(dp) ? dm : dp;
    return dm * dp * (dm + dp) / (dm * dm + dp * dp);
}

// Half slopes h[k] = slope_k / 2 of one cell along one direction from its two neighbours.
template <int NM>
__device__ __forceinline__ void half_slopes(const Params& p, const double (&Wm)[NM],
                                            const double (&W0)[NM], const double (&Wp)[NM],
                                            double (&hs)[NM])
{
    if (p.limiter == 0) {
#pragma unroll
        for (int k = 0; k < NM; ++k) hs[k] = 0.0;
        return;
    }
    if (p.shared_limiter) {
        // the same, most stringent psi for all primitives (L266); dm = dp = 0 imposes nothing
        double psi = 1.0;
#pragma unroll
        for (int k = 0; k < NM; ++k) {
            double dm = W0[k] - Wm[k], dp = Wp[k] - W0[k];
            if (dm == 0.0 && dp == 0.0) continue;
            psi = fmin(psi, limiter_psi(p.limiter, dm, dp));
        }
#pragma unroll
        for (int k = 0; k < NM; ++k) {
            double dm = W0[k] - Wm[k], dp = Wp[k] - W0[k];
            hs[k] = 0.5 * (psi * (0.5 * (dm + dp)));
        }
    } else {
#pragma unroll
        for (int k = 0; k < NM; ++k)
            hs[k] = 0.5 * limited_slope(p.limiter, W0[k] - Wm[k], Wp[k] - W0[k]);
    }
}

// ============================================================================ 5-moment
// Eq 12 (L129-137).
__device__ __forceinline__ void cons2prim5(const double (&U)[5], double (&W)[5])
{
    double rho = U[0], u = U[1] / rho;
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
    double D = sqrt(b * b + 8.0 * X);
    return b >= 0.0 ? 0.25 * (b + D) : 2.0 * X / (D - b);
}

// Eq 34-35 (L543-551): lambda*_max(q*, sigma_bar); radicand floored at 0 (R6).
struct WS5 { double E, C, Y4, inv2s; };
__device__ __forceinline__ WS5 ws5_common(double sb)
{
    WS5 w;
    double ss = sqrt(sb);
    w.C = sqrt(3.0 - 3.0 * sb);
    w.E = 0.8 * w.C;
    double B = 5.0 - 4.0 * ss + sqrt(fmax(10.0 - 16.0 * ss + 6.0 * sb, 0.0));
    double Y = B + w.E * w.E - 2.0 * w.E * sqrt(B);
    w.Y4 = 4.0 * sb * sb * Y;
    w.inv2s = 0.5 / sb;
    return w;
}
__device__ __forceinline__ double ws5_lambda(const WS5& w, double sb, double qs)
{
    double rad = fmax(qs * qs - 0.8 * qs * sb * w.C + w.Y4, 0.0);
    return (qs + sqrt(rad)) * w.inv2s + w.E;
}

// min / max wave speed of a 5-moment state (Eqs 30, 31, 34).  ok = rho > 0 && P > 0.
__device__ __forceinline__ void wavespeed5(const Params& p, const double (&W)[5], double& lmin,
                                           double& lmax)
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    double c2 = P / rho, c = sqrt(c2);
    double qs = q / (rho * c2 * c), rs = r / (rho * c2 * c2);
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
    double c2 = P / rho, c = sqrt(c2);
    double rc3 = rho * c2 * c;
    double qs = q / rc3, rs = r / (rho * c2 * c2);
    double sb = clamp_sigma(sigma5(qs, rs), p.sigma_lim);
    // Eq 15 (L155): s* = q*^3/sigma^2 + (10 - 8 sqrt(sigma)) q*;  s = rho c^5 s*
    double s = rc3 * c2 * (qs * qs * qs / (sb * sb) + (10.0 - 8.0 * sqrt(sb)) * qs);
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
    Un[4] += dt_over_tau * (-(4.0 * u * q + r - 3.0 * P * P / rho));
}

// =========================================================================== 14-moment
// Inverse of the conserved forms of Eq 16 (L169-181).
__device__ __forceinline__ void cons2prim14(const double (&U)[14], double (&W)[14])
{
    double rho = U[0], ir = 1.0 / rho;
    double ux = U[1] * ir, uy = U[2] * ir, uz = U[3] * ir;
    double Pxx = U[4] - rho * ux * ux, Pxy = U[5] - rho * ux * uy, Pxz = U[6] - rho * ux * uz;
    double Pyy = U[7] - rho * uy * uy, Pyz = U[8] - rho * uy * uz, Pzz = U[9] - rho * uz * uz;
    double u2 = ux * ux + uy * uy + uz * uz, trP = Pxx + Pyy + Pzz;
    double Pux = Pxx * ux + Pxy * uy + Pxz * uz;
    double Puy = Pxy * ux + Pyy * uy + Pyz * uz;
    double Puz = Pxz * ux + Pyz * uy + Pzz * uz;
    double e = rho * u2 + trP;
    double qx = U[10] - ux * e - 2.0 * Pux;
    double qy = U[11] - uy * e - 2.0 * Puy;
    double qz = U[12] - uz * e - 2.0 * Puz;
    double uPu = ux * Pux + uy * Puy + uz * Puz, uq = ux * qx + uy * qy + uz * qz;
    double R = U[13] - rho * u2 * u2 - 2.0 * u2 * trP - 4.0 * uPu - 4.0 * uq;
    W[0] = rho; W[1] = ux; W[2] = uy; W[3] = uz;
    W[4] = Pxx; W[5] = Pxy; W[6] = Pxz; W[7] = Pyy; W[8] = Pyz; W[9] = Pzz;
    W[10] = qx; W[11] = qy; W[12] = qz; W[13] = R;
}

__device__ __forceinline__ void prim2cons14(const double (&W)[14], double (&U)[14])
{
    double rho = W[0], ux = W[1], uy = W[2], uz = W[3];
    double Pxx = W[4], Pxy = W[5], Pxz = W[6], Pyy = W[7], Pyz = W[8], Pzz = W[9];
    double u2 = ux * ux + uy * uy + uz * uz, trP = Pxx + Pyy + Pzz;
    double Pux = Pxx * ux + Pxy * uy + Pxz * uz;
    double Puy = Pxy * ux + Pyy * uy + Pyz * uz;
    double Puz = Pxz * ux + Pyz * uy + Pzz * uz;
    double e = rho * u2 + trP;
    U[0] = rho; U[1] = rho * ux; U[2] = rho * uy; U[3] = rho * uz;
    U[4] = rho * ux * ux + Pxx; U[5] = rho * ux * uy + Pxy; U[6] = rho * ux * uz + Pxz;
    U[7] = rho * uy * uy + Pyy; U[8] = rho * uy * uz + Pyz; U[9] = rho * uz * uz + Pzz;
    U[10] = ux * e + 2.0 * Pux + W[10];
    U[11] = uy * e + 2.0 * Puy + W[11];
    U[12] = uz * e + 2.0 * Puz + W[12];
    double uPu = ux * Pux + uy * Puy + uz * Puz;
    double uq = ux * W[10] + uy * W[11] + uz * W[12];
    U[13] = rho * u2 * u2 + 2.0 * u2 * trP + 4.0 * uPu + 4.0 * uq + W[13];
}

// Dimensionless state (Eq 6, rho* = 1): c = sqrt(P/rho), P = P_ii/3, p = P_ij/P (tr p = 3),
// h = q/(rho c^3), Rs = R/(rho c^4); plus p^2, adj(p), det p, w = p^-1 h, and sigma (Eq 21).
struct Star14 {
    double c, Ph;
    double pxx, pxy, pxz, pyy, pyz, pzz;     // p
    double sxx, sxy, sxz, syy, syz, szz;     // p^2
    double t2, I3;                           // tr p^2, det p
    double hx, hy, hz, wx, wy, wz;           // h, w = p^-1 h
    double sigma;                            // Eq 21, unlimited
};

__device__ __forceinline__ void nondim_sigma14(const double (&W)[14], Star14& s)
{
    double rho = W[0];
    double Ph = (W[4] + W[7] + W[9]) / 3.0;
    double iP = 1.0 / Ph, ir = 1.0 / rho;
    double c2 = Ph * ir, c = sqrt(c2);
    s.c = c; s.Ph = Ph;
    s.pxx = W[4] * iP; s.pxy = W[5] * iP; s.pxz = W[6] * iP;
    s.pyy = W[7] * iP; s.pyz = W[8] * iP; s.pzz = W[9] * iP;
    double ih = iP * (c * rho * iP);                       // 1/(rho c^3) = 1/(P c)
    s.hx = W[10] * ih; s.hy = W[11] * ih; s.hz = W[12] * ih;
    double Rs = W[13] * rho * iP * iP;                     // R/(rho c^4) = R rho / P^2
    s.sxx = s.pxx * s.pxx + s.pxy * s.pxy + s.pxz * s.pxz;
    s.sxy = s.pxx * s.pxy + s.pxy * s.pyy + s.pxz * s.pyz;
    s.sxz = s.pxx * s.pxz + s.pxy * s.pyz + s.pxz * s.pzz;
    s.syy = s.pxy * s.pxy + s.pyy * s.pyy + s.pyz * s.pyz;
    s.syz = s.pxy * s.pxz + s.pyy * s.pyz + s.pyz * s.pzz;
    s.szz = s.pxz * s.pxz + s.pyz * s.pyz + s.pzz * s.pzz;
    s.t2 = s.sxx + s.syy + s.szz;
    // adjugate (cofactors) of p and det p
    double axx = s.pyy * s.pzz - s.pyz * s.pyz, axy = s.pxz * s.pyz - s.pxy * s.pzz;
    double axz = s.pxy * s.pyz - s.pxz * s.pyy, ayy = s.pxx * s.pzz - s.pxz * s.pxz;
    double ayz = s.pxy * s.pxz - s.pxx * s.pyz, azz = s.pxx * s.pyy - s.pxy * s.pxy;
    s.I3 = s.pxx * axx + s.pxy * axy + s.pxz * axz;
    double id = 1.0 / s.I3;
    s.wx = (axx * s.hx + axy * s.hy + axz * s.hz) * id;
    s.wy = (axy * s.hx + ayy * s.hy + ayz * s.hz) * id;
    s.wz = (axz * s.hx + ayz * s.hy + azz * s.hz) * id;
    // Eq 21 with P_ii P_jj = 9: sigma = [b + sqrt(b^2 + 8 t2 X)]/(4 t2), b = 2 t2 + 9 - R*,
    // X = h.p^-1.h; conjugate form when b < 0 (R4)
    double X = s.hx * s.wx + s.hy * s.wy + s.hz * s.wz;
    double b = 2.0 * s.t2 + 9.0 - Rs;
    double D = sqrt(b * b + 8.0 * s.t2 * X);
    s.sigma = b >= 0.0 ? (b + D) / (4.0 * s.t2) : 2.0 * X / (D - b);
}

// Eq 29a-e (L393-403): Lambda(zeta) for direction x given P* = p_xx, sigma_bar, qtilde;
// a P^1.1 e^{-P^2} and P^1.4 are evaluated through one log and exp (pow-free).
struct WS14 { double pref, E, sC, cst; };
__device__ __forceinline__ WS14 ws14_common(double Pdd, double sb, double qt2)
{
    WS14 w;
    double lnP = log(Pdd);
    double a = 1.4 * exp(1.1 * lnP - Pdd * Pdd);
    double b = 0.9 * Pdd * exp(-0.5 * exp(1.4 * lnP));
    double ss = sqrt(sb);
    double C = sqrt((3.0 - 3.0 * sb) * Pdd);
    w.E = 0.8 * C;
    double B = 5.0 - 4.0 * ss + sqrt(fmax(10.0 - 16.0 * ss + 6.0 * sb, 0.0));
    double Y = B + w.E * w.E - 2.0 * w.E * sqrt(B);
    w.pref = (a * sb + b) / (2.0 * sb);
    w.sC = 0.8 * sb * C;
    w.cst = 4.0 * sb * sb * Y + 0.1 * qt2;
    return w;
}
__device__ __forceinline__ double ws14_lambda(const WS14& w, double zeta)
{
    double rad = fmax(zeta * zeta - zeta * w.sC + w.cst, 0.0);      // floored (R6)
    return w.pref * (zeta + sqrt(rad)) + w.E;
}

// lambda_min / lambda_max along x of an (index-swapped for y) state, Eqs 28-31 (L388-411).
__device__ __forceinline__ void wavespeed14_x(const Params& p, const Star14& s, double sb,
                                              double ux, double& lmin, double& lmax)
{
    double qt2 = s.hy * s.hy + s.hz * s.hz;
    double qt = sqrt(qt2);                                           // Eq 28, qtilde >= 0 (R7)
    double alpha = (0.6 * s.pxx - 0.38) * s.pxx + 0.35;              // Eq 29b
    WS14 w = ws14_common(s.pxx, sb, qt2);
    double kc = p.ws_scale * s.c;
    lmax = ux + kc * ws14_lambda(w, s.hx + alpha * qt);
    lmin = ux - kc * ws14_lambda(w, -s.hx + alpha * qt);             // Eq 30
}
// the same along y without swapping the state: P* = p_yy, q_d = h_y, qtilde from (h_x, h_z)
__device__ __forceinline__ void wavespeed14_y(const Params& p, const Star14& s, double sb,
                                              double uy, double& lmin, double& lmax)
{
    double qt2 = s.hx * s.hx + s.hz * s.hz;
    double qt = sqrt(qt2);
    double alpha = (0.6 * s.pyy - 0.38) * s.pyy + 0.35;
    WS14 w = ws14_common(s.pyy, sb, qt2);
    double kc = p.ws_scale * s.c;
    lmax = uy + kc * ws14_lambda(w, s.hy + alpha * qt);
    lmin = uy - kc * ws14_lambda(w, -s.hy + alpha * qt);
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
__device__ __forceinline__ void eval_face14(const Params& p, const double (&W)[14],
                                            double (&F)[14], double (&U)[14], double& lmin,
                                            double& lmax)
{
    Star14 s;
    nondim_sigma14(W, s);
    const double sb = clamp_sigma(s.sigma, p.sigma_lim);
    const double isb = 1.0 / sb, ss = sqrt(sb);

    const double I2 = 0.5 * (9.0 - s.t2), I3 = s.I3;
    const double t3 = 3.0 * s.t2 - 3.0 * I2 + 3.0 * I3;
    // B = 12 p^2 + (2 t2 - 4 I2) p + 4 I3 I
    const double bp = 2.0 * s.t2 - 4.0 * I2, b0 = 4.0 * I3;
    const double Bxx = 12.0 * s.sxx + bp * s.pxx + b0, Bxy = 12.0 * s.sxy + bp * s.pxy;
    const double Bxz = 12.0 * s.sxz + bp * s.pxz, Byy = 12.0 * s.syy + bp * s.pyy + b0;
    const double Byz = 12.0 * s.syz + bp * s.pyz, Bzz = 12.0 * s.szz + bp * s.pzz + b0;
    const double cxx = Byy * Bzz - Byz * Byz, cxy = Bxz * Byz - Bxy * Bzz;
    const double cxz = Bxy * Byz - Bxz * Byy, cyy = Bxx * Bzz - Bxz * Bxz;
    const double cyz = Bxy * Bxz - Bxx * Byz, czz = Bxx * Byy - Bxy * Bxy;
    const double idB = 1.0 / (Bxx * cxx + Bxy * cxy + Bxz * cxz);
    const double vx = (cxx * s.hx + cxy * s.hy + cxz * s.hz) * idB;
    const double vy = (cxy * s.hx + cyy * s.hy + cyz * s.hz) * idB;
    const double vz = (cxz * s.hx + cyz * s.hy + czz * s.hz) * idB;
    const double ax = s.pxx * vx + s.pxy * vy + s.pxz * vz;
    const double ay = s.pxy * vx + s.pyy * vy + s.pyz * vz;
    const double az = s.pxz * vx + s.pyz * vy + s.pzz * vz;
    // Q*_ijx
    const double Qxx = 6.0 * ax * s.sxx;
    const double Qxy = 2.0 * (2.0 * ax * s.sxy + ay * s.sxx);
    const double Qxz = 2.0 * (2.0 * ax * s.sxz + az * s.sxx);
    const double Qyy = 2.0 * (2.0 * ay * s.sxy + ax * s.syy);
    const double Qyz = 2.0 * (ay * s.sxz + ax * s.syz + az * s.sxy);
    const double Qzz = 2.0 * (2.0 * az * s.sxz + ax * s.szz);
    // T_i = Q*_ixl w_l
    const double Tx = Qxx * s.wx + Qxy * s.wy + Qxz * s.wz;
    const double Ty = Qxy * s.wx + Qyy * s.wy + Qyz * s.wz;
    const double Tz = Qxz * s.wx + Qyz * s.wy + Qzz * s.wz;
    const double g = 2.0 * (1.0 - sb);
    const double Rxs = Tx * isb + g * s.sxx + 3.0 * s.pxx;
    const double Rys = Ty * isb + g * s.sxy + 3.0 * s.pxy;
    const double Rzs = Tz * isb + g * s.sxz + 3.0 * s.pxz;
    const double m2 = 14.0 * s.t2 + 306.0 - 20.0 * I2;
    const double m1 = 54.0 - 6.0 * s.t2 + 12.0 * t3 - 120.0 * I2 + 20.0 * I3;
    const double m0 = 120.0 * I3;
    const double pax = s.pxx * ax + s.pxy * ay + s.pxz * az;          // (p^2 v)_x
    const double Mvx = m2 * pax + m1 * ax + m0 * vx;
    const double Sxs = (s.wx * Tx + s.wy * Ty + s.wz * Tz) * (isb * isb) + 6.0 * ss * s.hx
                     + (1.0 - ss) * Mvx;
    // re-dimensionalise: Q = rho c^3 Q*, R = rho c^4 R*, S = rho c^5 S*  (rho c^2 = P)
    const double rc3 = s.Ph * s.c, rc4 = rc3 * s.c, rc5 = rc4 * s.c;
    const double Qxxx = rc3 * Qxx, Qxyx = rc3 * Qxy, Qxzx = rc3 * Qxz;
    const double Qyyx = rc3 * Qyy, Qyzx = rc3 * Qyz, Qzzx = rc3 * Qzz;
    const double Rx = rc4 * Rxs, Ry = rc4 * Rys, Rz = rc4 * Rzs, Sx = rc5 * Sxs;

    prim2cons14(W, U);
    const double ux = W[1], uy = W[2], uz = W[3];
    const double Pxx = W[4], Pxy = W[5], Pxz = W[6];
    const double qx = W[10];
    const double u2 = ux * ux + uy * uy + uz * uz;
    const double uPx = ux * Pxx + uy * Pxy + uz * Pxz;                 // u_j P_jx
    F[0] = U[1];                                                       // 16a
    F[1] = ux * U[1] + Pxx;                                            // 16b
    F[2] = ux * U[2] + Pxy;
    F[3] = ux * U[3] + Pxz;
    F[4] = ux * U[4] + 2.0 * ux * Pxx + Qxxx;                          // 16c
    F[5] = ux * U[5] + ux * Pxy + uy * Pxx + Qxyx;
    F[6] = ux * U[6] + ux * Pxz + uz * Pxx + Qxzx;
    F[7] = ux * U[7] + 2.0 * uy * Pxy + Qyyx;
    F[8] = ux * U[8] + uy * Pxz + uz * Pxy + Qyzx;
    F[9] = ux * U[9] + 2.0 * uz * Pxz + Qzzx;
    const double k1 = 2.0 * uPx + qx;                                  // 16d
    F[10] = ux * U[10] + ux * k1 + u2 * Pxx + 2.0 * (ux * Qxxx + uy * Qxyx + uz * Qxzx) + Rx;
    F[11] = ux * U[11] + uy * k1 + u2 * Pxy + 2.0 * (ux * Qxyx + uy * Qyyx + uz * Qyzx) + Ry;
    F[12] = ux * U[12] + uz * k1 + u2 * Pxz + 2.0 * (ux * Qxzx + uy * Qyzx + uz * Qzzx) + Rz;
    const double uuQ = ux * (ux * Qxxx + 2.0 * (uy * Qxyx + uz * Qxzx))
                     + uy * (uy * Qyyx + 2.0 * uz * Qyzx) + uz * uz * Qzzx;
    F[13] = ux * U[13] + 2.0 * u2 * k1 + 4.0 * (uuQ + ux * Rx + uy * Ry + uz * Rz) + Sx;   // 16e

    wavespeed14_x(p, s, sb, ux, lmin, lmax);
}

// max(|lmin|,|lmax|) along x and y of a cell-centre state, for the CFL reduction (L434).
// ok = false when rho <= 0 or P <= 0.
__device__ __forceinline__ bool cell_speeds14(const Params& p, const double (&W)[14], double& sx,
                                              double& sy)
{
    double Ph = W[4] + W[7] + W[9];
    if (!(W[0] > 0.0) || !(Ph > 0.0)) { sx = sy = 0.0; return false; }
    Star14 s;
    nondim_sigma14(W, s);
    const double sb = clamp_sigma(s.sigma, p.sigma_lim);
    double a, b;
    wavespeed14_x(p, s, sb, W[1], a, b);
    sx = fmax(fabs(a), fabs(b));
    wavespeed14_y(p, s, sb, W[2], a, b);
    sy = fmax(fabs(a), fabs(b));
    return true;
}
__device__ __forceinline__ bool cell_speed5(const Params& p, const double (&W)[5], double& sx)
{
    if (!(W[0] > 0.0) || !(W[2] > 0.0)) { sx = 0.0; return false; }
    double a, b;
    wavespeed5(p, W, a, b);
    sx = fmax(fabs(a), fabs(b));
    return true;
}

// 1/tau (L284, L474): tau = Kn L_ref (rho_ref/rho)/sqrt(8P/(pi rho)); 0 when collisionless.
__device__ __forceinline__ double inv_tau(const Params& p, double rho, double Ph)
{
    if (p.tau_model == 1) return p.inv_tau_const;
    if (p.tau_model == 2) return p.inv_tau_coef * rho * sqrt(8.0 * Ph / (3.14159265358979323846 * rho));
    return 0.0;
}

// BGK source Eqs 17-18 (L185-194), times dt: Un += dt * C(W).
__device__ __forceinline__ void add_source14(const double (&W)[14], double dt_over_tau,
                                             double (&Un)[14])
{
    const double rho = W[0], ux = W[1], uy = W[2], uz = W[3];
    const double Pxx = W[4], Pxy = W[5], Pxz = W[6], Pyy = W[7], Pyz = W[8], Pzz = W[9];
    const double Ph = (Pxx + Pyy + Pzz) / 3.0;
    const double k = -dt_over_tau;
    Un[4] += k * (Pxx - Ph); Un[5] += k * Pxy; Un[6] += k * Pxz;
    Un[7] += k * (Pyy - Ph); Un[8] += k * Pyz; Un[9] += k * (Pzz - Ph);
    const double Pux = Pxx * ux + Pxy * uy + Pxz * uz;
    const double Puy = Pxy * ux + Pyy * uy + Pyz * uz;
    const double Puz = Pxz * ux + Pyz * uy + Pzz * uz;
    Un[10] += k * (2.0 * Pux + W[10] - 2.0 * ux * Ph);
    Un[11] += k * (2.0 * Puy + W[11] - 2.0 * uy * Ph);
    Un[12] += k * (2.0 * Puz + W[12] - 2.0 * uz * Ph);
    const double u2 = ux * ux + uy * uy + uz * uz;
    const double uPu = ux * Pux + uy * Puy + uz * Puz;
    const double uq = ux * W[10] + uy * W[11] + uz * W[12];
    Un[13] += k * ((4.0 * uPu + 4.0 * uq + W[13]) - (4.0 * u2 * Ph + 15.0 * Ph * Ph / rho));
}

// HLL (L256-258; speeds combined as in DESIGN.md R12) or Rusanov (L258) interface flux.
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
    double inv = 1.0 / (SR - SL), SLR = SL * SR;
#pragma unroll
    for (int m = 0; m < NM; ++m)
        Fh[m] = (SR * FL[m] - SL * FR[m] + SLR * (UR[m] - UL[m])) * inv;
}

}  // namespace mm
