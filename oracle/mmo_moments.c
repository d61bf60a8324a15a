/*
 * mmo_moments.c -- CPU ORACLE (test infrastructure, not the product; see mmo.h).
 * Pointwise physics of the 5- and 14-moment maximum-entropy systems: conserved <-> primitive
 * maps, interpolative closure, physical fluxes, approximate wave speeds, BGK sources.
 * Written from PAPER.md equation by equation; loops over tensor indices instead of expanded
 * component formulas so each line can be checked against the paper by eye.
 * Compile with -O2 -ffp-contract=off (no fused multiply-add, no reassociation).
 */
#include "mmo.h"
#include <math.h>

/* position of the symmetric pair (i,j) inside the 6-vector (xx,xy,xz,yy,yz,zz) */
static const int SYM[3][3] = { {0, 1, 2}, {1, 3, 4}, {2, 4, 5} };

/* ===================================================================== 5-moment system */

/* Eq 12 (L129-137), conserved forms:
 *   U0 = rho, U1 = rho u, U2 = rho u^2 + P, U3 = rho u^3 + 3uP + q,
 *   U4 = rho u^4 + 6u^2 P + 4uq + r. */
void mmo_prim2cons5(const double W[5], double U[5])
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    U[0] = rho;
    U[1] = rho * u;
    U[2] = rho * u * u + P;
    U[3] = rho * u * u * u + 3.0 * u * P + q;
    U[4] = rho * u * u * u * u + 6.0 * u * u * P + 4.0 * u * q + r;
}

void mmo_cons2prim5(const double U[5], double W[5])
{
    double rho = U[0];
    double u = U[1] / rho;
    double P = U[2] - rho * u * u;
    double q = U[3] - rho * u * u * u - 3.0 * u * P;
    double r = U[4] - rho * u * u * u * u - 6.0 * u * u * P - 4.0 * u * q;
    W[0] = rho; W[1] = u; W[2] = P; W[3] = q; W[4] = r;
}

/* Eq 14 (L151): sigma = (1/4) [ 3 - r* + sqrt((3 - r*)^2 + 8 q*^2) ].
 * Reading R4: for b = 3 - r* < 0 the algebraically identical conjugate form
 * sigma = 2 q*^2 / (sqrt(b^2 + 8 q*^2) - b) is used (no cancellation near the Junk line). */
double mmo_sigma5(double qstar, double rstar)
{
    double b = 3.0 - rstar;
    double X = qstar * qstar;
    double D = sqrt(b * b + 8.0 * X);
    if (b >= 0.0) return 0.25 * (b + D);
    return 2.0 * X / (D - b);
}

/* Eq 15 (L155).  The printed "s" is dimensionless (reading R1). */
double mmo_sstar5(double qstar, double sigma_bar)
{
    return qstar * qstar * qstar / (sigma_bar * sigma_bar)
         + (10.0 - 8.0 * sqrt(sigma_bar)) * qstar;
}

static double clamp_sigma(double sigma, double sigma_lim)
{
    /* sigma_bar = max(sigma, sigma_lim) (L163, L512); upper clamp at the realizability
     * boundary sigma = 1 (reading R5). */
    double sb = sigma;
    if (sb < sigma_lim) sb = sigma_lim;
    if (sb > 1.0) sb = 1.0;
    return sb;
}

/* Non-dimensionalisation of Eq 6 (L75-81) for the 1D1V gas: c = sqrt(P/rho),
 * q* = q/(rho c^3), r* = r/(rho c^4); s = rho c^5 s*. */
double mmo_closure5(const double W[5], double sigma_lim, double *sigma, double *sigma_bar)
{
    double rho = W[0], P = W[2], q = W[3], r = W[4];
    double c = sqrt(P / rho);
    double qstar = q / (rho * c * c * c);
    double rstar = r / (rho * c * c * c * c);
    double sg = mmo_sigma5(qstar, rstar);
    double sb = clamp_sigma(sg, sigma_lim);
    if (sigma) *sigma = sg;
    if (sigma_bar) *sigma_bar = sb;
    return rho * c * c * c * c * c * mmo_sstar5(qstar, sb);
}

/* Fluxes of Eq 12a-e (L129-137). */
void mmo_flux5_given_s(const double W[5], double s, double F[5])
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    F[0] = rho * u;
    F[1] = rho * u * u + P;
    F[2] = rho * u * u * u + 3.0 * u * P + q;
    F[3] = rho * u * u * u * u + 6.0 * u * u * P + 4.0 * u * q + r;
    F[4] = rho * u * u * u * u * u + 10.0 * u * u * u * P + 10.0 * u * u * q + 5.0 * u * r + s;
}

void mmo_flux5(const double W[5], double sigma_lim, double F[5])
{
    double s = mmo_closure5(W, sigma_lim, 0, 0);
    mmo_flux5_given_s(W, s, F);
}

/* Eq 34 (L543) with Eq 35 (L547-551):
 *   lambda*max = (1/(2 sigma)) [ q* + sqrt(q*^2 - (4/5) q* sigma C + 4 sigma^2 Y) ] + E,
 *   E = (8/10) sqrt(3 - 3 sigma), C = sqrt(3 - 3 sigma),
 *   B = 5 - 4 sqrt(sigma) + sqrt(10 - 16 sqrt(sigma) + 6 sigma), Y = B + E^2 - 2 E sqrt(B).
 * Radicand floored at 0 (reading R6). */
static double lambda5_star(double qstar, double sb)
{
    double E = 0.8 * sqrt(3.0 - 3.0 * sb);
    double C = sqrt(3.0 - 3.0 * sb);
    double B = 5.0 - 4.0 * sqrt(sb) + sqrt(10.0 - 16.0 * sqrt(sb) + 6.0 * sb);
    double Y = B + E * E - 2.0 * E * sqrt(B);
    double rad = qstar * qstar - 0.8 * qstar * sb * C + 4.0 * sb * sb * Y;
    if (rad < 0.0) rad = 0.0;
    return (qstar + sqrt(rad)) / (2.0 * sb) + E;
}

/* lambda_min* = -lambda_max*(-q*) (Eq 30 L407 / Eq 44; L600 is a typo, reading R8);
 * inflation k (L409); lambda = u + lambda* sqrt(P/rho) (Eq 31). */
void mmo_wavespeed5(const double W[5], double sigma_lim, double k, double *lmin, double *lmax)
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    double c = sqrt(P / rho);
    double qstar = q / (rho * c * c * c);
    double rstar = r / (rho * c * c * c * c);
    double sb = clamp_sigma(mmo_sigma5(qstar, rstar), sigma_lim);
    double lmax_star = lambda5_star(qstar, sb);
    double lmin_star = -lambda5_star(-qstar, sb);
    *lmax = u + k * lmax_star * c;
    *lmin = u + k * lmin_star * c;
}

/* Eq 12d-e right-hand sides (L135-137): C = (0, 0, 0, -q/tau, -(4uq + r - 3P^2/rho)/tau). */
void mmo_source5(const double W[5], double tau, double C[5])
{
    double rho = W[0], u = W[1], P = W[2], q = W[3], r = W[4];
    C[0] = 0.0; C[1] = 0.0; C[2] = 0.0;
    C[3] = -q / tau;
    C[4] = -(4.0 * u * q + r - 3.0 * P * P / rho) / tau;
}

/* ==================================================================== 14-moment system */

static void unpack14(const double W[14], double *rho, double u[3], double P[3][3], double q[3],
                     double *R)
{
    *rho = W[0];
    for (int i = 0; i < 3; ++i) u[i] = W[1 + i];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) P[i][j] = W[4 + SYM[i][j]];
    for (int i = 0; i < 3; ++i) q[i] = W[10 + i];
    *R = W[13];
}

/* Conserved forms of Eq 16 (time-derivative arguments, L169-181):
 *   rho; rho u_i; rho u_i u_j + P_ij; rho u_i u^2 + u_i P_jj + 2 u_j P_ij + Q_ijj;
 *   rho u^4 + 2 u^2 P_jj + 4 u_i u_j P_ij + 4 u_i Q_ijj + R_iijj. */
void mmo_prim2cons14(const double W[14], double U[14])
{
    double rho, u[3], P[3][3], q[3], R;
    unpack14(W, &rho, u, P, q, &R);
    double u2 = 0.0, trP = 0.0, uPu = 0.0, uq = 0.0;
    for (int i = 0; i < 3; ++i) { u2 += u[i] * u[i]; trP += P[i][i]; uq += u[i] * q[i]; }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) uPu += u[i] * u[j] * P[i][j];
    U[0] = rho;
    for (int i = 0; i < 3; ++i) U[1 + i] = rho * u[i];
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j) U[4 + SYM[i][j]] = rho * u[i] * u[j] + P[i][j];
    for (int i = 0; i < 3; ++i) {
        double Pu = 0.0;
        for (int j = 0; j < 3; ++j) Pu += u[j] * P[i][j];
        U[10 + i] = rho * u[i] * u2 + u[i] * trP + 2.0 * Pu + q[i];
    }
    U[13] = rho * u2 * u2 + 2.0 * u2 * trP + 4.0 * uPu + 4.0 * uq + R;
}

void mmo_cons2prim14(const double U[14], double W[14])
{
    double rho = U[0], u[3], P[3][3], q[3];
    for (int i = 0; i < 3; ++i) u[i] = U[1 + i] / rho;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) P[i][j] = U[4 + SYM[i][j]] - rho * u[i] * u[j];
    double u2 = 0.0, trP = 0.0, uPu = 0.0, uq = 0.0;
    for (int i = 0; i < 3; ++i) { u2 += u[i] * u[i]; trP += P[i][i]; }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) uPu += u[i] * u[j] * P[i][j];
    for (int i = 0; i < 3; ++i) {
        double Pu = 0.0;
        for (int j = 0; j < 3; ++j) Pu += u[j] * P[i][j];
        q[i] = U[10 + i] - rho * u[i] * u2 - u[i] * trP - 2.0 * Pu;
        uq += u[i] * q[i];
    }
    double R = U[13] - rho * u2 * u2 - 2.0 * u2 * trP - 4.0 * uPu - 4.0 * uq;
    W[0] = rho;
    for (int i = 0; i < 3; ++i) W[1 + i] = u[i];
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j) W[4 + SYM[i][j]] = P[i][j];
    for (int i = 0; i < 3; ++i) W[10 + i] = q[i];
    W[13] = R;
}

/* --- small dense 3x3 helpers (plain definitions) --- */
static void matmul3(const double A[3][3], const double B[3][3], double C[3][3])
{
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double s = 0.0;
            for (int k = 0; k < 3; ++k) s += A[i][k] * B[k][j];
            C[i][j] = s;
        }
}
static void matvec3(const double A[3][3], const double x[3], double y[3])
{
    for (int i = 0; i < 3; ++i) {
        double s = 0.0;
        for (int k = 0; k < 3; ++k) s += A[i][k] * x[k];
        y[i] = s;
    }
}
static double trace3(const double A[3][3]) { return A[0][0] + A[1][1] + A[2][2]; }
/* inverse by the adjugate (cofactor) formula */
static void inverse3(const double A[3][3], double Ai[3][3])
{
    double c00 = A[1][1] * A[2][2] - A[1][2] * A[2][1];
    double c01 = A[1][2] * A[2][0] - A[1][0] * A[2][2];
    double c02 = A[1][0] * A[2][1] - A[1][1] * A[2][0];
    double det = A[0][0] * c00 + A[0][1] * c01 + A[0][2] * c02;
    Ai[0][0] = c00 / det;
    Ai[1][0] = c01 / det;
    Ai[2][0] = c02 / det;
    Ai[0][1] = (A[0][2] * A[2][1] - A[0][1] * A[2][2]) / det;
    Ai[1][1] = (A[0][0] * A[2][2] - A[0][2] * A[2][0]) / det;
    Ai[2][1] = (A[0][1] * A[2][0] - A[0][0] * A[2][1]) / det;
    Ai[0][2] = (A[0][1] * A[1][2] - A[0][2] * A[1][1]) / det;
    Ai[1][2] = (A[0][2] * A[1][0] - A[0][0] * A[1][2]) / det;
    Ai[2][2] = (A[0][0] * A[1][1] - A[0][1] * A[1][0]) / det;
}

/* Dimensionless variables of Eq 6 (L75-81) with rho* = 1:
 *   c = sqrt(P/rho), P = P_ii/3;  p_ij = P_ij/P;  h_i = q_i/(rho c^3);  Rs = R/(rho c^4). */
typedef struct { double rho, c, p[3][3], h[3], Rs; } star14;

static void nondim14(const double W[14], star14 *s)
{
    double u[3], P[3][3], q[3], R;
    unpack14(W, &s->rho, u, P, q, &R);
    double Ph = (P[0][0] + P[1][1] + P[2][2]) / 3.0;
    s->c = sqrt(Ph / s->rho);
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) s->p[i][j] = P[i][j] / Ph;
    double rc3 = s->rho * s->c * s->c * s->c;
    for (int i = 0; i < 3; ++i) s->h[i] = q[i] / rc3;
    s->Rs = R / (rc3 * s->c);
}

/* Eq 21 (L210) with rho* = 1, P_ii P_jj = 9, t2 = P_ij P_ji:
 *   sigma = [ b + sqrt(b^2 + 8 t2 X) ] / (4 t2),  b = 2 t2 + 9 - R*,  X = h.(p^-1 h).
 * Reading R4: conjugate form 2X/(sqrt(.) - b) when b < 0. */
static double sigma14_star(const star14 *s)
{
    double p2[3][3], pinv[3][3], w[3];
    matmul3(s->p, s->p, p2);
    double t2 = trace3(p2);
    inverse3(s->p, pinv);
    matvec3(pinv, s->h, w);
    double X = s->h[0] * w[0] + s->h[1] * w[1] + s->h[2] * w[2];
    double b = 2.0 * t2 + 9.0 - s->Rs;
    double D = sqrt(b * b + 8.0 * t2 * X);
    if (b >= 0.0) return (b + D) / (4.0 * t2);
    return 2.0 * X / (D - b);
}

double mmo_sigma14(const double W[14])
{
    star14 s;
    nondim14(W, &s);
    return sigma14_star(&s);
}

void mmo_closure14(const double W[14], double sigma_lim, double *sigma, double *sigma_bar,
                   double Q[3][3][3], double R2[3][3], double S[3])
{
    star14 s;
    nondim14(W, &s);
    double sg = sigma14_star(&s);
    double sb = clamp_sigma(sg, sigma_lim);
    if (sigma) *sigma = sg;
    if (sigma_bar) *sigma_bar = sb;

    double p2[3][3], p3[3][3], p4[3][3], pinv[3][3];
    matmul3(s.p, s.p, p2);
    matmul3(p2, s.p, p3);
    matmul3(p3, s.p, p4);
    inverse3(s.p, pinv);
    double t1 = trace3(s.p);         /* P_aa  (= 3)  */
    double t2 = trace3(p2);          /* (P^2)_aa     */
    double t3 = trace3(p3);          /* (P^3)_aa     */

    /* Eq 25a (L226): B_lm = 2 P_lm (P^2)_aa + 4 (P^3)_lm */
    double B[3][3], Binv[3][3];
    for (int l = 0; l < 3; ++l)
        for (int m = 0; m < 3; ++m) B[l][m] = 2.0 * s.p[l][m] * t2 + 4.0 * p3[l][m];
    inverse3(B, Binv);

    /* Eq 25b (L228): K_ijkm = [2 P_il (P^2)_jk + 2 P_kl (P^2)_ij + 2 P_jl (P^2)_ik] B^-1_lm
     * Eq 22  (L214): Q_ijk = K_ijkm Q_mnn */
    double Qs[3][3][3];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j)
            for (int k = 0; k < 3; ++k) {
                double acc = 0.0;
                for (int m = 0; m < 3; ++m) {
                    double K = 0.0;
                    for (int l = 0; l < 3; ++l)
                        K += (2.0 * s.p[i][l] * p2[j][k] + 2.0 * s.p[k][l] * p2[i][j]
                              + 2.0 * s.p[j][l] * p2[i][k]) * Binv[l][m];
                    acc += K * s.h[m];
                }
                Qs[i][j][k] = acc;
            }

    /* Eq 23 (L218): R_ijkk = (1/sigma) Q_ijl (P^-1)_lm Q_mkk
     *                        + [2 (1 - sigma) P_ik P_kj + P_ij P_kk] / rho */
    double w[3];
    matvec3(pinv, s.h, w);
    double Rs2[3][3];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) {
            double acc = 0.0;
            for (int l = 0; l < 3; ++l) acc += Qs[i][j][l] * w[l];
            Rs2[i][j] = acc / sb + 2.0 * (1.0 - sb) * p2[i][j] + s.p[i][j] * t1;
        }

    /* Eq 25c (L230): W_im = (1/rho) [ 2 P_il (P_aa)^3 + 12 P_il (P^3)_aa + 14 (P^2)_aa (P^2)_il
     *   + 20 P_aa (P^3)_il + 20 (P^4)_il - 2 (P^2)_aa P_bb P_il - 6 (P_aa)^2 (P^2)_il ] B^-1_lm */
    double M[3][3], Wm[3][3];
    for (int i = 0; i < 3; ++i)
        for (int l = 0; l < 3; ++l)
            M[i][l] = 2.0 * s.p[i][l] * t1 * t1 * t1 + 12.0 * s.p[i][l] * t3
                    + 14.0 * t2 * p2[i][l] + 20.0 * t1 * p3[i][l] + 20.0 * p4[i][l]
                    - 2.0 * t2 * t1 * s.p[i][l] - 6.0 * t1 * t1 * p2[i][l];
    matmul3(M, Binv, Wm);

    /* Eq 24 (L222): S_ijjkk = (1/sigma^2) P^-1_kn P^-1_lm Q_npp Q_mjj Q_ikl
     *                         + 2 sigma^(1/2) P_jj Q_ikk / rho + (1 - sigma^(1/2)) W_im Q_mnn */
    double Ss[3], Wh[3];
    matvec3(Wm, s.h, Wh);
    double sqs = sqrt(sb);
    for (int i = 0; i < 3; ++i) {
        double acc = 0.0;
        for (int k = 0; k < 3; ++k)
            for (int l = 0; l < 3; ++l) acc += w[k] * w[l] * Qs[i][k][l];
        Ss[i] = acc / (sb * sb) + 2.0 * sqs * t1 * s.h[i] + (1.0 - sqs) * Wh[i];
    }

    /* re-dimensionalise (Eq 6): Q = rho c^3 Q*, R = rho c^4 R*, S = rho c^5 S* */
    double rc3 = s.rho * s.c * s.c * s.c, rc4 = rc3 * s.c, rc5 = rc4 * s.c;
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 3; ++j) {
            for (int k = 0; k < 3; ++k) Q[i][j][k] = rc3 * Qs[i][j][k];
            R2[i][j] = rc4 * Rs2[i][j];
        }
        S[i] = rc5 * Ss[i];
    }
}

/* Flux of Eq 16 in direction k (the argument of d/dx_k; the line "+ u_i Q_kjj ..." of 16d
 * belongs inside the bracket, reading R2).  Q_kjj = q_k, Q_ijj = q_i. */
void mmo_flux14_given_closure(const double W[14], const double Q[3][3][3],
                              const double R2[3][3], const double S[3], int k, double F[14])
{
    double rho, u[3], P[3][3], q[3], R;
    unpack14(W, &rho, u, P, q, &R);
    double u2 = 0.0, trP = 0.0;
    for (int i = 0; i < 3; ++i) { u2 += u[i] * u[i]; trP += P[i][i]; }

    /* 16a */
    F[0] = rho * u[k];
    /* 16b */
    for (int i = 0; i < 3; ++i) F[1 + i] = rho * u[i] * u[k] + P[i][k];
    /* 16c */
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j)
            F[4 + SYM[i][j]] = rho * u[i] * u[j] * u[k] + u[i] * P[j][k] + u[j] * P[i][k]
                             + u[k] * P[i][j] + Q[i][j][k];
    /* 16d: rho u_i u_k u_j u_j + u_i u_k P_jj + 2 u_i u_j P_jk + 2 u_j u_k P_ij + u_j u_j P_ik
     *      + u_i Q_kjj + u_k Q_ijj + 2 u_j Q_ijk + R_ikjj */
    for (int i = 0; i < 3; ++i) {
        double a = 0.0, b = 0.0, c = 0.0;
        for (int j = 0; j < 3; ++j) {
            a += u[j] * P[j][k];
            b += u[j] * P[i][j];
            c += u[j] * Q[i][j][k];
        }
        F[10 + i] = rho * u[i] * u[k] * u2 + u[i] * u[k] * trP + 2.0 * u[i] * a
                  + 2.0 * u[k] * b + u2 * P[i][k] + u[i] * q[k] + u[k] * q[i] + 2.0 * c
                  + R2[i][k];
    }
    /* 16e: rho u_k u^4 + 2 u_k u^2 P_jj + 4 u^2 u_j P_jk + 4 u_i u_j u_k P_ij + 2 u^2 Q_kjj
     *      + 4 u_i u_k Q_ijj + 4 u_i u_j Q_ijk + 4 u_i R_ikjj + u_k R_iijj + S_kiijj */
    {
        double a = 0.0, b = 0.0, c = 0.0, d = 0.0, e = 0.0;
        for (int j = 0; j < 3; ++j) a += u[j] * P[j][k];
        for (int i = 0; i < 3; ++i) {
            c += u[i] * q[i];
            e += u[i] * R2[i][k];
            for (int j = 0; j < 3; ++j) {
                b += u[i] * u[j] * P[i][j];
                d += u[i] * u[j] * Q[i][j][k];
            }
        }
        F[13] = rho * u[k] * u2 * u2 + 2.0 * u[k] * u2 * trP + 4.0 * u2 * a + 4.0 * u[k] * b
              + 2.0 * u2 * q[k] + 4.0 * u[k] * c + 4.0 * d + 4.0 * e + u[k] * R + S[k];
    }
}

void mmo_flux14(const double W[14], int k, double sigma_lim, double F[14])
{
    double Q[3][3][3], R2[3][3], S[3];
    mmo_closure14(W, sigma_lim, 0, 0, Q, R2, S);
    mmo_flux14_given_closure(W, Q, R2, S, k, F);
}

/* Eq 29a-e (L393-403) = Eq 43a-e (L632-643):
 *   lambda*max = (a sigma + b)/(2 sigma) [ zeta + sqrt(zeta^2 - (4/5) zeta sigma C
 *                                         + 4 sigma^2 Y + qtilde^2/10) ] + E
 *   zeta = q_d* + sqrt(qtilde^2) (0.6 Pdd^2 - 0.38 Pdd + 0.35)
 *   a = 1.4 Pdd^1.1 exp(-Pdd^2),  b = 0.9 Pdd exp(-(1/2) Pdd^1.4)
 *   E = (8/10) sqrt((3 - 3 sigma) Pdd),  C = sqrt((3 - 3 sigma) Pdd)
 *   B = 5 - 4 sqrt(sigma) + sqrt(10 - 16 sqrt(sigma) + 6 sigma),  Y = B + E^2 - 2 E sqrt(B)
 * sqrt(qtilde^2) = qtilde >= 0 (reading R7); radicand floored at 0 (reading R6). */
double mmo_wavespeed14_star(double Pdd, double qd, double qtilde, double sb)
{
    double zeta = qd + sqrt(qtilde * qtilde) * (0.6 * Pdd * Pdd - 0.38 * Pdd + 0.35);
    double a = 1.4 * pow(Pdd, 1.1) * exp(-Pdd * Pdd);
    double b = 0.9 * Pdd * exp(-0.5 * pow(Pdd, 1.4));
    double E = 0.8 * sqrt((3.0 - 3.0 * sb) * Pdd);
    double C = sqrt((3.0 - 3.0 * sb) * Pdd);
    double B = 5.0 - 4.0 * sqrt(sb) + sqrt(10.0 - 16.0 * sqrt(sb) + 6.0 * sb);
    double Y = B + E * E - 2.0 * E * sqrt(B);
    double rad = zeta * zeta - 0.8 * zeta * sb * C + 4.0 * sb * sb * Y + qtilde * qtilde / 10.0;
    if (rad < 0.0) rad = 0.0;
    return (a * sb + b) / (2.0 * sb) * (zeta + sqrt(rad)) + E;
}

/* Eqs 28-31 for direction d (L388-414): qtilde = sqrt of the two other q*^2 (Eq 28);
 * lambda_min* = -lambda_max*(-q_d*) (Eq 30); inflation k (L409);
 * lambda = u_d + lambda* sqrt(P/rho) (Eq 31). */
void mmo_wavespeed14(const double W[14], int d, double sigma_lim, double k,
                     double *lmin, double *lmax)
{
    star14 s;
    nondim14(W, &s);
    double sb = clamp_sigma(sigma14_star(&s), sigma_lim);
    int e = (d + 1) % 3, f = (d + 2) % 3;
    double qtilde = sqrt(s.h[e] * s.h[e] + s.h[f] * s.h[f]);
    double Pdd = s.p[d][d];
    double lmax_star = mmo_wavespeed14_star(Pdd, s.h[d], qtilde, sb);
    double lmin_star = -mmo_wavespeed14_star(Pdd, -s.h[d], qtilde, sb);
    double ud = W[1 + d];
    *lmax = ud + k * lmax_star * s.c;
    *lmin = ud + k * lmin_star * s.c;
}

/* Eq 17 (L185-186): C_1 = 0, C_i = 0, C_ij = -(P_ij - P delta_ij)/tau;
 * Eq 18a (L190): C_ijj = -(2 u_j P_ij + Q_ijj - 2 u_i P)/tau;
 * Eq 18b (L193): C_iijj = -[(4 u_i u_j P_ij + 4 u_i Q_ijj + R_iijj) - (4 |u|^2 P + 15 P^2/rho)]/tau */
void mmo_source14(const double W[14], double tau, double C[14])
{
    double rho, u[3], P[3][3], q[3], R;
    unpack14(W, &rho, u, P, q, &R);
    double Ph = (P[0][0] + P[1][1] + P[2][2]) / 3.0;
    double u2 = 0.0, uPu = 0.0, uq = 0.0;
    for (int i = 0; i < 3; ++i) { u2 += u[i] * u[i]; uq += u[i] * q[i]; }
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) uPu += u[i] * u[j] * P[i][j];
    C[0] = 0.0;
    for (int i = 0; i < 3; ++i) C[1 + i] = 0.0;
    for (int i = 0; i < 3; ++i)
        for (int j = i; j < 3; ++j)
            C[4 + SYM[i][j]] = -(P[i][j] - (i == j ? Ph : 0.0)) / tau;
    for (int i = 0; i < 3; ++i) {
        double Pu = 0.0;
        for (int j = 0; j < 3; ++j) Pu += u[j] * P[i][j];
        C[10 + i] = -(2.0 * Pu + q[i] - 2.0 * u[i] * Ph) / tau;
    }
    C[13] = -((4.0 * uPu + 4.0 * uq + R) - (4.0 * u2 * Ph + 15.0 * Ph * Ph / rho)) / tau;
}

/* tau = (n sigma_c v_th)^-1 = lambda / v_th, lambda ~ 1/rho, v_th = sqrt(8 k_B T / (pi m))
 * = sqrt(8 P / (pi rho)) (L284, L474).  With Kn = lambda_ref / L_ref at rho_ref (reading R17):
 *   tau(rho, P) = Kn L_ref (rho_ref / rho) / sqrt(8 P / (pi rho)). */
double mmo_tau(int model, double tau_const, double Kn, double L_ref, double rho_ref,
               double rho, double P)
{
    if (model == MMO_TAU_CONST) return tau_const;
    if (model == MMO_TAU_KN) {
        const double pi = 3.14159265358979323846;
        return Kn * L_ref * (rho_ref / rho) / sqrt(8.0 * P / (pi * rho));
    }
    return INFINITY;  /* collisionless: source disabled (L432) */
}
