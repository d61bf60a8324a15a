// opcount_host.cpp -- counts the source-level FP64 operations the CUDA path executes per cell
// update (the "algorithmic flops" of the roofline line).
// mm_physics.cuh is compiled on the HOST with `double` replaced by a counting type; the
// composition below mirrors what the fused step kernel does for ONE cell with no tile overhead:
//   per direction 1 limited slope and 1 interface (2 face evaluations, HLL), the update, the BGK
//   source, and the tail: cons->prim of the new state and its CFL wave speeds.  The 14-moment kernel
//   reads the primitives the previous step's tail stored (one cons->prim per cell and step); the
//   5-moment kernel converts on load as well.
// Convention: each + - * / sqrt exp pow = 1 (an FMA is 2); comparisons, fabs,
// fmin/fmax, negation and copies = 0.  The wave-speed functions a(P*), b(P*) are booked as the method's
// formulas (10 operations per call), not as the table evaluation the kernel executes.  Measurement tooling only; nothing here is linked into libmm.so.
#include <cmath>
#include <cstdio>

struct cnt {
    double v;
    static long long ops;
    cnt() = default;
    cnt(double x) : v(x) {}
    cnt(int x) : v(x) {}
};
long long cnt::ops = 0;
#define B(op)                                                                       \
    inline cnt operator op(cnt a, cnt b) { ++cnt::ops; return cnt(a.v op b.v); }    \
    inline cnt operator op(cnt a, double b) { ++cnt::ops; return cnt(a.v op b); }   \
    inline cnt operator op(double a, cnt b) { ++cnt::ops; return cnt(a op b.v); }
B(+) B(-) B(*) B(/)
#undef B
inline cnt operator-(cnt a) { return cnt(-a.v); }
inline cnt& operator+=(cnt& a, cnt b) { ++cnt::ops; a.v += b.v; return a; }
#define R(op)                                                       \
    inline bool operator op(cnt a, cnt b) { return a.v op b.v; }    \
    inline bool operator op(cnt a, double b) { return a.v op b; }
R(<) R(>) R(<=) R(>=) R(==)
#undef R
inline cnt sqrt(cnt a) { ++cnt::ops; return cnt(std::sqrt(a.v)); }
inline cnt exp(cnt a) { ++cnt::ops; return cnt(std::exp(a.v)); }
inline cnt log(cnt a) { ++cnt::ops; return cnt(std::log(a.v)); }
inline cnt pow(cnt a, double b) { ++cnt::ops; return cnt(std::pow(a.v, b)); }
inline cnt fabs(cnt a) { return cnt(std::fabs(a.v)); }
inline cnt fmin(cnt a, cnt b) { return cnt(std::fmin(a.v, b.v)); }
inline cnt fmax(cnt a, cnt b) { return cnt(std::fmax(a.v, b.v)); }
inline cnt fmin(cnt a, double b) { return cnt(std::fmin(a.v, b)); }
inline cnt fmax(cnt a, double b) { return cnt(std::fmax(a.v, b)); }

#include <type_traits>
#define MM_OPCOUNT_HOST
#define __device__
#define __host__
#define __forceinline__ inline
#define double cnt
#include "mm_physics.cuh"
using namespace mm;

// one limited half slope of cell c from its neighbours (computed once per cell and direction)
template <int NM, int LIM>
static void half_slope_lim(const Params& p, const cnt (&Wm)[NM], const cnt (&Wc)[NM], const cnt (&Wp)[NM],
                           cnt (&h)[NM], bool zs)
{
    PsiShared<LIM> pm;                                 // the shared limiter value of this limiter kind
    for (int k = 0; k < NM; ++k) {
        if (NM == 14 && zs && z_odd(k)) continue;
        const cnt dm = Wc[k] - Wm[k], dp = Wp[k] - Wc[k];
        h[k] = dm + dp;
        if (p.shared_limiter) pm.add(dm, dp, h[k]);
        else h[k] = 0.5 * limited_slope(p.limiter, dm, dp);
    }
    if (p.shared_limiter) {
        const cnt q = 0.25 * pm.psi();
        for (int k = 0; k < NM; ++k) {
            if (NM == 14 && zs && z_odd(k)) continue;
            h[k] = q * h[k];
        }
    }
}

template <int NM>
static void half_slope(const Params& p, const cnt (&Wm)[NM], const cnt (&Wc)[NM], const cnt (&Wp)[NM],
                       cnt (&h)[NM], bool zs)
{
    if (p.limiter == 2) half_slope_lim<NM, 2>(p, Wm, Wc, Wp, h, zs);
    else half_slope_lim<NM, 1>(p, Wm, Wc, Wp, h, zs);
}

// interface M|C: face states from the two half slopes, two face evaluations, HLL or Rusanov (p.flux)
template <int NM, class Z>
static void interface(const Params& p, const cnt (&Wm)[NM], const cnt (&hm)[NM], const cnt (&Wc)[NM],
                      const cnt (&hc)[NM], cnt (&Fh)[NM])
{
    constexpr bool zs = std::is_same<Z, zero_t>::value;
    cnt WL[NM], WR[NM];
    for (int k = 0; k < NM; ++k) {
        if (NM == 14 && zs && z_odd(k)) continue;
        WL[k] = Wm[k] + hm[k]; WR[k] = Wc[k] - hc[k];
    }
    cnt FL[NM], UL[NM], FR[NM], UR[NM], a, b, c, d;
    if constexpr (NM == 5) { eval_face5(p, WL, FL, UL, a, b); eval_face5(p, WR, FR, UR, c, d); }
    else { eval_face14<Z>(p, WL, FL, UL, a, b); eval_face14<Z>(p, WR, FR, UR, c, d); }
    if (p.flux == 1) {                                 // Rusanov, as mm_tm14.cuh / mm_kernels.cuh write it
        const cnt S = fmax(fmax(fabs(a), fabs(b)), fmax(fabs(c), fabs(d)));
        for (int k = 0; k < NM; ++k) {
            if (NM == 14 && zs && z_odd(k)) continue;
            Fh[k] = 0.5 * (FL[k] + FR[k]) - 0.5 * S * (UR[k] - UL[k]);
        }
        return;
    }
    const cnt SL = fmin(fmin(a, c), 0.0), SR = fmax(fmax(b, d), 0.0);
    const cnt inv = rcp(SR - SL), cL = SR * inv, cR = -SL * inv, cU = SL * cL;
    for (int k = 0; k < NM; ++k) {
        if (NM == 14 && zs && z_odd(k)) continue;
        Fh[k] = hll1(cL, cR, cU, FL[k], FR[k], UL[k], UR[k]);
    }
}

template <int NM, class Z>
static long long one_cell(Params p, int ndim)
{
    constexpr bool zs = std::is_same<Z, zero_t>::value;
    // four smooth, non-equilibrium neighbouring states (all limiter branches active)
    cnt W[4][NM];
    for (int c = 0; c < 4; ++c) {
        const cnt e = 0.02 * c;
        if constexpr (NM == 5) {
            const cnt w[5] = {1.0 + e, 0.3 + e, 1.1 + e, 0.2 + e, 3.9 + 4.0 * e};
            for (int k = 0; k < 5; ++k) W[c][k] = w[k];
        } else {
            const cnt w[14] = {1.0 + e, 0.3 + e, -0.2 + e, 0.1 + e, 1.1 + e, 0.05 + e, 0.02 + e, 0.9 + e,
                               0.03 + e, 1.0 + e, 0.2 + e, -0.1 + e, 0.05 + e, 16.0 + 9.0 * e};
            for (int k = 0; k < 14; ++k) W[c][k] = (zs && z_odd(k)) ? cnt(0.0) : w[k];
        }
    }
    cnt U[NM], Wc[NM], Fw[NM], Fe[NM], Un[NM], hm[NM], hc[NM];
    if constexpr (NM == 5) prim2cons5(W[1], U); else prim2cons14<Z>(W[1], U);
    half_slope<NM>(p, W[0], W[1], W[2], hm, zs);       // the neighbour's slope (its own cost)
    cnt::ops = 0;
    if constexpr (NM == 5) cons2prim5(U, Wc);
    else for (int k = 0; k < NM; ++k) Wc[k] = W[1][k];     // stored by the previous step's tail (mm_tm14.cuh)
    const cnt dt = 1e-3, dtdx = dt / p.dx, dtdy = dt / p.dy;
    for (int d = 0; d < ndim; ++d) {          // each cell owns one slope and one interface per direction
        half_slope<NM>(p, W[1], W[2], W[3], hc, zs);
        interface<NM, Z>(p, W[1], hm, W[2], hc, Fe);
        for (int k = 0; k < NM; ++k) Fw[k] = Fe[k];         // neighbour's flux (not counted twice)
        for (int k = 0; k < NM; ++k) {
            if (NM == 14 && zs && z_odd(k)) continue;
            // x: acc = U - dtdx (F' - F); y: acc + dtdy G, then - dtdy G'  (2 flops each per moment)
            Un[k] = (d == 0 ? U[k] : Un[k]) - (d == 0 ? dtdx : dtdy) * (Fe[k] - Fw[k]);
        }
    }
    if constexpr (NM == 5) add_source5(Wc, dt * inv_tau(p, Wc[0], Wc[2]), Un);
    else add_source14<Z>(Wc, dt * inv_tau(p, Wc[0], (Wc[4] + Wc[7] + Wc[9]) * (1.0 / 3.0)), Un);
    cnt Wn[NM], sx, sy;
    if constexpr (NM == 5) { cons2prim5(Un, Wn); cell_speed5(p, Wn, sx); sx = sx / p.dx; }
    else { cons2prim14<Z>(Un, Wn); cell_speeds14<Z>(p, Wn, sx, sy); sx = fmax(sx / p.dx, sy / p.dy); }
    return cnt::ops;
}

int main()
{
    Params p{};
    static cnt dummy_tab[AbTable::kStride];        // coefficients do not matter for the count
    for (auto& c : dummy_tab) c = cnt(0.5);
    p.ab = dummy_tab;
    p.set_constants();
    p.sigma_lim = 1e-4; p.ws_scale = 1.0; p.dx = 0.01; p.dy = 0.01;
    p.inv_tau_coef = 100.0; p.tau_model = 2; p.limiter = 1; p.flux = 0;
    // a(P*), b(P*) of Eq 29c-d are booked at the METHOD's operation count (pow, exp = 1 each: 10 per call);
    // the *_executed lines add what the kernel's table evaluation executes beyond that.
    // keys: ..._{shared|per_variable}_limiter for minmod + HLL (the BASELINE configs); the other limiter / flux
    // combinations carry the suffix _vanalbada and / or _rusanov (the paper's own jets: both)
    for (int combo = 0; combo < 4; ++combo)
    for (int shared = 0; shared < 2; ++shared) {
        p.shared_limiter = shared;
        p.limiter = (combo & 1) ? 2 : 1; p.flux = (combo & 2) ? 1 : 0;
        char nm[96];
        snprintf(nm, sizeof nm, "%s%s%s", shared ? "shared_limiter" : "per_variable_limiter",
                 (combo & 1) ? "_vanalbada" : "", (combo & 2) ? "_rusanov" : "");
        long long n;
        g_ab_executed_flops = 0; n = one_cell<14, double>(p, 2);
        printf("kernel_flops_per_cell_update_14_%s %lld\n", nm, n);
        printf("kernel_flops_per_cell_update_14_%s_executed %lld\n", nm, n + g_ab_executed_flops);
        g_ab_executed_flops = 0; n = one_cell<14, zero_t>(p, 2);
        printf("kernel_flops_per_cell_update_14_zsym_%s %lld\n", nm, n);
        printf("kernel_flops_per_cell_update_14_zsym_%s_executed %lld\n", nm, n + g_ab_executed_flops);
        printf("kernel_flops_per_cell_update_5_%s %lld\n", nm, one_cell<5, double>(p, 1));
    }
    return 0;
}
