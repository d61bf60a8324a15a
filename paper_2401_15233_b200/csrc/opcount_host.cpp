// opcount_host.cpp -- counts the source-level FP64 operations the CUDA path executes per cell
// update (the "algorithmic flops" of the roofline line).
// mm_physics.cuh is compiled on the HOST with `double` replaced by a counting type; the
// composition below mirrors what the fused step kernel does for ONE cell with no tile overhead:
//   1 cons->prim, 2 interfaces (x and y: slopes of both cells, 2 face evaluations, HLL),
//   the update, the BGK source and the tail CFL evaluation of the new state.
// Convention: each + - * / sqrt exp log = 1 (an FMA is 2); comparisons, fabs, fmin/fmax,
// negation and copies = 0.  Measurement tooling only; nothing here is linked into libmm.so.
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
inline cnt fabs(cnt a) { return cnt(std::fabs(a.v)); }
inline cnt fmin(cnt a, cnt b) { return cnt(std::fmin(a.v, b.v)); }
inline cnt fmax(cnt a, cnt b) { return cnt(std::fmax(a.v, b.v)); }
inline cnt fmin(cnt a, double b) { return cnt(std::fmin(a.v, b)); }
inline cnt fmax(cnt a, double b) { return cnt(std::fmax(a.v, b)); }

#define MM_OPCOUNT_HOST
#define __device__
#define __host__
#define __forceinline__ inline
#define double cnt
#include "mm_physics.cuh"
using namespace mm;

template <int NM>
static void interface(const Params& p, const cnt (&Wam)[NM], const cnt (&Wa)[NM], const cnt (&Wb)[NM],
                      const cnt (&Wbp)[NM], cnt (&Fh)[NM])
{
    cnt ha[NM], hb[NM], WL[NM], WR[NM];
    half_slopes<NM>(p, Wam, Wa, Wb, ha);
    half_slopes<NM>(p, Wa, Wb, Wbp, hb);
    for (int k = 0; k < NM; ++k) { WL[k] = Wa[k] + ha[k]; WR[k] = Wb[k] - hb[k]; }
    cnt FL[NM], UL[NM], FR[NM], UR[NM], a, b, c, d;
    if constexpr (NM == 5) { eval_face5(p, WL, FL, UL, a, b); eval_face5(p, WR, FR, UR, c, d); }
    else { eval_face14(p, WL, FL, UL, a, b); eval_face14(p, WR, FR, UR, c, d); }
    numflux<NM>(p.flux, FL, FR, UL, UR, a, b, c, d, Fh);
}

template <int NM>
static long long one_cell(Params p, int ndim)
{
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
            for (int k = 0; k < 14; ++k) W[c][k] = w[k];
        }
    }
    cnt U[NM], Wc[NM], Fw[NM], Fe[NM], Un[NM];
    if constexpr (NM == 5) prim2cons5(W[1], U); else prim2cons14(W[1], U);
    cnt::ops = 0;
    if constexpr (NM == 5) cons2prim5(U, Wc); else cons2prim14(U, Wc);
    const cnt dt = 1e-3, dtdx = dt / p.dx, dtdy = dt / p.dy;
    for (int d = 0; d < ndim; ++d) {          // each cell owns one interface per direction
        interface<NM>(p, W[0], W[1], W[2], W[3], Fe);
        for (int k = 0; k < NM; ++k) Fw[k] = Fe[k] * 0.99;   // neighbour's flux (not counted twice)
        cnt::ops -= NM;
        for (int k = 0; k < NM; ++k) Un[k] = (d == 0 ? U[k] : Un[k]) - (d == 0 ? dtdx : dtdy) * (Fe[k] - Fw[k]);
    }
    if constexpr (NM == 5) add_source5(Wc, dt * inv_tau(p, Wc[0], Wc[2]), Un);
    else add_source14(Wc, dt * inv_tau(p, Wc[0], (Wc[4] + Wc[7] + Wc[9]) / 3.0), Un);
    cnt Wn[NM], sx, sy;
    if constexpr (NM == 5) { cons2prim5(Un, Wn); cell_speed5(p, Wn, sx); sx = sx / p.dx; }
    else { cons2prim14(Un, Wn); cell_speeds14(p, Wn, sx, sy); sx = fmax(sx / p.dx, sy / p.dy); }
    return cnt::ops;
}

int main()
{
    Params p{};
    p.sigma_lim = 1e-4; p.ws_scale = 1.0; p.dx = 0.01; p.dy = 0.01;
    p.inv_tau_coef = 100.0; p.tau_model = 2; p.limiter = 1; p.flux = 0;
    for (int shared = 0; shared < 2; ++shared) {
        p.shared_limiter = shared;
        printf("kernel_flops_per_cell_update_14_%s %lld\n", shared ? "shared_limiter" : "per_variable_limiter",
               one_cell<14>(p, 2));
        printf("kernel_flops_per_cell_update_5_%s %lld\n", shared ? "shared_limiter" : "per_variable_limiter",
               one_cell<5>(p, 1));
    }
    return 0;
}
