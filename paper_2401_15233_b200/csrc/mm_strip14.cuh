// mm_strip14.cuh -- the fused 14-moment 2-D time step (steps a2-a9 of DESIGN.md section 2).
//
// One WARP owns a strip of 30 cells in x and marches through a chunk of rows in y; warps never
// synchronise with one another.  Per warp, in shared memory (NV = moments carried: 14, or the
// 10 z-even ones on the z-symmetric path):
//   ring  [3][NV][34]  primitives of the rows r-1 .. r+1 (cells x0-2 .. x0+31), a ring over r;
//   cons  [2][NV][34]  conserved rows in flight: filled by cp.async one row ahead of use, so the
//                      HBM latency of row r+2 hides behind the work on row r at no register cost;
//   acc   [NV][32]     partial update of the row being assembled;
//   hsv   [NV][32]     half slopes in y of the previous row (each slope is computed once);
// and per block the 9 KB table of the wave-speed functions a(P*), b(P*) (mm_physics.cuh).
// Every interface is evaluated in one form: the lane holds a centre cell C with its two
// neighbours M and P along the direction, computes C's limited half slope h (a3), obtains the
// half slope hM of M from the lane / row that computed it, and evaluates the interface M|C
// from the face states W_M + hM and W_C - h (a4-a7).
//   y (d = 0): lane l, C = cell l of row r, M = row r-1; hM from `hsv`; G_r completes row r-1:
//              U^{n+1} = acc - dt/dy G_r + dt C(W) (a8), store, wave speeds of the new state
//              into the running CFL maximum (a9); then acc = U_r + dt/dy G_r.  The product
//              dt/dy G_r is rounded on its own both times (no FMA contraction), so that equal
//              fluxes through the two y faces of a cell cancel exactly.
//   x (d = 1): lane L, C = cell L-1 of row r, M = cell L-2; hM by shuffle from lane L-1;
//              acc(cell L-1) -= dt/dx (F from lane L+1 - own F).
// The two directions run through ONE copy of the slope / closure / wave-speed / HLL code (a
// non-unrolled loop over d), which keeps the kernel inside the instruction cache.
#pragma once
#include "mm_kernels.cuh"

namespace mm {

constexpr int kSW = 30;                 // cells per strip
constexpr int kRW = 34;                 // staged cells per row: 2 + 30 + 2
#ifndef MM_STRIP_WPB
#define MM_STRIP_WPB 1
#endif
constexpr int kStripWPB = MM_STRIP_WPB; // warps per block (a block is only a container of warps)

// Moments carried by a kernel variant and their compact numbering.
template <bool ZS>
struct Mom {
    static constexpr int NV = ZS ? 10 : 14;
    __host__ __device__ static constexpr int full(int k)          // compact -> moment index
    {
        const int t[14] = {0, 1, 2, 4, 5, 7, 9, 10, 11, 13, 0, 0, 0, 0};
        return ZS ? t[k] : k;
    }
    __host__ __device__ static constexpr int compact(int m)       // moment index -> compact
    {
        const int t[14] = {0, 1, 2, -1, 3, 4, -1, 5, -1, 6, 7, 8, -1, 9};
        return ZS ? t[m] : m;
    }
    __host__ __device__ static constexpr int cswap(int k) { return compact(swap_xy(full(k))); }
    static constexpr int warp_smem_doubles = 3 * NV * kRW + 2 * NV * kRW + 2 * NV * 32;
    // The general variant's strip buffers are 26 KB per warp: with the 9 KB table beside them only 6
    // warps fit an SM, without it 8.  It reads the table from global memory through L1 instead.
    static constexpr bool table_in_smem = ZS;
};

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Work decomposition: item = (strip, chunk); chunk c covers rows [c ny / nchunks, (c+1) ny / nchunks).
// EXT = false is the plain forward-Euler step with the explicit source (Ubase = nullptr,
// dt_scale = 1, do_rate = 1, source_scheme = 0 folded at compile time); EXT = true takes them at
// run time (midpoint passes, point-implicit source).
template <bool ZS, int MINB, bool EXT>
__global__ void __launch_bounds__(32 * kStripWPB, MINB)
k_step14_strip(const Params pg, const double* __restrict__ Uin, double* Uout, Ctrl* ctrl,
               int slot_next, int nstrips, int nchunks, const double* Ubase_, double dt_scale_, int do_rate_)
{
    const double* Ubase = EXT ? Ubase_ : nullptr;
    const double dt_scale = EXT ? dt_scale_ : 1.0;
    const int do_rate = EXT ? do_rate_ : 1;
    using Z = typename std::conditional<ZS, zero_t, double>::type;
    using M = Mom<ZS>;
    constexpr int NM = 14, NV = M::NV, RS = NV * kRW;          // RS: doubles per staged row
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // the block's copy of the a(P*), b(P*) table (Eq 29c-d), behind the warps' buffers
    Params p = pg;
    if constexpr (M::table_in_smem) {
        double* tab = smem + kStripWPB * M::warp_smem_doubles;
        for (int i = threadIdx.x; i < AbTable::kDoubles; i += 32 * kStripWPB) tab[i] = pg.ab[i];
        __syncthreads();
        p.ab = tab;
    }
    const int item = blockIdx.x * kStripWPB + warp;
    if (item >= nstrips * nchunks) return;
    const int strip = item % nstrips, chunk = item / nstrips;
    const int x0 = strip * kSW;
    const int y0 = (int)((long long)chunk * p.ny / nchunks);
    const int y1 = (int)((long long)(chunk + 1) * p.ny / nchunks);
    if (y1 <= y0) return;
    double* ring = smem + warp * M::warp_smem_doubles;
    double* cons = ring + 3 * RS;
    double* acc = cons + 2 * RS;
    double* hsv = acc + NV * 32;
    const size_t plane = (size_t)p.rows * p.pitch;
    const int ncell = min(kSW, p.nx - x0);            // cells of this strip
    const int ncol = min(kRW, p.nx + 4 - x0);         // staged columns that exist
    const bool cell_ok = lane < ncell;                // y phase: the lane's cell is cell `lane`
    const bool xcell_ok = lane >= 1 && lane - 1 < ncell;  // x phase: cell lane-1 is updated
    const size_t ccol = (size_t)x0 + lane + 2;        // padded column of the lane's cell (y phase)

    if (ctrl->skip) {                  // failed / past t_end: carry the state over unchanged
        if (cell_ok)
            for (int r = y0; r < y1; ++r)
#pragma unroll
                for (int m = 0; m < NM; ++m)
                    Uout[m * plane + (size_t)(r + 2) * p.pitch + ccol] = Uin[m * plane + (size_t)(r + 2) * p.pitch + ccol];
        return;
    }
    // U_out = B - dt div F(U_in) + source:  B = U_in for forward Euler and for the half step of the
    // midpoint scheme (dt_scale = 1/2, no CFL reduction); B = Ubase = U^n for its full step, which
    // may be written in place (Uout == Ubase: a cell's B is read by the lane that later writes it).
    const double dt = ctrl->dt * dt_scale;
    const double dtdx = dt / p.dx, dtdy = dt / p.dy;

    auto load_row = [&](int r, int cslot) {          // interior row r in [-2, ny+1] -> cons[cslot]
        const double* src = Uin + (size_t)(r + 2) * p.pitch + x0;
        double* dst = cons + cslot * RS;
        if (lane < ncol) {
#pragma unroll
            for (int k = 0; k < NV; ++k) cp_async8(dst + k * kRW + lane, src + M::full(k) * plane + lane);
        }
        if (lane + 32 < ncol) {
#pragma unroll
            for (int k = 0; k < NV; ++k) cp_async8(dst + k * kRW + 32 + lane, src + M::full(k) * plane + 32 + lane);
        }
        cp_async_commit();
    };
    auto convert_row = [&](int cslot, int rslot) {   // cons[cslot] -> primitives in ring[rslot] (a2)
        const double* src = cons + cslot * RS;
        double* dst = ring + rslot * RS;
#pragma unroll 1
        for (int c = lane; c < ncol; c += 32) {
            double U[NM], W[NM];
#pragma unroll
            for (int k = 0; k < NV; ++k) U[M::full(k)] = src[k * kRW + c];
            cons2prim14<Z>(U, W);
#pragma unroll
            for (int k = 0; k < NV; ++k) dst[k * kRW + c] = W[M::full(k)];
        }
    };

    load_row(y0 - 2, 0); load_row(y0 - 1, 1);
    cp_async_wait_all(); __syncwarp();
    convert_row(0, 0); convert_row(1, 1);
    __syncwarp();
    load_row(y0, 0); load_row(y0 + 1, 1);            // stay in cons: U of rows y0, y0+1
    cp_async_wait_all(); __syncwarp();
    convert_row(0, 2);
    __syncwarp();
    int sm = 0, sc = 1, sp = 2;                      // ring slots of the rows r-1, r, r+1

    double rate = 0.0, speed = 0.0;
    int bad = 0;
    for (int r = y0 - 1; r <= y1; ++r) {
        const int cs = (r - y0) & 1;
#pragma unroll 1
        for (int d = 0; d < 2; ++d) {
            // Lanes without an interface of their own (beyond the strip's last cell / staged column)
            // take the last valid cell's data, so every lane evaluates a valid state; their
            // results are never used.
            const double *qm, *qc, *qp;              // plane 0 of the cells M, C, P
            if (d == 0) {                            // y: C = (row r, cell lane)
                const double* b = ring + min(lane, ncell - 1) + 2;
                qm = b + sm * RS; qc = b + sc * RS; qp = b + sp * RS;
            } else {                                 // x: C = (row r, cell lane-1)
                if (r < y0 || r == y1) break;
                __syncwarp();                        // every lane has taken U_r out of cons[cs]
                load_row(r + 2, cs);
                qm = ring + sc * RS + min(lane, ncol - 3); qc = qm + 1; qp = qm + 2;
            }
            // ---- a3: limited half slope of C; face states of the interface M|C
            double WL[NM], WR[NM];
            {
                double Wm[NV], Wc[NV], Wp[NV], h[NV];
#pragma unroll
                for (int k = 0; k < NV; ++k) {
                    const int o = (d == 0 ? M::cswap(k) : k) * kRW;
                    Wm[k] = qm[o]; Wc[k] = qc[o]; Wp[k] = qp[o];
                }
                if (p.limiter == 0) {
#pragma unroll
                    for (int k = 0; k < NV; ++k) h[k] = 0.0;
                } else if (p.shared_limiter) {
                    PsiShared pm;
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const double dm = Wc[k] - Wm[k], dp = Wp[k] - Wc[k];
                        h[k] = dm + dp;
                        pm.add(p.limiter, dm, dp, h[k]);
                    }
                    const double q = 0.25 * pm.psi();
#pragma unroll
                    for (int k = 0; k < NV; ++k) h[k] = q * h[k];
                } else {
#pragma unroll
                    for (int k = 0; k < NV; ++k)
                        h[k] = 0.5 * limited_slope(p.limiter, Wc[k] - Wm[k], Wp[k] - Wc[k]);
                }
                if (d == 0) {
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const double hm = hsv[k * 32 + lane];
                        hsv[k * 32 + lane] = h[k];
                        WL[M::full(k)] = Wm[k] + hm; WR[M::full(k)] = Wc[k] - h[k];
                    }
                    if (r < y0) continue;            // first pass of a chunk: slope of row y0-1 only
                } else {
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const double hm = __shfl_up_sync(0xffffffffu, h[k], 1);
                        WL[M::full(k)] = Wm[k] + hm; WR[M::full(k)] = Wc[k] - h[k];
                    }
                }
            }
            // ---- a4-a7: both face states through the closure, HLL / Rusanov
            double Fh[NV];
            {
                double FL[NM], UL[NM], FR[NM], UR[NM], lminL, lmaxL, lminR, lmaxR;
                eval_face14<Z>(p, WL, FL, UL, lminL, lmaxL);
                eval_face14<Z>(p, WR, FR, UR, lminR, lmaxR);
                if (p.flux == 1) {
                    const double S = dmax(dmax(fabs(lminL), fabs(lmaxL)), dmax(fabs(lminR), fabs(lmaxR)));
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const int m = M::full(k);
                        Fh[k] = 0.5 * (FL[m] + FR[m]) - 0.5 * S * (UR[m] - UL[m]);
                    }
                } else {
                    const double SL = dmin(dmin(lminL, lminR), 0.0), SR = dmax(dmax(lmaxL, lmaxR), 0.0);
                    const double inv = rcp(SR - SL), cL = SR * inv, cR = -SL * inv, cU = SL * cL;
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const int m = M::full(k);
                        Fh[k] = hll1(cL, cR, cU, FL[m], FR[m], UL[m], UR[m]);
                    }
                }
            }
            if (d == 0) {
                if (cell_ok) {
                    double G[NV];                    // back to unswapped numbering (L414)
#pragma unroll
                    for (int k = 0; k < NV; ++k) G[k] = Fh[M::cswap(k)];
                    if (r > y0) {                    // row r-1 is complete (a8), then a9 on the new state
                        double Un[NM], W[NM];
                        const double* w = ring + sm * RS + lane + 2;
#pragma unroll
                        for (int k = 0; k < NV; ++k) {
                            Un[M::full(k)] = __dsub_rn(acc[k * 32 + lane], __dmul_rn(dtdy, G[k]));
                            W[M::full(k)] = w[k * kRW];
                        }
                        if (p.tau_model != 0) {
                            if (EXT && p.source_scheme == 1) {   // point-implicit (L348): relax U* itself
                                double Ws[NM];
                                cons2prim14<Z>(Un, Ws);
                                const double x = dt * inv_tau(p, Ws[0], (Ws[4] + Ws[7] + Ws[9]) * (1.0 / 3.0));
                                add_source14<Z>(Ws, x * rcp(1.0 + x), Un);
                            } else {
                                add_source14<Z>(W, dt * inv_tau(p, W[0], (W[4] + W[7] + W[9]) * (1.0 / 3.0)), Un);
                            }
                        }
                        double* out = Uout + (size_t)(r + 1) * p.pitch + ccol;
#pragma unroll
                        for (int m = 0; m < NM; ++m) {
                            if (ZS && z_odd(m)) out[m * plane] = 0.0;
                            else out[m * plane] = Un[m];
                        }
                        if (do_rate) {
                            double rr, ss;
                            cell_rate<NM, Z>(p, Un, rr, ss, bad);
                            rate = dmax(rate, rr); speed = dmax(speed, ss);
                        }
                    }
                    if (r < y1) {
                        if (Ubase) {
                            const double* ub = Ubase + (size_t)(r + 2) * p.pitch + ccol;
#pragma unroll
                            for (int k = 0; k < NV; ++k)
                                acc[k * 32 + lane] = __dadd_rn(ub[M::full(k) * plane], __dmul_rn(dtdy, G[k]));
                        } else {
#pragma unroll
                            for (int k = 0; k < NV; ++k)
                                acc[k * 32 + lane] = __dadd_rn(cons[cs * RS + k * kRW + lane + 2], __dmul_rn(dtdy, G[k]));
                        }
                    }
                }
            } else {
                __syncwarp();                        // acc of row r was written by the y phase
#pragma unroll
                for (int k = 0; k < NV; ++k) {
                    const double Fn = __shfl_down_sync(0xffffffffu, Fh[k], 1);
                    if (xcell_ok) acc[k * 32 + lane - 1] = acc[k * 32 + lane - 1] - dtdx * (Fn - Fh[k]);
                }
            }
        }
        if (r < y1) {                                // row r+2 has landed: primitives into the slot of row r-1
            cp_async_wait_all(); __syncwarp();
            convert_row(cs, sm);
            __syncwarp();
            const int t = sm; sm = sc; sc = sp; sp = t;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
        speed = fmax(speed, __shfl_xor_sync(0xffffffffu, speed, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if (lane == 0 && do_rate) {
        atomic_max_pos(&ctrl->rate_bits[slot_next], rate);
        atomic_max_pos(&ctrl->speed_bits[slot_next], speed);
        if (bad) atomicOr(&ctrl->bad[slot_next], 1);
    }
}

}  // namespace mm
