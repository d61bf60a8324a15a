// mm_strip14.cuh -- the fused 14-moment 2-D time step (steps a2-a9 of DESIGN.md section 2).
//
// One WARP owns a strip of 31 cells in x and marches through a chunk of rows in y; warps never
// synchronise with one another.  Lane l owns the x-interface between strip cells l-1 and l
// (32 interfaces for 31 cells) and the y-interfaces and the update of strip cell l (l < 31).
// Per warp, in shared memory:
//   ring  [4][14][35]  primitives of the rows r-2 .. r+1 (cells x0-2 .. x0+32), a ring over r;
//   cons  [2][14][35]  conserved rows in flight: filled by cp.async one row ahead of use, so the
//                      HBM latency of row r+2 hides behind the x pass of row r at no register cost;
//   acc   [14][32]     per-lane partial update of the row being assembled.
// Row iteration r:  G_r (y-interface r-1|r) -> finish row r-1 in the scheme's order of operations (x then y then source),
// (acc - dt/dy (G_r - G_{r-1})) + dt C(W_{r-1}) (a8), store, cell-centre wave speeds of the new
// state -> running CFL maximum (a9); then row r: x-interfaces, neighbour flux by warp shuffle,
// acc = U_r - dt/dx (F_{i+1} - F_i).  The two interface directions run through
// ONE copy of the slope / closure / wave-speed / HLL code (a non-unrolled loop over the
// direction), which keeps the kernel inside the instruction cache.
#pragma once
#include "mm_kernels.cuh"

namespace mm {

constexpr int kSW = 31;                 // cells per strip
constexpr int kRW = 35;                 // staged cells per row: 2 + 31 + 2
constexpr int kRingD = 4 * 14 * kRW;    // doubles
constexpr int kConsD = 2 * 14 * kRW;
constexpr int kAccD = 14 * 32;
constexpr int kWarpSmemD = kRingD + kConsD + kAccD;
constexpr int kStripWPB = 2;            // warps per block (a container only)

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Interface flux from the four stencil cells (am | a || b | bp) along one direction.  q0..q3
// point at moment plane 0 of those cells, ps is the plane stride.  MUSCL on primitives
// (L262-264), both face states through the closure (eval_face14), HLL / Rusanov.  For the y
// direction (swap) the state is index-swapped on load (L414); the caller swaps the flux back.
__device__ __forceinline__ void iface_flux14(const Params& p, const double* __restrict__ q0,
                                             const double* __restrict__ q1,
                                             const double* __restrict__ q2,
                                             const double* __restrict__ q3, int ps, bool swap,
                                             double (&Fh)[14])
{
    constexpr int NM = 14;
    double WL[NM], WR[NM];
    if (p.limiter != 0 && p.shared_limiter) {
        double Wam[NM], Wa[NM], Wb[NM], Wbp[NM], ha[NM], hb[NM];
#pragma unroll
        for (int k = 0; k < NM; ++k) {
            const int o = (swap ? swap_xy(k) : k) * ps;
            Wam[k] = q0[o]; Wa[k] = q1[o]; Wb[k] = q2[o]; Wbp[k] = q3[o];
        }
        half_slopes<NM>(p, Wam, Wa, Wb, ha);
        half_slopes<NM>(p, Wa, Wb, Wbp, hb);
#pragma unroll
        for (int k = 0; k < NM; ++k) { WL[k] = Wa[k] + ha[k]; WR[k] = Wb[k] - hb[k]; }
    } else {
#pragma unroll
        for (int k = 0; k < NM; ++k) {
            const int o = (swap ? swap_xy(k) : k) * ps;
            const double am = q0[o], a = q1[o], b = q2[o], bp = q3[o];
            double ha = 0.0, hb = 0.0;
            if (p.limiter != 0) {
                const double d = b - a;
                ha = 0.5 * limited_slope(p.limiter, a - am, d);
                hb = 0.5 * limited_slope(p.limiter, d, bp - b);
            }
            WL[k] = a + ha; WR[k] = b - hb;
        }
    }
    double FL[NM], UL[NM], FR[NM], UR[NM], lminL, lmaxL, lminR, lmaxR;
    eval_face14(p, WL, FL, UL, lminL, lmaxL);
    eval_face14(p, WR, FR, UR, lminR, lmaxR);
    numflux<NM>(p.flux, FL, FR, UL, UR, lminL, lmaxL, lminR, lmaxR, Fh);
}

// Work decomposition: item = (strip, chunk); chunk c covers rows [c ny / nchunks, (c+1) ny / nchunks).
__global__ void __launch_bounds__(32 * kStripWPB, 8 / kStripWPB)
k_step14_strip(Params p, const double* __restrict__ Uin, double* __restrict__ Uout, Ctrl* ctrl,
               int slot_next, int nstrips, int nchunks)
{
    constexpr int NM = 14, RS = NM * kRW;           // doubles per staged row
    extern __shared__ double smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int item = blockIdx.x * kStripWPB + warp;
    if (item >= nstrips * nchunks) return;
    const int strip = item % nstrips, chunk = item / nstrips;
    const int x0 = strip * kSW;
    const int y0 = (int)((long long)chunk * p.ny / nchunks);
    const int y1 = (int)((long long)(chunk + 1) * p.ny / nchunks);
    if (y1 <= y0) return;
    double* ring = smem + warp * kWarpSmemD;
    double* cons = ring + kRingD;
    double* acc = cons + kConsD;
    const size_t plane = (size_t)p.rows * p.pitch;
    const bool cell_ok = lane < kSW && x0 + lane < p.nx;
    const bool xif_ok = x0 + lane <= p.nx;
    const size_t ccol = (size_t)x0 + lane + 2;       // padded column of the lane's cell

    if (ctrl->skip) {                  // failed / past t_end: carry the state over unchanged
        if (cell_ok)
            for (int r = y0; r < y1; ++r)
#pragma unroll
                for (int m = 0; m < NM; ++m)
                    Uout[m * plane + (size_t)(r + 2) * p.pitch + ccol] = Uin[m * plane + (size_t)(r + 2) * p.pitch + ccol];
        return;
    }
    const double dt = ctrl->dt;
    const double dtdx = dt / p.dx, dtdy = dt / p.dy;
    const int ncol = min(kRW, p.nx + 4 - x0);        // staged columns that exist

    auto load_row = [&](int r, int cslot) {          // interior row r in [-2, ny+1] -> cons[cslot]
        const double* src = Uin + (size_t)(r + 2) * p.pitch + x0;
        double* dst = cons + cslot * RS;
        if (lane < ncol) {
#pragma unroll
            for (int m = 0; m < NM; ++m) cp_async8(dst + m * kRW + lane, src + m * plane + lane);
        }
        if (lane + 32 < ncol) {
#pragma unroll
            for (int m = 0; m < NM; ++m) cp_async8(dst + m * kRW + 32 + lane, src + m * plane + 32 + lane);
        }
        cp_async_commit();
    };
    auto convert_row = [&](int r, int cslot) {       // cons[cslot] -> primitives in the ring (a2)
        const double* src = cons + cslot * RS;
        double* dst = ring + ((r + 2) & 3) * RS;
#pragma unroll 1
        for (int c = lane; c < ncol; c += 32) {
            double U[NM], W[NM];
#pragma unroll
            for (int m = 0; m < NM; ++m) U[m] = src[m * kRW + c];
            cons2prim14(U, W);
#pragma unroll
            for (int m = 0; m < NM; ++m) dst[m * kRW + c] = W[m];
        }
    };

    load_row(y0 - 2, 0); load_row(y0 - 1, 1);
    cp_async_wait_all(); __syncwarp();
    convert_row(y0 - 2, 0); convert_row(y0 - 1, 1);
    __syncwarp();
    load_row(y0, 0); load_row(y0 + 1, 1);
    cp_async_wait_all(); __syncwarp();
    convert_row(y0, 0); convert_row(y0 + 1, 1);
    __syncwarp();

    double rate = 0.0, speed = 0.0;
    int bad = 0;
    double Gp[NM];                                   // y-interface flux of the previous row
#pragma unroll
    for (int m = 0; m < NM; ++m) Gp[m] = 0.0;
    for (int r = y0; r <= y1; ++r) {
        const int cs = (r - y0) & 1;
#pragma unroll 1
        for (int d = 0; d < 2; ++d) {
            const double *q0, *q1, *q2, *q3;
            bool act;
            if (d == 0) {                            // y-interface between rows r-1 and r
                const double* b = ring + lane + 2;
                q0 = b + (r & 3) * RS; q1 = b + ((r + 1) & 3) * RS;
                q2 = b + ((r + 2) & 3) * RS; q3 = b + ((r + 3) & 3) * RS;
                act = cell_ok;
            } else {                                 // x-interface between cells lane-1 and lane of row r
                if (r == y1) break;
                __syncwarp();                        // every lane has taken U_r out of cons[cs]
                load_row(r + 2, cs);
                const double* b = ring + ((r + 2) & 3) * RS + lane;
                q0 = b; q1 = b + 1; q2 = b + 2; q3 = b + 3;
                act = xif_ok;
            }
            double Fh[NM];
#pragma unroll
            for (int m = 0; m < NM; ++m) Fh[m] = 0.0;
            if (act) iface_flux14(p, q0, q1, q2, q3, kRW, d == 0, Fh);
            if (d == 0) {
                if (cell_ok) {
                    double G[NM];
#pragma unroll
                    for (int m = 0; m < NM; ++m) G[m] = Fh[swap_xy(m)];
                    if (r > y0) {                    // row r-1 is complete (a8), then a9 on the new state
                        double Un[NM], W[NM];
                        const double* w = ring + ((r + 1) & 3) * RS + lane + 2;
#pragma unroll
                        for (int m = 0; m < NM; ++m) {
                            Un[m] = acc[m * 32 + lane] - dtdy * (G[m] - Gp[m]);
                            W[m] = w[m * kRW];
                        }
                        if (p.tau_model != 0)
                            add_source14(W, dt * inv_tau(p, W[0], (W[4] + W[7] + W[9]) / 3.0), Un);
#pragma unroll
                        for (int m = 0; m < NM; ++m)
                            Uout[m * plane + (size_t)(r + 1) * p.pitch + ccol] = Un[m];
                        double rr, ss;
                        cell_rate<NM>(p, Un, rr, ss, bad);
                        rate = fmax(rate, rr); speed = fmax(speed, ss);
                    }
#pragma unroll
                    for (int m = 0; m < NM; ++m) Gp[m] = G[m];
                    if (r < y1) {
#pragma unroll
                        for (int m = 0; m < NM; ++m)
                            acc[m * 32 + lane] = cons[cs * RS + m * kRW + lane + 2];
                    }
                }
            } else {
                double Fn[NM];
#pragma unroll
                for (int m = 0; m < NM; ++m) Fn[m] = __shfl_down_sync(0xffffffffu, Fh[m], 1);
                if (cell_ok) {
#pragma unroll
                    for (int m = 0; m < NM; ++m)
                        acc[m * 32 + lane] = acc[m * 32 + lane] - dtdx * (Fn[m] - Fh[m]);
                }
            }
        }
        if (r < y1) {                                // row r+2 has landed: primitives into the slot of row r-2
            cp_async_wait_all(); __syncwarp();
            convert_row(r + 2, cs);
            __syncwarp();
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
        speed = fmax(speed, __shfl_xor_sync(0xffffffffu, speed, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if (lane == 0) {
        atomic_max_pos(&ctrl->rate_bits[slot_next], rate);
        atomic_max_pos(&ctrl->speed_bits[slot_next], speed);
        if (bad) atomicOr(&ctrl->bad[slot_next], 1);
    }
}

}  // namespace mm
