// mm_kernels.cuh -- CUDA kernels of the moment-method time step (sm_100a, fp64, SoA).
//
// Data layout: each state copy is NM planes of `rows` x `pitch` doubles,
// rows = ny + 4, pitch = roundup(nx + 4, 16); interior cell (i, j) sits at
// plane[(j + 2) * pitch + (i + 2)], two ghost layers on every side (corner ghosts are never
// read).  Two copies ping-pong; a control block in device memory carries t, dt, the step
// counter and the CFL max-reduction accumulators, so a sequence of steps needs no host sync.
#pragma once
#include "mm_physics.cuh"

namespace mm {

constexpr int kMaxBands = 8;
constexpr int kDtHistory = 1 << 16;     // time steps kept in the device-side dt history (ring)

// Control block (device memory).  rate = max_cells max(s_x/dx, s_y/dy), speed = max_cells s_d.
struct Ctrl {
    double t, dt, last_dt;
    unsigned long long rate_bits[2], speed_bits[2];   // max-reduced as ordered bit patterns (>= 0)
    double ghost_rate, ghost_speed;                   // constant part from Dirichlet ghost states
    long long bc_bad;                                 // a Dirichlet state has rho <= 0 or P <= 0
    long long bc_znz;                                 // a Dirichlet state has a non-zero z-odd moment
    long long steps;
    int bad[2];                                       // reduction saw rho<=0, P<=0 or non-finite
    int failed;                                       // sticky: stepping stopped (MM_ENONFINITE)
    int skip;                                         // this step leaves the state untouched
    int znz;                                          // the state set by mm_set_state has a non-zero z-odd moment
};

// Boundary tables (device memory): conserved ghost states of the Dirichlet sides.
struct BcSide {
    int type, nbands, has_default;
    int maxwellian;                                   // W[k][0..4] = (rho, u_x, u_y, u_z, T): expanded by k_bc_table
    unsigned used;                                    // bit k: table entry k is selected by a ghost cell
    double lo[kMaxBands], hi[kMaxBands];
    double W[kMaxBands + 1][14];                      // primitive band states, [nbands] = default
    double U[kMaxBands + 1][14];                      // conserved, filled by k_bc_table
};
struct BcTable { BcSide side[4]; };

__device__ __forceinline__ void atomic_max_pos(unsigned long long* a, double v)
{
    atomicMax(a, (unsigned long long)__double_as_longlong(v));
}

// block-wide max of two non-negative values and OR of a flag, then one atomic per block
template <int NT>
__device__ __forceinline__ void block_reduce_rate(double rate, double speed, int bad, Ctrl* ctrl,
                                                  int slot)
{
    __shared__ double s_rate[NT / 32], s_speed[NT / 32];
    __shared__ int s_bad[NT / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
        speed = fmax(speed, __shfl_xor_sync(0xffffffffu, speed, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { s_rate[w] = rate; s_speed[w] = speed; s_bad[w] = bad; }
    __syncthreads();
    if (w == 0) {
        rate = l < NT / 32 ? s_rate[l] : 0.0;
        speed = l < NT / 32 ? s_speed[l] : 0.0;
        bad = l < NT / 32 ? s_bad[l] : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
            speed = fmax(speed, __shfl_xor_sync(0xffffffffu, speed, o));
            bad |= __shfl_xor_sync(0xffffffffu, bad, o);
        }
        if (l == 0) {
            atomic_max_pos(&ctrl->rate_bits[slot], rate);
            atomic_max_pos(&ctrl->speed_bits[slot], speed);
            if (bad) atomicOr(&ctrl->bad[slot], 1);
        }
    }
}

// rate / speed / validity of one cell from its conserved moments
template <int NM, class Z = double>
__device__ __forceinline__ void cell_rate(const Params& p, const double (&U)[NM], double& rate,
                                          double& speed, int& bad)
{
    double W[NM];
    bool ok;
    if constexpr (NM == 5) {
        cons2prim5(U, W);
        double sx;
        ok = cell_speed5(p, W, sx);
        rate = sx * p.inv_dx; speed = sx;
    } else {
        cons2prim14<Z>(U, W);
        double sx, sy;
        ok = cell_speeds14<Z>(p, W, sx, sy);
        rate = dmax(sx * p.inv_dx, sy * p.inv_dy); speed = dmax(sx, sy);
    }
    // finite test: NaN or Inf fail (x - x != 0)
    if (!ok || !(rate - rate == 0.0)) { bad = 1; rate = 0.0; speed = 0.0; }
}

// rate / speed / validity of one 14-moment cell from its primitives (the step kernel's tail holds them)
template <class Z>
__device__ __forceinline__ void prim_rate14(const Params& p, const double (&W)[14], double& rate,
                                            double& speed, int& bad)
{
    double sx, sy;
    const bool ok = cell_speeds14<Z>(p, W, sx, sy);
    rate = dmax(sx * p.inv_dx, sy * p.inv_dy); speed = dmax(sx, sy);
    if (!ok || !(rate - rate == 0.0)) { bad = 1; rate = 0.0; speed = 0.0; }
}

// ---------------------------------------------------------------- state in / out kernels
// interior [NM][ny][nx] (conserved, or primitive when PRIM) -> padded conserved planes `dst` and, for the
// 14-moment system (dstW != nullptr), the padded primitive planes beside them (mm_tm14.cuh reads both)
template <int NM, bool PRIM>
__global__ void k_pack(Params p, const double* __restrict__ src, double* __restrict__ dst, double* __restrict__ dstW)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nx) return;
    const size_t plane = (size_t)p.rows * p.pitch, n = (size_t)p.nx * p.ny;
    for (int j = blockIdx.y; j < p.ny; j += gridDim.y) {     // gridDim.y <= 65535 rows per sweep
    double a[NM], b[NM];
#pragma unroll
    for (int m = 0; m < NM; ++m) a[m] = src[m * n + (size_t)j * p.nx + i];
    if constexpr (PRIM) {
        if constexpr (NM == 5) prim2cons5(a, b); else prim2cons14<double>(a, b);
    } else {
#pragma unroll
        for (int m = 0; m < NM; ++m) b[m] = a[m];
    }
#pragma unroll
    for (int m = 0; m < NM; ++m) dst[m * plane + (size_t)(j + 2) * p.pitch + i + 2] = b[m];
    if constexpr (NM == 14) {
        if (dstW) {
            if constexpr (!PRIM) cons2prim14<double>(b, a);      // a = W(U); given primitives are kept as they are
#pragma unroll
            for (int m = 0; m < NM; ++m) dstW[m * plane + (size_t)(j + 2) * p.pitch + i + 2] = a[m];
        }
    }
    }
}

template <int NM, bool PRIM>
__global__ void k_unpack(Params p, const double* __restrict__ src, double* __restrict__ dst)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= p.nx) return;
    const size_t plane = (size_t)p.rows * p.pitch, n = (size_t)p.nx * p.ny;
    for (int j = blockIdx.y; j < p.ny; j += gridDim.y) {
    double a[NM], b[NM];
#pragma unroll
    for (int m = 0; m < NM; ++m) a[m] = src[m * plane + (size_t)(j + 2) * p.pitch + i + 2];
    if constexpr (PRIM) {
        if constexpr (NM == 5) cons2prim5(a, b); else cons2prim14<double>(a, b);
    } else {
#pragma unroll
        for (int m = 0; m < NM; ++m) b[m] = a[m];
    }
#pragma unroll
    for (int m = 0; m < NM; ++m) dst[m * n + (size_t)j * p.nx + i] = b[m];
    }
}

// Dirichlet tables: primitive -> conserved, and the constant ghost contribution to the CFL max
// (ghost cells are part of the maximum, R13).  One thread per (side, state).
template <int NM>
__global__ void k_bc_table(Params p, BcTable* tab, Ctrl* ctrl, int nsides)
{
    const int side = blockIdx.x, k = threadIdx.x;
    if (side >= nsides) return;
    BcSide& b = tab->side[side];
    if (b.type != 2) return;
    const bool is_default = (k == b.nbands);
    if (k > b.nbands || (is_default && !b.has_default)) return;
    double W[NM], U[NM];
    if (b.maxwellian) {
        // Maxwellian of (rho, u, T): P = rho R_gas T (Eq 6), q = 0, R_iijj = 15 P^2/rho (L73),
        // 5-moment r = 3 P^2/rho (L127)
        const double rho = b.W[k][0], P = rho * p.R_gas * b.W[k][4];
#pragma unroll
        for (int m = 0; m < NM; ++m) W[m] = 0.0;
        W[0] = rho; W[1] = b.W[k][1];
        if constexpr (NM == 5) { W[2] = P; W[4] = 3.0 * P * P / rho; }
        else { W[2] = b.W[k][2]; W[3] = b.W[k][3]; W[4] = P; W[7] = P; W[9] = P; W[13] = 15.0 * P * P / rho; }
#pragma unroll
        for (int m = 0; m < NM; ++m) b.W[k][m] = W[m];
    } else {
#pragma unroll
        for (int m = 0; m < NM; ++m) W[m] = b.W[k][m];
    }
    if constexpr (NM == 5) prim2cons5(W, U); else prim2cons14<double>(W, U);
#pragma unroll
    for (int m = 0; m < NM; ++m) b.U[k][m] = U[m];
    // Every entry is converted (k_ghost may select any of them); only entries that some ghost cell
    // actually takes (b.used, set at mm_create) count for the CFL maximum and the validity flags.
    if (!((b.used >> k) & 1u)) return;
    double rate, speed; int bad = 0;
    cell_rate<NM>(p, U, rate, speed, bad);
    atomic_max_pos(reinterpret_cast<unsigned long long*>(&ctrl->ghost_rate), rate);
    atomic_max_pos(reinterpret_cast<unsigned long long*>(&ctrl->ghost_speed), speed);
    if (bad) ctrl->bc_bad = 1;
    if constexpr (NM == 14) {
        if (W[3] != 0.0 || W[6] != 0.0 || W[8] != 0.0 || W[12] != 0.0) ctrl->bc_znz = 1;
    }
}

// ------------------------------------------------------------------- ghost cells (L426)
// How a step chooses its dt.
struct StepCtl {
    int mode;          // 0: dt = value (fixed), 1: dt = value (= CFL number) / rate
    double value;
    double t_end;      // < 0: none; else the step is clipped to land on t_end, later steps skip
};

// One thread per ghost cell: side-major index over (side, position along the side, layer).
// Thread 0 also closes the CFL reduction of the state that is about to be stepped:
// dt = cfl / max(rate, ghost_rate) (L434), advances t and the step counter, and clears the
// accumulator slot the step kernel will max-reduce the NEXT state into.
// `U` is the array the step kernel reconstructs from: the conserved planes of the 5-moment system, the
// PRIMITIVE planes of the 14-moment system (prim = 1: Dirichlet cells take the table's W instead of its U;
// the conserved planes of that system are only read at interior cells and need no ghost values).
template <int NM>
__global__ void k_ghost(Params p, double* __restrict__ U, const BcTable* __restrict__ tab,
                        Ctrl* ctrl, int slot, StepCtl sc, int finalize, double* __restrict__ dt_hist, int prim)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (finalize && tid == 0) {
        const int bad = ctrl->bad[slot] | ctrl->failed | (int)ctrl->bc_bad;
        double rate = fmax(__longlong_as_double((long long)ctrl->rate_bits[slot]), ctrl->ghost_rate);
        double dt = sc.mode == 1 ? sc.value / rate : sc.value;
        int skip = 0;
        if (bad || (sc.mode == 1 && !(rate > 0.0))) { ctrl->failed = 1; skip = 1; }
        double t = ctrl->t, tn = t + dt;
        if (sc.t_end >= 0.0 && !skip) {
            if (t >= sc.t_end) skip = 1;
            else if (tn >= sc.t_end) { dt = sc.t_end - t; tn = sc.t_end; }
        }
        if (skip) dt = 0.0;
        else {
            dt_hist[ctrl->steps & (kDtHistory - 1)] = dt;     // step number `steps` (0-based) took dt
            ctrl->t = tn; ctrl->steps += 1; ctrl->last_dt = dt;
        }
        ctrl->dt = dt;
        ctrl->skip = skip;
        // a skipped step carries the state over unchanged, and its reduction with it
        ctrl->rate_bits[slot ^ 1] = skip ? ctrl->rate_bits[slot] : 0ull;
        ctrl->speed_bits[slot ^ 1] = skip ? ctrl->speed_bits[slot] : 0ull;
        ctrl->bad[slot ^ 1] = skip ? ctrl->bad[slot] : 0;
    }
    const int nx = p.nx, ny = p.ny;
    const int nxs = 2 * ny;                     // ghost cells per x side
    const int nys = (NM == 5) ? 0 : 2 * nx;     // per y side (1-D system has none)
    if (tid >= 2 * nxs + 2 * nys) return;
    int side, r;
    if (tid < 2 * nxs) { side = tid / nxs; r = tid % nxs; }
    else { const int d = nys > 0 ? nys : 1; side = 2 + (tid - 2 * nxs) / d; r = (tid - 2 * nxs) % d; }
    const int g = (r & 1) + 1, pos = r >> 1;    // layer 1..2, index along the side
    const BcSide& b = tab->side[side];
    int gi, gj, si, sj;                          // ghost cell, source cell (interior coords)
    double coord;
    if (side < 2) {
        gj = sj = pos;
        coord = __dadd_rn(p.y0, __dmul_rn((double)pos + 0.5, p.dy));
        if (side == 0) { gi = -g; si = b.type == 1 ? ((nx - g) % nx + nx) % nx : 0; }
        else { gi = nx - 1 + g; si = b.type == 1 ? (g - 1) % nx : nx - 1; }
    } else {
        gi = si = pos;
        coord = __dadd_rn(p.x0, __dmul_rn((double)pos + 0.5, p.dx));
        if (side == 2) { gj = -g; sj = b.type == 1 ? ((ny - g) % ny + ny) % ny : 0; }
        else { gj = ny - 1 + g; sj = b.type == 1 ? (g - 1) % ny : ny - 1; }
    }
    const size_t plane = (size_t)p.rows * p.pitch;
    const size_t gidx = (size_t)(gj + 2) * p.pitch + gi + 2, sidx = (size_t)(sj + 2) * p.pitch + si + 2;
    const double* fixed = nullptr;
    if (b.type == 2) {
        int k = b.has_default ? b.nbands : -1;
        for (int q = b.nbands - 1; q >= 0; --q)          // first matching band wins
            if (coord >= b.lo[q] && coord <= b.hi[q]) k = q;
        if (k >= 0) fixed = prim ? b.W[k] : b.U[k];
    }
    // all loads first: a store through U may alias the next load, which would chain NM memory round trips
    double v[NM];
#pragma unroll
    for (int m = 0; m < NM; ++m) v[m] = fixed ? fixed[m] : U[m * plane + sidx];
#pragma unroll
    for (int m = 0; m < NM; ++m) U[m * plane + gidx] = v[m];
}

// Standalone CFL reduction over the interior (used after mm_set_state).
template <int NM, int NT>
__global__ void __launch_bounds__(NT) k_rate(Params p, const double* __restrict__ U, Ctrl* ctrl,
                                             int slot)
{
    const size_t plane = (size_t)p.rows * p.pitch;
    double rate = 0.0, speed = 0.0;
    int bad = 0, znz = 0;
    const long long n = (long long)p.nx * p.ny;
    for (long long c = (long long)blockIdx.x * NT + threadIdx.x; c < n; c += (long long)gridDim.x * NT) {
        const int i = (int)(c % p.nx), j = (int)(c / p.nx);
        double u[NM];
#pragma unroll
        for (int m = 0; m < NM; ++m) u[m] = U[m * plane + (size_t)(j + 2) * p.pitch + i + 2];
        double r, s;
        cell_rate<NM>(p, u, r, s, bad);
        rate = fmax(rate, r); speed = fmax(speed, s);
        if constexpr (NM == 14) {
            if (u[3] != 0.0 || u[6] != 0.0 || u[8] != 0.0 || u[12] != 0.0) znz = 1;
        }
    }
    if (__syncthreads_or(znz) && threadIdx.x == 0) ctrl->znz = 1;
    block_reduce_rate<NT>(rate, speed, bad, ctrl, slot);
}

// ------------------------------------------------------------------ the fused time step
// (the 14-moment step kernel is in mm_tm14.cuh)
// 5-moment interface flux between cell a (low side) and cell b (high side) from the primitives
// staged in shared memory.  `w` points at cell b of moment plane 0, `ms` is the plane stride.
// MUSCL on primitives (L262-264): face states W_a + slope_a/2 and W_b - slope_b/2; closure flux,
// conserved state and wave speeds of both (eval_face5), then HLL / Rusanov.
// psi/4 of the cells a and b of the stencil (am, a, b, bp) with the shared limiter (L266)
template <int LIM>
__device__ __forceinline__ void shared_psi_pair5(const double (&Wam)[5], const double (&Wa)[5], const double (&Wb)[5],
                                                 const double (&Wbp)[5], double& qa, double& qb)
{
    PsiShared<LIM> ma, mb;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        ma.add(Wa[k] - Wam[k], Wb[k] - Wa[k], (Wa[k] - Wam[k]) + (Wb[k] - Wa[k]));
        mb.add(Wb[k] - Wa[k], Wbp[k] - Wb[k], (Wb[k] - Wa[k]) + (Wbp[k] - Wb[k]));
    }
    qa = 0.25 * ma.psi(); qb = 0.25 * mb.psi();
}

__device__ __forceinline__ void interface_flux5(const Params& p, const double* __restrict__ w,
                                                int ms, double (&Fh)[5])
{
    constexpr int NM = 5;
    double Wam[NM], Wa[NM], Wb[NM], Wbp[NM], WL[NM], WR[NM];
#pragma unroll
    for (int k = 0; k < NM; ++k) {
        const double* q = w + k * ms;
        Wam[k] = q[-2]; Wa[k] = q[-1]; Wb[k] = q[0]; Wbp[k] = q[1];
    }
    if (p.limiter != 0 && p.shared_limiter) {
        double qa, qb;
        if (p.limiter == 1) shared_psi_pair5<1>(Wam, Wa, Wb, Wbp, qa, qb);
        else shared_psi_pair5<2>(Wam, Wa, Wb, Wbp, qa, qb);
#pragma unroll
        for (int k = 0; k < NM; ++k) {
            WL[k] = Wa[k] + qa * ((Wa[k] - Wam[k]) + (Wb[k] - Wa[k]));
            WR[k] = Wb[k] - qb * ((Wb[k] - Wa[k]) + (Wbp[k] - Wb[k]));
        }
    } else {
#pragma unroll
        for (int k = 0; k < NM; ++k) {
            double ha = 0.0, hb = 0.0;
            if (p.limiter != 0) {
                const double d = Wb[k] - Wa[k];
                ha = 0.5 * limited_slope(p.limiter, Wa[k] - Wam[k], d);
                hb = 0.5 * limited_slope(p.limiter, d, Wbp[k] - Wb[k]);
            }
            WL[k] = Wa[k] + ha; WR[k] = Wb[k] - hb;
        }
    }
    double FL[NM], UL[NM], FR[NM], UR[NM], lminL, lmaxL, lminR, lmaxR;
    eval_face5(p, WL, FL, UL, lminL, lmaxL);
    eval_face5(p, WR, FR, UR, lminR, lmaxR);
    numflux<NM>(p.flux, FL, FR, UL, UR, lminL, lmaxL, lminR, lmaxR, Fh);
}

// 5-moment 1-D step: one block = NT consecutive cells, same four stages.
template <int NT>
__global__ void __launch_bounds__(NT)
k_step5(Params p, const double* __restrict__ Uin, double* Uout, Ctrl* ctrl, int slot_next,
        const double* Ubase, double dt_scale, int do_rate)
{
    constexpr int NM = 5, PW = NT + 4, PF = NT + 1;
    __shared__ double Ws[NM * PW];
    __shared__ double Fx[NM * PF];
    const int tid = threadIdx.x, gx0 = blockIdx.x * NT;
    const size_t plane = (size_t)p.rows * p.pitch;
    const size_t row = (size_t)2 * p.pitch;
    const double dt = ctrl->dt * dt_scale;          // see k_step14_strip for Ubase / dt_scale / do_rate
    const bool cell_ok = gx0 + tid < p.nx;
    const size_t cidx = row + gx0 + tid + 2;
    if (ctrl->skip) {
        if (cell_ok)
#pragma unroll
            for (int m = 0; m < NM; ++m) Uout[m * plane + cidx] = Uin[m * plane + cidx];
        return;
    }
    for (int idx = tid; idx < PW; idx += NT) {
        if (gx0 + idx >= p.nx + 4) continue;
        double U[NM], W[NM];
#pragma unroll
        for (int m = 0; m < NM; ++m) U[m] = Uin[m * plane + row + gx0 + idx];
        cons2prim5(U, W);
#pragma unroll
        for (int m = 0; m < NM; ++m) Ws[m * PW + idx] = W[m];
    }
    __syncthreads();
    for (int idx = tid; idx < PF; idx += NT) {
        if (gx0 + idx > p.nx) continue;
        double Fh[NM];
        interface_flux5(p, Ws + idx + 2, PW, Fh);
#pragma unroll
        for (int m = 0; m < NM; ++m) Fx[m * PF + idx] = Fh[m];
    }
    __syncthreads();
    double rate = 0.0, speed = 0.0;
    int bad = 0;
    if (cell_ok) {
        const double dtdx = dt * p.inv_dx;
        double Un[NM], W[NM];
#pragma unroll
        for (int m = 0; m < NM; ++m) {
            Un[m] = (Ubase ? Ubase : Uin)[m * plane + cidx] - dtdx * (Fx[m * PF + tid + 1] - Fx[m * PF + tid]);
            W[m] = Ws[m * PW + tid + 2];
        }
        if (p.tau_model != 0) {
            if (p.source_scheme == 1) {                  // point-implicit (L348): relax U* itself
                double Wst[NM];
                cons2prim5(Un, Wst);
                const double x = dt * inv_tau(p, Wst[0], Wst[2]);
                add_source5(Wst, x * rcp(1.0 + x), Un);
            } else {
                add_source5(W, dt * inv_tau(p, W[0], W[2]), Un);
            }
        }
#pragma unroll
        for (int m = 0; m < NM; ++m) Uout[m * plane + cidx] = Un[m];
        if (do_rate) cell_rate<NM>(p, Un, rate, speed, bad);
    }
    if (do_rate) block_reduce_rate<NT>(rate, speed, bad, ctrl, slot_next);
}

// cos(pi n / d) for integers n >= 0, d > 0, reduced exactly to the first quadrant so that the
// argument handed to cospi is at most 1/2 and carries one rounding only
__device__ inline double cos_quarter(int n, int d)
{
    n %= 2 * d;                                   // period 2 pi
    if (n > d) n = 2 * d - n;                     // cos(2 pi - x) = cos x
    const bool neg = 2 * n > d;                   // cos(pi - x) = -cos x
    if (neg) n = d - n;
    const double c = cospi((double)n / (double)d);
    return neg ? -c : c;
}

// Builds the AbTable (mm_physics.cuh): one thread per (interval, function).  Chebyshev
// interpolation of the direct formula at 14 nodes, then re-expansion in powers of the local
// coordinate t in [-1, 1] (coefficients stored highest power first, for Horner).
__global__ void k_ab_table(double* __restrict__ tab)
{
    constexpr int N = AbTable::kDeg + 1;
    const int i = blockIdx.x, f = threadIdx.x;              // interval, 0 = a / 1 = b
    if (i >= AbTable::kIntervals || f >= 2) return;
    const double half = 1.0 / AbTable::inv_half(i), mid = AbTable::lower(i) + half;
    double fv[N], c[N];
    for (int j = 0; j < N; ++j) {
        const double P = mid + half * cos_quarter(2 * j + 1, 2 * N);
        double a, b;
        ab_direct(P, &a, &b);
        fv[j] = f == 0 ? a : b;
    }
    for (int k = 0; k < N; ++k) {                           // Chebyshev coefficients, compensated sums
        double hi = 0.0, lo = 0.0;
        for (int j = 0; j < N; ++j) {
            const double w = cos_quarter(k * (2 * j + 1), 2 * N);
            const double pr = fv[j] * w, pe = fma(fv[j], w, -pr);          // two-product
            const double sm = hi + pr, bb = sm - hi;                       // two-sum
            lo += (hi - (sm - bb)) + (pr - bb) + pe;
            hi = sm;
        }
        c[k] = (hi + lo) * (k == 0 ? 1.0 : 2.0) / N;
    }
    double m[N], Tkm1[N], Tk[N];                            // monomial coefficients of sum c_k T_k
    for (int j = 0; j < N; ++j) { m[j] = 0.0; Tkm1[j] = 0.0; Tk[j] = 0.0; }
    Tkm1[0] = 1.0; Tk[1] = 1.0;                             // T_0, T_1
    m[0] += c[0]; m[1] += c[1];
    for (int k = 2; k < N; ++k) {
        double Tn[N];
        for (int j = 0; j < N; ++j) Tn[j] = (j > 0 ? 2.0 * Tk[j - 1] : 0.0) - Tkm1[j];
        for (int j = 0; j < N; ++j) { m[j] = fma(c[k], Tn[j], m[j]); Tkm1[j] = Tk[j]; Tk[j] = Tn[j]; }
    }
    double* out = tab + i * AbTable::kStride;
    for (int j = 0; j < N; ++j) out[2 * j + f] = m[N - 1 - j];
}

}  // namespace mm
