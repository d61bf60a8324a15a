// mm_tm14.cuh -- the fused 14-moment 2-D time step (steps a2-a9 of DESIGN.md section 2).
//
// One WARP owns a strip of 30 cells in x and marches through a chunk of rows in y; warps never
// synchronise with one another.  One block of NW warps runs per SM (the block is only a container:
// it shares one copy of the a(P*), b(P*) table of Eq 29c-d and one tensor-memory allocation).
//
// What limits this FP64 method on an SM is how many independent dependency chains are in flight: a
// DFMA has a latency of 8 cycles and the pipe accepts one per 2 cycles and scheduler (3 when it reads
// three distinct registers).  A face evaluation (closure + flux + wave speeds,
// Eqs 16, 21-25, 28-31) needs ~110 registers; evaluating the two faces of an interface side by side in
// one thread (round 1: 240 registers, 8 warps per SM) gives each of 2 warps per scheduler an
// instruction-level parallelism of ~2.  Here every thread evaluates ONE face at a time and 16 warps of
// 128 registers are resident (4 per scheduler; throughput scales linearly with resident warps).  The
// state that has to survive a face evaluation -- the finished left face of the interface (F, U,
// lambda: 2 NV + 1 doubles), the right face state (NV), the partial update of the row (NV) and the half
// slopes of the previous row (NV) -- is private to a lane, and is parked in TENSOR MEMORY (tcgen05.st /
// tcgen05.ld, 32 lanes x 128 columns per warp), Blackwell's 256 KB per SM that this tensor-core-free
// method would otherwise leave unused: registers hold one face, shared memory only what lanes exchange
// (the primitives ring and the row of own cells in flight).  The kernel sits exactly at the 128-register
// limit: measured variants that add live values to the sweep (ghost handling, earlier tensor-memory
// loads, part A of both faces side by side) spill and lose 3-10 %.
//
// The state lives in HBM twice: the conserved moments U (what the update advances, Eq 16) and the
// primitives W = W(U) (what the reconstruction reads, L264), both written by the tail of the step that
// produced them -- the tail needs W(U^{n+1}) anyway for the CFL wave speeds (a9), so cons->prim runs
// exactly once per cell and step, and no row is converted on load.  HBM has the bandwidth to spare
// (this method runs at ~20 % of it), the FP64 pipe does not.
// Per warp, in shared memory (NV = moments carried: 14, or the 10 z-even ones on the z-symmetric path):
//   ring  [3][NV][34]  primitives of the rows r-1 .. r+1 (cells x0-2 .. x0+31), a ring over r: row r+2
//                      is copied by cp.async from W in HBM into the slot of row r-1 while the x
//                      interfaces of row r are in work, at no register cost;
//   own   [NV][32]     conserved moments of the lanes' own cells in row r+1 (the base of the update),
//                      copied by cp.async in the same group;
// per lane, in tensor memory (columns of 32 bit, 2 per double):
//   face  [2 NV + 1]   F_k, U_k, lambda_min, lambda_max of the left face state of the interface in work
//                      (without F_0, which is U_1: Eq 16a);
//   wr    [NV]         the right face state W_C - h while the left one is evaluated;
//   acc   [NV]         partial update of the lane's cell in the row being assembled;
//   hsv   [NV]         half slope in y of the lane's cell in the previous row (each slope is computed once).
// Lane L holds cell L-1 of the strip in both directions (L = 1 .. 30; lanes 0 and 31 only supply the
// slopes of the two halo cells): its centre cell C has the neighbours M and P along the direction; the
// lane computes C's limited half slope h (a3), obtains the half slope hM of M, and evaluates the
// interface M|C from the face states W_M + hM and W_C - h, one after the other (a4-a7).
//   y (d = 0): C = row r, M = row r-1; hM from `hsv`; G_r completes row r-1:
//              U^{n+1} = acc - dt/dy G_r + dt C(W) (a8), store, wave speeds of the new state
//              into the running CFL maximum (a9); then acc = U_r + dt/dy G_r.  The product
//              dt/dy G_r is rounded on its own both times (no FMA contraction), so that equal
//              fluxes through the two y faces of a cell cancel exactly.
//   x (d = 1): M = cell L-2; hM by shuffle from lane L-1; acc -= dt/dx (F from lane L+1 - own F).
// Both directions and both sides run through ONE copy of the slope / closure / wave-speed code (non-
// unrolled loops), which keeps the kernel inside the instruction cache.
#pragma once
#include "mm_kernels.cuh"

namespace mm {

constexpr int kSW = 30;                 // cells per strip
constexpr int kRW = 34;                 // staged cells per row: 2 + 30 + 2

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
    static constexpr int warp_smem_doubles = 3 * NV * kRW + NV * 32;
#ifndef MM_TM_NW_ZS
#define MM_TM_NW_ZS 16
#endif
#ifndef MM_TM_NW_GEN
#define MM_TM_NW_GEN 8
#endif
    // Warps per block (one block per SM).  Registers are private to a scheduler (16384 each): 4 warps per
    // scheduler leave 128 registers per thread, 3 leave 168, 2 leave 255.  Shared memory: table 31.5 KB +
    // NW x 10.5 KB (z-symmetric) resp. 14.7 KB (general).
    static constexpr int NW = ZS ? MM_TM_NW_ZS : MM_TM_NW_GEN;
    static constexpr size_t smem_bytes = ((size_t)AbTable::kDoubles + (size_t)NW * warp_smem_doubles) * sizeof(double) + 16;
    // tensor-memory columns of a lane: [face | acc | hsv]
    static constexpr int tm_face = 0, tm_acc = 2 * (2 * NV + 1), tm_hsv = tm_acc + 2 * NV, tm_wr = tm_hsv + 2 * NV,
                         tm_cols = tm_wr + 2 * NV;
    // a warp may only touch the 32-lane quarter warp % 4: the (NW + 3) / 4 warps of a quarter split its 512 columns
    static constexpr int tm_stride = (512 / ((NW + 3) / 4)) & ~1;
    static_assert(tm_cols <= tm_stride, "tensor-memory columns of a warp");
};

__device__ __forceinline__ void cp_async8(double* smem_dst, const double* gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---- tensor memory as lane-private scratch: doubles of the calling lane at column `taddr` (each
// thread of the warp touches its own lane; the instructions are warp-collective, .sync.aligned).
// One double per instruction (32x32b.x2): its register pair is the operand as it stands, whereas the wider
// shapes need their 8-32 registers contiguous and cost a register move per word (measured: 100 moves per
// cell update with .x8 stores; same run time either way).
__device__ __forceinline__ void tm_st2(unsigned taddr, double a)
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(__double2loint(a)),
                 "r"(__double2hiint(a)) : "memory");
}
__device__ __forceinline__ double tm_ld2(unsigned taddr)
{
    int lo, hi;
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(lo), "=r"(hi) : "r"(taddr) : "memory");
    return __hiloint2double(hi, lo);
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

template <int N>
__device__ __forceinline__ void tm_store(unsigned taddr, const double (&v)[N])
{
#pragma unroll
    for (int k = 0; k < N; ++k) tm_st2(taddr + 2 * k, v[k]);
}
template <int N>
__device__ __forceinline__ void tm_load(unsigned taddr, double (&v)[N])   // includes the wait
{
#pragma unroll
    for (int k = 0; k < N; ++k) v[k] = tm_ld2(taddr + 2 * k);
    tm_wait_ld();
}

// Work decomposition: item = (strip, chunk); chunk c covers rows [c ny / nchunks, (c+1) ny / nchunks).
// EXT = false is the plain forward-Euler step with the explicit source (Ubase = nullptr,
// dt_scale = 1, do_rate = 1, source_scheme = 0 folded at compile time); EXT = true takes them at
// run time (midpoint passes, point-implicit source).
#ifdef MM_TM_MAXNREG
#define MM_TM_REGATTR __maxnreg__(MM_TM_MAXNREG)
#else
#define MM_TM_REGATTR __launch_bounds__(32 * Mom<ZS>::NW, 1)
#endif
template <bool ZS, bool EXT>
__global__ void MM_TM_REGATTR
k_step14_tm(const Params pg, const double* __restrict__ Win, const double* __restrict__ Uin, double* Wout, double* Uout,
            Ctrl* ctrl, int slot_next, int nstrips, int nchunks, const double* Ubase_, double dt_scale_, int do_rate_)
{
    const double* Ubase = EXT ? Ubase_ : nullptr;
    const double dt_scale = EXT ? dt_scale_ : 1.0;
    const int do_rate = EXT ? do_rate_ : 1;
    using Z = typename std::conditional<ZS, zero_t, double>::type;
    using M = Mom<ZS>;
    constexpr int NM = 14, NV = M::NV, NF = 2 * NV + 1, RS = NV * kRW;   // RS: doubles per staged row
    extern __shared__ __align__(16) double smem[];
    // the warp index through a shuffle: the compiler then knows it is warp-uniform and keeps what derives
    // from it (buffer bases, tensor-memory addresses) in uniform registers
    const int lane = threadIdx.x & 31, warp = __shfl_sync(0xffffffffu, threadIdx.x >> 5, 0);

    // the block's copy of the a(P*), b(P*) table (Eq 29c-d), and its tensor-memory allocation
    Params p = pg;
    for (int i = threadIdx.x; i < AbTable::kDoubles; i += 32 * M::NW) smem[i] = pg.ab[i];
    unsigned* tm_slot = reinterpret_cast<unsigned*>(smem + AbTable::kDoubles + M::NW * M::warp_smem_doubles);
    if (warp == 0) {
        const unsigned dst = (unsigned)__cvta_generic_to_shared(tm_slot);
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(dst) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const unsigned tm_base = *tm_slot;
    p.ab = smem;
    // this warp's 32 lanes x tm_stride columns: lane quarter warp % 4 (the only one the warp may touch)
    const unsigned tm = __shfl_sync(0xffffffffu, tm_base + ((unsigned)(32 * (warp & 3)) << 16)
                                                     + (unsigned)(M::tm_stride * (warp >> 2)), 0);

    const int item = blockIdx.x * M::NW + warp;
    bool work = item < nstrips * nchunks;
    const int strip = work ? item % nstrips : 0, chunk = work ? item / nstrips : 0;
    const int x0 = strip * kSW;
    const int y0 = (int)((long long)chunk * p.ny / nchunks);
    const int y1 = (int)((long long)(chunk + 1) * p.ny / nchunks);
    work = work && y1 > y0;
    double* ring = smem + AbTable::kDoubles + warp * M::warp_smem_doubles;
    double* own = ring + 3 * RS;
    const size_t plane = (size_t)p.rows * p.pitch;
    const int ncell = min(kSW, p.nx - x0);            // cells of this strip
    const int ncol = min(kRW, p.nx + 4 - x0);         // staged columns that exist
    const bool cell_ok = lane >= 1 && lane - 1 < ncell;   // the lane's cell is cell lane-1
    const size_t ccol = (size_t)x0 + lane + 1;        // padded column of the lane's cell

    if (work && ctrl->skip) {          // failed / past t_end: carry the state over unchanged
        if (cell_ok)
            for (int r = y0; r < y1; ++r)
#pragma unroll
                for (int m = 0; m < NM; ++m) {
                    if (ZS && z_odd(m)) continue;
                    const size_t o = m * plane + (size_t)(r + 2) * p.pitch + ccol;
                    Uout[o] = Uin[o]; Wout[o] = Win[o];
                }
        work = false;
    }
    if (work) {
    // U_out = B - dt div F(W_in) + source:  B = U_in for forward Euler and for the half step of the
    // midpoint scheme (dt_scale = 1/2, no CFL reduction); B = Ubase = U^n for its full step, which
    // may be written in place (Uout == Ubase: a cell's B is read by the lane that later writes it).
    const double dt = ctrl->dt * dt_scale;
    const double dtdx = dt / p.dx, dtdy = dt / p.dy;
    const int cl = min(max(lane, 1), ncell) + 1;     // y: ring column of the lane's cell (clamped to valid cells)
    const int cx = min(lane, ncol - 3);              // x: ring column of cell M (= cell C - 1), clamped

    auto load_row = [&](int r, int rslot) {          // primitives of interior row r in [-2, ny+1] -> ring[rslot]
        const double* src = Win + (size_t)(r + 2) * p.pitch + x0;
        double* dst = ring + rslot * RS;
        if (lane < ncol) {
#pragma unroll
            for (int k = 0; k < NV; ++k) cp_async8(dst + k * kRW + lane, src + M::full(k) * plane + lane);
        }
        if (lane + 32 < ncol) {
#pragma unroll
            for (int k = 0; k < NV; ++k) cp_async8(dst + k * kRW + 32 + lane, src + M::full(k) * plane + 32 + lane);
        }
    };
    auto load_own = [&](int r) {                     // conserved moments of the lanes' own cells in row r -> own
        if (!Ubase) {
            const double* src = Uin + (size_t)(r + 2) * p.pitch + x0 + cl;
#pragma unroll
            for (int k = 0; k < NV; ++k) cp_async8(own + k * 32 + lane, src + M::full(k) * plane);
        }
    };

    load_row(y0 - 2, 0); load_row(y0 - 1, 1); load_row(y0, 2);
    cp_async_commit();
    cp_async_wait_all(); __syncwarp();
    int sm = 0, sc = 1, sp = 2;                      // ring slots of the rows r-1, r, r+1

    double rate = 0.0, speed = 0.0;
    int bad = 0;
    for (int r = y0 - 1; r <= y1; ++r) {
#pragma unroll 1
        for (int d = 0; d < 2; ++d) {
            // Lanes without an interface of their own (beyond the strip's last cell / staged column)
            // take the last valid cell's data, so every lane evaluates a valid state; their
            // results are never used.
            const double *qm, *qc, *qp;              // plane 0 of the cells M, C, P
            if (d == 0) {                            // y: C = (row r, cell lane-1)
                const double* b = ring + cl;
                qm = b + sm * RS; qc = b + sc * RS; qp = b + sp * RS;
            } else {                                 // x: C = (row r, cell lane-1), M = cell lane-2
                if (r == y1) break;
                // row r-1 and the own cells of row r are done with: rows r+2 / r+1 into their places
                __syncwarp();
                load_row(r + 2, sm);
                if (r + 1 < y1) load_own(r + 1);
                cp_async_commit();
                if (r < y0) break;
                qm = ring + sc * RS + cx; qc = qm + 1; qp = qm + 2;
            }
            // ---- a3: limited half slope of C; face states of the interface M|C
            double Wf[NM];                           // the face state in work
            double WR[NV];                           // the right face state, evaluated second
            {
                double Wm[NV], Wc[NV], Wp[NV], h[NV];
                if (d == 0) {                        // the y stencil in x <-> y swapped numbering (L414); two copies of the
                                                     // loads: a run-time offset costs an integer multiply-add per load
#pragma unroll
                    for (int k = 0; k < NV; ++k) { Wm[k] = qm[M::cswap(k) * kRW]; Wc[k] = qc[M::cswap(k) * kRW]; Wp[k] = qp[M::cswap(k) * kRW]; }
                } else {
#pragma unroll
                    for (int k = 0; k < NV; ++k) { Wm[k] = qm[k * kRW]; Wc[k] = qc[k * kRW]; Wp[k] = qp[k * kRW]; }
                }
                half_slopes<NV>(p, Wm, Wc, Wp, h);
                if (d == 0) {
                    double hm[NV];
                    tm_load<NV>(tm + M::tm_hsv, hm);     // slope of row r-1 (garbage on the chunk's first pass: unused)
                    tm_store<NV>(tm + M::tm_hsv, h);

#pragma unroll
                    for (int k = 0; k < NV; ++k) { Wf[M::full(k)] = Wm[k] + hm[k]; WR[k] = Wc[k] - h[k]; }
                    if (r < y0) {                    // first pass of a chunk: slope of row y0-1 only.  The next pass loads it
                        tm_wait_st();                // back before any other wait::st: tcgen05.st -> tcgen05.ld of one thread
                        continue;                    // is not ordered without it
                    }
                    tm_store<NV>(tm + M::tm_wr, WR);
                } else {
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const double hm = __shfl_up_sync(0xffffffffu, h[k], 1);
                        Wf[M::full(k)] = Wm[k] + hm; WR[k] = Wc[k] - h[k];
                    }
                    tm_store<NV>(tm + M::tm_wr, WR);
                }
            }
            // ---- a4-a7: the two face states through the closure, one after the other; the left face's
            // results wait in tensor memory
            double F[NM], U[NM], lmin, lmax;
#pragma unroll 1          // one copy of the face evaluation (two copies: 0.74 instead of 0.69 ms, instruction cache)
            for (int side = 0; side < 2; ++side) {
                eval_face14<Z>(p, Wf, F, U, lmin, lmax);
                if (side == 0) {
                    double park[NF];                 // [U_0 | F_k, U_k (k >= 1) | lambda_min, lambda_max]: F_0 = U_1 (Eq 16a) is not parked
                    park[0] = U[0];
#pragma unroll
                    for (int k = 1; k < NV; ++k) { park[2 * k - 1] = F[M::full(k)]; park[2 * k] = U[M::full(k)]; }
                    park[2 * NV - 1] = lmin; park[2 * NV] = lmax;
                    tm_store<NF>(tm + M::tm_face, park);
                    double wr[NV];
                    tm_wait_st();
                    tm_load<NV>(tm + M::tm_wr, wr);
#pragma unroll
                    for (int k = 0; k < NV; ++k) Wf[M::full(k)] = wr[k];
                }
            }
            double Fh[NV];
            {
                double L[NF];
                tm_wait_st();
                tm_load<NF>(tm + M::tm_face, L);
                const double lminL = L[2 * NV - 1], lmaxL = L[2 * NV];
                // left face: U_k = LU(k), F_k = LF(k) with F_0 = U_1
#define MM_LU(k) L[(k) == 0 ? 0 : 2 * (k)]
#define MM_LF(k) L[(k) == 0 ? 2 : 2 * (k) - 1]
                if (p.flux == 1) {
                    const double S = dmax(dmax(fabs(lminL), fabs(lmaxL)), dmax(fabs(lmin), fabs(lmax)));
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const int m = M::full(k);
                        Fh[k] = 0.5 * (MM_LF(k) + F[m]) - 0.5 * S * (U[m] - MM_LU(k));
                    }
                } else {
                    const double SL = dmin(dmin(lminL, lmin), 0.0), SR = dmax(dmax(lmaxL, lmax), 0.0);
                    const double inv = rcp(SR - SL), cL = SR * inv, cR = -SL * inv, cU = SL * cL;
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        const int m = M::full(k);
                        Fh[k] = hll1(cL, cR, cU, MM_LF(k), F[m], MM_LU(k), U[m]);
                    }
                }
#undef MM_LU
#undef MM_LF
            }
            if (d == 0) {
                double G[NV];                        // back to unswapped numbering (L414)
#pragma unroll
                for (int k = 0; k < NV; ++k) G[k] = Fh[M::cswap(k)];
                double A[NV];
                if (r > y0) {                        // row r-1 is complete (a8), then a9 on the new state
                    tm_load<NV>(tm + M::tm_acc, A);
                    double Un[NM], W[NM];
                    const double* w = ring + sm * RS + cl;
#pragma unroll
                    for (int k = 0; k < NV; ++k) {
                        Un[M::full(k)] = __dsub_rn(A[k], __dmul_rn(dtdy, G[k]));
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
                    // the primitives of the new state (a2 of the next step) and its CFL wave speeds (a9)
                    double Wn[NM];
                    cons2prim14<Z>(Un, Wn);
                    if (cell_ok) {
                        const size_t o = (size_t)(r + 1) * p.pitch + ccol;
#pragma unroll
                        for (int k = 0; k < NV; ++k) {
                            Uout[M::full(k) * plane + o] = Un[M::full(k)];
                            Wout[M::full(k) * plane + o] = Wn[M::full(k)];
                        }
                        if (do_rate) {
                            double rr, ss;
                            prim_rate14<Z>(p, Wn, rr, ss, bad);
                            rate = dmax(rate, rr); speed = dmax(speed, ss);
                        }
                    }
                }
                if (r < y1) {
                    if (Ubase) {
                        const double* ub = Ubase + (size_t)(r + 2) * p.pitch + x0 + cl;
#pragma unroll
                        for (int k = 0; k < NV; ++k) A[k] = __dadd_rn(ub[M::full(k) * plane], __dmul_rn(dtdy, G[k]));
                    } else {
#pragma unroll
                        for (int k = 0; k < NV; ++k) A[k] = __dadd_rn(own[k * 32 + lane], __dmul_rn(dtdy, G[k]));
                    }
                    tm_store<NV>(tm + M::tm_acc, A);
                }
            } else {
                double A[NV];
                tm_wait_st();
                tm_load<NV>(tm + M::tm_acc, A);
#pragma unroll
                for (int k = 0; k < NV; ++k) {
                    const double Fn = __shfl_down_sync(0xffffffffu, Fh[k], 1);
                    A[k] = A[k] - dtdx * (Fn - Fh[k]);
                }
                tm_store<NV>(tm + M::tm_acc, A);
            }
        }
        if (r < y1) {                                // rows r+2 (primitives) and r+1 (own cells) have landed
            cp_async_wait_all(); __syncwarp();
            const int t = sm; sm = sc; sc = sp; sp = t;
        }
    }
    tm_wait_st();
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
    }   // work
    // every warp is done with its tensor-memory columns: release the allocation
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tm_base) : "memory");
    }
}

}  // namespace mm
