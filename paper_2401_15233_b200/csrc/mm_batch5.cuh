// mm_batch5.cuh -- batched 1-D 5-moment solver: many independent
// shock tubes advanced side by side, each with its own sigma_lim, Knudsen number, CFL time step and
// clock, so that parameter sweeps like the paper's sigma_lim x Kn study (section 4.3,
// L340-356, Fig 7) load the GPU, which a single 1000-cell tube cannot.
// Same scheme as k_step5 (steps a1-a9 of DESIGN.md section 2 for the 5-moment system, Eq 12/14/15/34):
// transmissive ends (zero-gradient ghost cells, formed on load by clamping the cell index),
// MUSCL + limiter on primitives, closure flux + Baradaran wave speeds, HLL / Rusanov, forward Euler
// with the explicit BGK source, CFL reduction of the new state per tube.
#pragma once
#include "mm_kernels.cuh"

#ifndef MM_BATCH5_MINB
#define MM_BATCH5_MINB 8        // resident blocks of 128 threads per SM the step kernel is compiled for
#endif

namespace mm {

struct TubeCtl {                       // one per tube, device memory
    double t, dt;
    unsigned long long rate_bits[2];   // CFL rate max_cells s/dx of the current / next state
    long long steps;
    int bad[2];
    int failed;                        // sticky: reduction met rho <= 0, P <= 0 or a non-finite speed
    int skip;                          // this step leaves the tube untouched (failed, or t_end reached)
};

// per-tube Params: the solver-wide ones with this tube's sigma_lim and collision coefficient
__device__ __forceinline__ Params tube_params(const Params& p, const double* __restrict__ sigma_lim,
                                              const double* __restrict__ inv_tau_coef, int j)
{
    Params q = p;
    q.sigma_lim = sigma_lim[j];
    q.inv_tau_coef = inv_tau_coef[j];
    q.tau_model = inv_tau_coef[j] > 0.0 ? 2 : 0;
    return q;
}

// One thread per tube, before every step: dt from the tube's own CFL rate (L434) or the fixed
// value, clipped to land on t_end; advances the tube's clock; clears the accumulator of the next state.
__global__ void k_batch5_finalize(int ntubes, TubeCtl* ctl, int slot, StepCtl sc)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= ntubes) return;
    TubeCtl& c = ctl[j];
    const double rate = __longlong_as_double((long long)c.rate_bits[slot]);
    double dt = sc.mode == 1 ? sc.value / rate : sc.value;
    int skip = 0;
    if (c.bad[slot] || c.failed || (sc.mode == 1 && !(rate > 0.0))) { c.failed = 1; skip = 1; }
    const double t = c.t;
    double tn = t + dt;
    if (sc.t_end >= 0.0 && !skip) {
        if (t >= sc.t_end) skip = 1;
        else if (tn >= sc.t_end) { dt = sc.t_end - t; tn = sc.t_end; }
    }
    if (skip) dt = 0.0;
    else { c.t = tn; c.steps += 1; }
    c.dt = dt;
    c.skip = skip;
    c.rate_bits[slot ^ 1] = skip ? c.rate_bits[slot] : 0ull;
    c.bad[slot ^ 1] = skip ? c.bad[slot] : 0;
}

// block-wide max of the rate and OR of the flag into the tube's accumulator
template <int NT>
__device__ __forceinline__ void tube_reduce(double rate, int bad, TubeCtl* c, int slot)
{
    __shared__ double s_rate[NT / 32];
    __shared__ int s_bad[NT / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        rate = fmax(rate, __shfl_xor_sync(0xffffffffu, rate, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { s_rate[w] = rate; s_bad[w] = bad; }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 1; k < NT / 32; ++k) { rate = fmax(rate, s_rate[k]); bad |= s_bad[k]; }
        atomic_max_pos(&c->rate_bits[slot], rate);
        if (bad) atomicOr(&c->bad[slot], 1);
    }
}

// CFL rate of the state just set (slot 0).  grid = (blocks along x, tubes)
template <int NT>
__global__ void __launch_bounds__(NT)
k_batch5_rate(Params p, const double* __restrict__ sigma_lim, const double* __restrict__ inv_tau_coef,
              const double* __restrict__ U, TubeCtl* ctl)
{
    const int j = blockIdx.y, i = blockIdx.x * NT + threadIdx.x;
    const Params q = tube_params(p, sigma_lim, inv_tau_coef, j);
    const double* u = U + (size_t)j * 5 * p.nx;
    double rate = 0.0, speed;
    int bad = 0;
    if (i < p.nx) {
        double Uc[5];
#pragma unroll
        for (int m = 0; m < 5; ++m) Uc[m] = u[(size_t)m * p.nx + i];
        cell_rate<5>(q, Uc, rate, speed, bad);
    }
    tube_reduce<NT>(rate, bad, &ctl[j], 0);
}

// One step of every tube.  State layout: [tube][moment][nx], no ghost storage.
// A block of NT threads owns NT - 1 cells: thread t evaluates the interface on the LEFT of cell gx0 + t
// (t = 0 .. NT-1, one per thread -- an (NT+1)-th interface would be a second pass of warp 0 alone, with every
// other warp waiting at the barrier), threads 0 .. NT-2 update their cells.
template <int NT>
__global__ void __launch_bounds__(NT, MM_BATCH5_MINB)
k_batch5_step(Params p, const double* __restrict__ sigma_lim, const double* __restrict__ inv_tau_coef,
              const double* __restrict__ Uin, double* __restrict__ Uout, TubeCtl* ctl, int slot_next)
{
    constexpr int NM = 5, NC = NT - 1, PW = NT + 3, PF = NT;
    __shared__ double Ws[NM * PW];
    __shared__ double Fx[NM * PF];
    const int j = blockIdx.y, tid = threadIdx.x, gx0 = blockIdx.x * NC;
    const size_t off = (size_t)j * NM * p.nx;
    const double* uin = Uin + off;
    double* uout = Uout + off;
    const bool cell_ok = tid < NC && gx0 + tid < p.nx;
    TubeCtl* c = &ctl[j];
    if (c->skip) {
        if (cell_ok)
#pragma unroll
            for (int m = 0; m < NM; ++m) uout[(size_t)m * p.nx + gx0 + tid] = uin[(size_t)m * p.nx + gx0 + tid];
        return;
    }
    const Params q = tube_params(p, sigma_lim, inv_tau_coef, j);
    const double dt = c->dt;
    // stage cells gx0-2 .. gx0+NT; beyond the ends the boundary cell is repeated (L426, zero gradient)
    for (int idx = tid; idx < PW; idx += NT) {
        const int i = min(max(gx0 + idx - 2, 0), p.nx - 1);
        double U[NM], W[NM];
#pragma unroll
        for (int m = 0; m < NM; ++m) U[m] = uin[(size_t)m * p.nx + i];
        cons2prim5(U, W);
#pragma unroll
        for (int m = 0; m < NM; ++m) Ws[m * PW + idx] = W[m];
    }
    __syncthreads();
    if (gx0 + tid <= p.nx) {
        double Fh[NM];
        interface_flux5(q, Ws + tid + 2, PW, Fh);
#pragma unroll
        for (int m = 0; m < NM; ++m) Fx[m * PF + tid] = Fh[m];
    }
    __syncthreads();
    double rate = 0.0, speed;
    int bad = 0;
    if (cell_ok) {
        const double dtdx = dt * p.inv_dx;
        double Un[NM], W[NM];
#pragma unroll
        for (int m = 0; m < NM; ++m) {
            Un[m] = uin[(size_t)m * p.nx + gx0 + tid] - dtdx * (Fx[m * PF + tid + 1] - Fx[m * PF + tid]);
            W[m] = Ws[m * PW + tid + 2];
        }
        if (q.tau_model != 0) add_source5(W, dt * inv_tau(q, W[0], W[2]), Un);
#pragma unroll
        for (int m = 0; m < NM; ++m) uout[(size_t)m * p.nx + gx0 + tid] = Un[m];
        cell_rate<NM>(q, Un, rate, speed, bad);
    }
    tube_reduce<NT>(rate, bad, c, slot_next);
}

// primitives [5][nx] (one tube, broadcast) or [ntubes][5][nx] -> conserved [ntubes][5][nx]
__global__ void k_batch5_pack(int nx, int ntubes, int per_tube, const double* __restrict__ W, double* __restrict__ U)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y;
    if (i >= nx) return;
    const double* w = W + (per_tube ? (size_t)j * 5 * nx : 0);
    double a[5], b[5];
#pragma unroll
    for (int m = 0; m < 5; ++m) a[m] = w[(size_t)m * nx + i];
    prim2cons5(a, b);
#pragma unroll
    for (int m = 0; m < 5; ++m) U[((size_t)j * 5 + m) * nx + i] = b[m];
}

}  // namespace mm
